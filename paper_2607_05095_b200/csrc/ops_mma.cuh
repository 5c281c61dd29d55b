// ops_mma.cuh -- the three fused attention operators with their per-head dot products on the tensor cores
// (mma_dot.cuh), for the WARP tier.  State, merge, partial and final formulas are those of ops.cuh (the operators derive
// from them and stay interchangeable with them: the group tiers and the hub merges keep the FHFMA operators); what
// changes is the edge loop: a lane owns the softmax scalars of ONE (head, group) pair -- head = lane >> 2, group =
// lane & 3, "head layout" -- and one shuffle per slot hands each lane the scalars of its own vectors for the axpy.
// bf16 rows of 256 bytes with D in {16, 32} only (MmaDotOk); every other shape keeps the FHFMA operators.
#pragma once
#include "mma_dot.cuh"
#include "ops.cuh"

// position of edge u of the group whose scalars this lane owns (warp tier: group g walks pos = begin + g + n * stride)
template <class Tr>
__device__ __forceinline__ bool tg_mma_ok(const MmaLane<Tr>& ml, int pos0, int u, int stride, int end) {
    return pos0 - ml.grp + ml.gt + u * stride < end;
}

// -------------------------------------------------------------------------------------------------
// Forward.  During the edge loop st[0] / st[NHL] hold the reference max / the sum of (head, group) in head layout;
// end_edges() turns them into FwdOp's slot layout.
// -------------------------------------------------------------------------------------------------
template <class Tr_>
struct FwdMmaOp : FwdOp<Tr_> {
    using Base = FwdOp<Tr_>;
    using Tr = Tr_;
    using T = typename Tr::T;
    using Params = typename Base::Params;
    using Buf = typename Base::Buf;
    static constexpr int NHL = Base::NHL, NS = Base::NS, NS1 = Base::NS1;
    static_assert(MmaDotOk<Tr>::value, "layout not covered by the HMMA dot products");
    MmaLane<Tr> ml;
    MmaFixed<Tr> fq;
    __device__ __forceinline__ FwdMmaOp(const Params& p_, int lig) : Base(p_, lig), ml(threadIdx.x & 31) {}
    __device__ __forceinline__ void init_row(int row) { fq.load(this->p.Q + (size_t)row * Tr::F, threadIdx.x & 31); }
    template <int UNR, bool MASK>
    __device__ __forceinline__ void compute(float (&st)[NS], const Buf (&b)[UNR], int pos0, int stride, int end) {
        float s2[UNR];
        bool need = false;
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            const float c = fq.dot(b[u].k, ml.odd);
            const bool ok = !MASK || tg_mma_ok(ml, pos0, u, stride, end);
            s2[u] = ok ? c * this->p.scale2 : TG_NEG_INF;
            need |= s2[u] > st[0] + TG_TAU;
        }
        if (__any_sync(0xffffffffu, need)) {     // rare: raise the reference maximum, rescale l and the accumulators
            float mn = st[0];
#pragma unroll
            for (int u = 0; u < UNR; ++u) mn = fmaxf(mn, s2[u]);
            const float f = tg_exp2(st[0] - mn);
            st[0] = mn;
            st[NHL] *= f;
            float fs[NHL];
#pragma unroll
            for (int k = 0; k < Tr::NK; ++k) fs[k] = ml.to_slot(f, k);
            row_scale_heads(st + 2 * NHL, fs, this->lp);
        }
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            const float pr = tg_exp2(s2[u] - st[0]);
            st[NHL] += pr;
            float ps[NHL];
#pragma unroll
            for (int k = 0; k < Tr::NK; ++k) ps[k] = ml.to_slot(pr, k);
            row_axpy_heads(st + 2 * NHL, ps, b[u].v, this->lp);
        }
    }
    // head layout -> slot layout of {m, l}: from here on the state is FwdOp's
    __device__ __forceinline__ void end_edges(float (&st)[NS]) {
        float m[NHL], l[NHL];
#pragma unroll
        for (int k = 0; k < Tr::NK; ++k) { m[k] = ml.to_slot(st[0], k); l[k] = ml.to_slot(st[NHL], k); }
#pragma unroll
        for (int k = 0; k < Tr::NK; ++k) { st[k] = m[k]; st[NHL + k] = l[k]; }
    }
};

// -------------------------------------------------------------------------------------------------
// Backward, destination-major (bf16 storage: delta accumulated from the edges).
// State {A1[NE], A2[NE], d[NHL]}; during the loop d lives in st[2*NE] in head layout.
// -------------------------------------------------------------------------------------------------
template <class Tr_>
struct Bwd1MmaOp : Bwd1Op<Tr_> {
    using Base = Bwd1Op<Tr_>;
    using Tr = Tr_;
    using T = typename Tr::T;
    using Params = typename Base::Params;
    using Buf = typename Base::Buf;
    static constexpr int NHL = Base::NHL, NS = Base::NS, NS1 = Base::NS1;
    static_assert(MmaDotOk<Tr>::value && Base::EDGE_DELTA, "layout not covered by the HMMA dot products");
    MmaLane<Tr> ml;
    MmaFixed<Tr> fq, fg;
    float lse2h;     // lse * log2(e) of (row, head lane >> 2)
    __device__ __forceinline__ Bwd1MmaOp(const Params& p_, int lig) : Base(p_, lig), ml(threadIdx.x & 31) {}
    __device__ __forceinline__ void init_row(int row) {
        this->cur = row;
        fq.load(this->p.Q + (size_t)row * Tr::F, threadIdx.x & 31);
        fg.load(this->p.dO + (size_t)row * Tr::F, threadIdx.x & 31);
        lse2h = ml.live ? tg_ldg_f32(this->p.lse + (size_t)row * Tr::H + ml.hd) * TG_LOG2E : 0.f;
    }
    template <int UNR, bool MASK>
    __device__ __forceinline__ void compute(float (&st)[NS], const Buf (&b)[UNR], int pos0, int stride, int end) {
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            const float s = fq.dot(b[u].k, ml.odd);
            const float da = fg.dot(b[u].v, ml.odd);
            const bool ok = !MASK || tg_mma_ok(ml, pos0, u, stride, end);
            const float a = ok ? tg_exp2(fmaf(s, this->p.scale2, -lse2h)) : 0.f;
            const float ada = a * da;
            st[2 * Tr::NE] += ada;
            float as[NHL], adas[NHL];
#pragma unroll
            for (int k = 0; k < Tr::NK; ++k) { as[k] = ml.to_slot(a, k); adas[k] = ml.to_slot(ada, k); }
            row_axpy2_heads(st, st + Tr::NE, adas, as, b[u].k, this->lp);
        }
    }
    __device__ __forceinline__ void end_edges(float (&st)[NS]) {
        float d[NHL];
#pragma unroll
        for (int k = 0; k < Tr::NK; ++k) d[k] = ml.to_slot(st[2 * Tr::NE], k);
#pragma unroll
        for (int k = 0; k < Tr::NK; ++k) st[2 * Tr::NE + k] = d[k];
    }
};

// -------------------------------------------------------------------------------------------------
// Backward, source-major over the transposed CSR.  Fixed rows K[u], V[u]; gathered Q[v], dO[v] and the {lse2, delta}
// record of (v, head lane >> 2) for the edge of group lane & 3.
// -------------------------------------------------------------------------------------------------
template <class Tr_>
struct Bwd2MmaOp : Bwd2Op<Tr_> {
    using Base = Bwd2Op<Tr_>;
    using Tr = Tr_;
    using T = typename Tr::T;
    using Params = typename Base::Params;
    static constexpr int NHL = Base::NHL, NS = Base::NS, NS1 = Base::NS1;
    static_assert(MmaDotOk<Tr>::value, "layout not covered by the HMMA dot products");
    struct Buf { RowReg<Tr> q, g; float2 x; };
    MmaLane<Tr> ml;
    MmaFixed<Tr> fk, fv;
    __device__ __forceinline__ Bwd2MmaOp(const Params& p_, int lig) : Base(p_, lig), ml(threadIdx.x & 31) {}
    __device__ __forceinline__ void load(Buf& b, int r, int) const {
        row_load(b.q, this->p.Q + this->lp.off + (size_t)r * Tr::F, this->lp);
        row_load(b.g, this->p.dO + this->lp.off + (size_t)r * Tr::F, this->lp);
        const int rg = __shfl_sync(0xffffffffu, r, 8 * ml.gt);      // destination of the edge of group lane & 3
        b.x = __ldg(this->p.ld + (size_t)rg * Tr::H + (ml.live ? ml.hd : 0));
    }
    __device__ __forceinline__ void init_row(int row) {
        fk.load(this->p.K + (size_t)row * Tr::F, threadIdx.x & 31);
        fv.load(this->p.V + (size_t)row * Tr::F, threadIdx.x & 31);
    }
    template <int UNR, bool MASK>
    __device__ __forceinline__ void compute(float (&st)[NS], const Buf (&b)[UNR], int pos0, int stride, int end) {
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            const float s = fk.dot(b[u].q, ml.odd);
            const float da = fv.dot(b[u].g, ml.odd);
            const bool ok = !MASK || tg_mma_ok(ml, pos0, u, stride, end);
            const float a = ok ? tg_exp2(fmaf(s, this->p.scale2, -b[u].x.x)) : 0.f;
            const float c = a * (da - b[u].x.y);
            float as[NHL], cs[NHL];
#pragma unroll
            for (int k = 0; k < Tr::NK; ++k) { as[k] = ml.to_slot(a, k); cs[k] = ml.to_slot(c, k); }
            row_axpy_heads(st, cs, b[u].q, this->lp);
            row_axpy_heads(st + Tr::NE, as, b[u].g, this->lp);
        }
    }
};

// operator of the warp tier for the base operator Op: the HMMA variant where the layout allows it
template <class Op, bool ENABLE> struct tg_warp_op { using type = Op; };
template <class Tr> struct tg_warp_op<FwdOp<Tr>, true> { using type = FwdMmaOp<Tr>; };
template <class Tr> struct tg_warp_op<Bwd1Op<Tr>, true> { using type = Bwd1MmaOp<Tr>; };
template <class Tr> struct tg_warp_op<Bwd2Op<Tr>, true> { using type = Bwd2MmaOp<Tr>; };
