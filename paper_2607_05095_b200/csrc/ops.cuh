// ops.cuh -- the row-gather operators that plug into tiers.cuh.
//
// All softmax arithmetic is done in the base-2 domain: s2 = s*log2(e), m2 = reference max of s2,
// p = exp2(s2 - m2) (one MUFU.EX2 each), LSE = (m2 + log2 l) * ln 2.
// Per-edge scalars are per-lane arrays over the lane's NHL head slots (rowops.cuh).
#pragma once
#include "tiers.cuh"

#define TG_NEG_INF (-__int_as_float(0x7f800000))
// "no edge seen yet" reference maximum: finite, so that (-inf) - m and m - m never give NaN
constexpr float TG_NEG_BIG = -1.0e30f;
// The online softmax rescales its accumulators only when a logit exceeds the reference maximum by more
// than TG_TAU (base-2 units), so p <= 2^TG_TAU and the common trip carries no rescale at all.  The state
// (m, l, acc) then stands for l*2^m, acc*2^m with m any reference <= true max + 0, >= true max - TG_TAU:
// the merge and the final division are exact in the same way as with the true maximum.
constexpr float TG_TAU = 8.0f;

// -------------------------------------------------------------------------------------------------
// Fused forward: online softmax (reference max m2, sum l, weighted accumulator) + aggregation.
// PAPER.md:225 (stable softmax, online normaliser ref [16]) + PAPER.md:215 (AGG).
// State {m2[NHL], l[NHL], acc[NE]}.
// -------------------------------------------------------------------------------------------------
template <class Tr_>
struct FwdOp {
    using Tr = Tr_;
    using T = typename Tr::T;
    static constexpr int NHL = Tr::NHL, NS = Tr::NE + 2 * NHL, NS1 = NS;
    struct Params {
        const T *Q, *K, *V;
        const int32_t* kv;
        T* O;
        float* lse;
        float* part;
        float scale2;  // scale * log2(e)
        float* O32;    // nullable: fp32 copy of O for the backward (bf16 storage: delta = <dO, O> without O's bf16 rounding)
    };
    struct Buf { RowReg<Tr> k, v; };
    const Params& p;
    LanePos<Tr> lp;
    RowReg<Tr> q;
    __device__ __forceinline__ FwdOp(const Params& p_, int lig) : p(p_), lp(lig) {}
    __device__ __forceinline__ const int32_t* idx_ptr() const { return p.kv; }
    __device__ __forceinline__ void load(Buf& b, int r, int) const {
        row_load(b.k, p.K + lp.off + (size_t)r * Tr::F, lp);
        row_load(b.v, p.V + lp.off + (size_t)r * Tr::F, lp);
    }
    __device__ __forceinline__ void init_row(int row) { row_load(q, p.Q + lp.off + (size_t)row * Tr::F, lp); }
    __device__ __forceinline__ void init_state(float (&st)[NS]) {
#pragma unroll
        for (int j = 0; j < NHL; ++j) { st[j] = TG_NEG_BIG; st[NHL + j] = 0.f; }
#pragma unroll
        for (int i = 0; i < Tr::NE; ++i) st[2 * NHL + i] = 0.f;
    }
    template <int UNR, bool MASK>
    __device__ __forceinline__ void compute(float (&st)[NS], const Buf (&b)[UNR], int pos0, int stride, int end) {
        float s[UNR][NHL];
        bool need = false;
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            row_dot_heads(q, b[u].k, lp, s[u]);
            const bool ok = !MASK || (pos0 + u * stride < end);
#pragma unroll
            for (int j = 0; j < NHL; ++j) {
                s[u][j] = ok ? s[u][j] * p.scale2 : TG_NEG_INF;
                need |= s[u][j] > st[j] + TG_TAU;
            }
        }
        if (__any_sync(0xffffffffu, need)) {
            float c[NHL];
#pragma unroll
            for (int j = 0; j < NHL; ++j) {
                float mn = st[j];
#pragma unroll
                for (int u = 0; u < UNR; ++u) mn = fmaxf(mn, s[u][j]);
                c[j] = tg_exp2(st[j] - mn);
                st[j] = mn;
                st[NHL + j] *= c[j];
            }
            row_scale_heads(st + 2 * NHL, c, lp);
        }
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            float pr[NHL];
#pragma unroll
            for (int j = 0; j < NHL; ++j) {
                pr[j] = tg_exp2(s[u][j] - st[j]);
                st[NHL + j] += pr[j];
            }
            row_axpy_heads(st + 2 * NHL, pr, b[u].v, lp);
        }
    }
    __device__ __forceinline__ void merge(float (&a)[NS], const float (&b)[NS]) {
        float ca[NHL], cb[NHL];
#pragma unroll
        for (int j = 0; j < NHL; ++j) {
            const float mn = fmaxf(a[j], b[j]);
            ca[j] = tg_exp2(a[j] - mn); cb[j] = tg_exp2(b[j] - mn);
            a[j] = mn;
            a[NHL + j] = a[NHL + j] * ca[j] + b[NHL + j] * cb[j];
        }
        float tmp[Tr::NE];
#pragma unroll
        for (int i = 0; i < Tr::NE; ++i) tmp[i] = b[2 * NHL + i];
        row_scale_heads(a + 2 * NHL, ca, lp);
        row_scale_heads(tmp, cb, lp);
#pragma unroll
        for (int i = 0; i < Tr::NE; ++i) a[2 * NHL + i] += tmp[i];
    }
    __device__ __forceinline__ void write_final(int row, float (&st)[NS], bool) {
        float inv[NHL];
#pragma unroll
        for (int j = 0; j < NHL; ++j) inv[j] = st[NHL + j] > 0.f ? 1.f / st[NHL + j] : 0.f;
        row_scale_heads(st + 2 * NHL, inv, lp);
        row_store(p.O + (size_t)row * Tr::F, lp, st + 2 * NHL, 1.f);
        if (p.O32) row_store_f32<Tr>(p.O32 + (size_t)row * Tr::F, lp, st + 2 * NHL);
        if (lp.head_writer()) {
#pragma unroll
            for (int j = 0; j < NHL; ++j)
                p.lse[(size_t)row * Tr::H + lp.head(j)] = st[NHL + j] > 0.f ? (st[j] + log2f(st[NHL + j])) * TG_LN2 : TG_NEG_INF;
        }
    }
    __device__ __forceinline__ void write_partial(int slot, float (&st)[NS], bool) { tg_partial_store<Tr, NS>(p.part, slot, lp.lig, st); }
    __device__ __forceinline__ void load_partial(int slot, float (&st)[NS]) { tg_partial_load<Tr, NS>(p.part, slot, lp.lig, st); }
};

// -------------------------------------------------------------------------------------------------
// Fused backward, destination-major pass: delta, dQ.  Plain-sum state.
//   alpha = exp2(s2 - lse2); dalpha = <dO[v], V[r]>; ds = alpha*(dalpha - delta); dQ = scale * sum ds*K[r]
// delta[v,h] = sum_{N(v)} alpha*dalpha (= <dO[v,h,:], O[v,h,:]>).
//   fp32 storage: delta is taken from <dO, O> up front; state dq[NE].
//   bf16 storage: O was rounded to bf16, which puts ~2^-9 relative noise on <dO, O> -- enough to push a few
//     dQ elements per 10^4 outside 1e-3 + 2e-2|ref| (measured).  delta is therefore
//     accumulated from the edges in fp32 in the same sweep: state {A1 = sum alpha*dalpha*K, A2 = sum alpha*K,
//     d = sum alpha*dalpha}, dQ = scale*(A1 - d*A2).  One extra axpy per edge, O is not read.
// Also writes ld[v,h] = {lse2, delta} for the source-major pass.
// -------------------------------------------------------------------------------------------------
template <class Tr_, bool EDGE_DELTA_ = Tr_::BF16>
struct Bwd1Op {
    using Tr = Tr_;
    using T = typename Tr::T;
    // bf16 storage without an fp32 copy of O: delta from the edges.  EDGE_DELTA_ = false with bf16 storage needs Params::O32.
    static constexpr bool EDGE_DELTA = EDGE_DELTA_;
    static constexpr int NHL = Tr::NHL;
    static constexpr int NS = EDGE_DELTA ? 2 * Tr::NE + NHL : Tr::NE, NS1 = NS;
    struct Params {
        const T *Q, *K, *V, *O, *dO;
        const int32_t* kv;
        const float* lse;
        T* dQ;
        float2* ld;
        float* part;
        float scale, scale2;
        const float* O32;   // nullable: the forward's fp32 copy of O (bf16 storage)
    };
    struct Buf { RowReg<Tr> k, v; };
    const Params& p;
    LanePos<Tr> lp;
    RowReg<Tr> q, g;
    float lse2[NHL], delta[NHL];
    int cur;
    __device__ __forceinline__ Bwd1Op(const Params& p_, int lig) : p(p_), lp(lig) {}
    __device__ __forceinline__ const int32_t* idx_ptr() const { return p.kv; }
    __device__ __forceinline__ void load(Buf& b, int r, int) const {
        row_load(b.k, p.K + lp.off + (size_t)r * Tr::F, lp);
        row_load(b.v, p.V + lp.off + (size_t)r * Tr::F, lp);
    }
    __device__ __forceinline__ void init_row(int row) {
        cur = row;
        row_load(q, p.Q + lp.off + (size_t)row * Tr::F, lp);
        row_load(g, p.dO + lp.off + (size_t)row * Tr::F, lp);
        if constexpr (!EDGE_DELTA && Tr::BF16) {      // delta = <dO, O> with O taken from its fp32 side copy
            float of[Tr::NE], gf[Tr::NE];
            row_load_f32<Tr>(of, p.O32 + (size_t)row * Tr::F, lp);
            row_to_float(g, gf);
            row_dotf_heads<Tr>(gf, of, lp, delta);
        } else if constexpr (!EDGE_DELTA) {
            RowReg<Tr> o;
            row_load(o, p.O + lp.off + (size_t)row * Tr::F, lp);
            row_dot_heads(g, o, lp, delta);
        } else {
#pragma unroll
            for (int j = 0; j < NHL; ++j) delta[j] = 0.f;
        }
#pragma unroll
        for (int j = 0; j < NHL; ++j) lse2[j] = tg_ldg_f32(p.lse + (size_t)row * Tr::H + lp.head(j)) * TG_LOG2E;
    }
    __device__ __forceinline__ void init_state(float (&st)[NS]) {
#pragma unroll
        for (int i = 0; i < NS; ++i) st[i] = 0.f;
    }
    template <int UNR, bool MASK>
    __device__ __forceinline__ void compute(float (&st)[NS], const Buf (&b)[UNR], int pos0, int stride, int end) {
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            float s2[NHL], da[NHL], a[NHL];
            row_dot_heads(q, b[u].k, lp, s2);
            row_dot_heads(g, b[u].v, lp, da);
            const bool ok = !MASK || (pos0 + u * stride < end);
#pragma unroll
            for (int j = 0; j < NHL; ++j) a[j] = ok ? tg_exp2(fmaf(s2[j], p.scale2, -lse2[j])) : 0.f;
            if constexpr (EDGE_DELTA) {
                float ada[NHL];
#pragma unroll
                for (int j = 0; j < NHL; ++j) {
                    ada[j] = a[j] * da[j];
                    st[2 * Tr::NE + j] += ada[j];
                }
                row_axpy2_heads(st, st + Tr::NE, ada, a, b[u].k, lp);
            } else {
                float c[NHL];
#pragma unroll
                for (int j = 0; j < NHL; ++j) c[j] = a[j] * (da[j] - delta[j]);
                row_axpy_heads(st, c, b[u].k, lp);
            }
        }
    }
    __device__ __forceinline__ void merge(float (&a)[NS], const float (&b)[NS]) {
#pragma unroll
        for (int i = 0; i < NS; ++i) a[i] += b[i];
    }
    __device__ __forceinline__ void write_final(int row, float (&st)[NS], bool first) {
        if constexpr (EDGE_DELTA) {
            float d[NHL];
#pragma unroll
            for (int j = 0; j < NHL; ++j) d[j] = st[2 * Tr::NE + j];
            row_fnma_heads(st, d, st + Tr::NE, lp);
            row_store(p.dQ + (size_t)row * Tr::F, lp, st, p.scale);
            // `first` is false only in the hub merge, which owns the row's delta
            if (lp.head_writer()) {
#pragma unroll
                for (int j = 0; j < NHL; ++j) {
                    const size_t o = (size_t)row * Tr::H + lp.head(j);
                    p.ld[o] = make_float2(tg_ldg_f32(p.lse + o) * TG_LOG2E, d[j]);
                }
            }
        } else {
            row_store(p.dQ + (size_t)row * Tr::F, lp, st, p.scale);
            if (first) write_ld();
        }
    }
    __device__ __forceinline__ void write_ld() {
        if (lp.head_writer()) {
#pragma unroll
            for (int j = 0; j < NHL; ++j) p.ld[(size_t)cur * Tr::H + lp.head(j)] = make_float2(lse2[j], delta[j]);
        }
    }
    __device__ __forceinline__ void write_partial(int slot, float (&st)[NS], bool first) {
        tg_partial_store<Tr, NS>(p.part, slot, lp.lig, st);
        if constexpr (!EDGE_DELTA) {
            if (first) write_ld();
        }
    }
    __device__ __forceinline__ void load_partial(int slot, float (&st)[NS]) { tg_partial_load<Tr, NS>(p.part, slot, lp.lig, st); }
};

// -------------------------------------------------------------------------------------------------
// Fused backward, source-major pass over the transposed CSR: dK, dV gathered, no float atomics.
// State {dk[NE], dv[NE]}.  Row u keeps K[u], V[u]; each transposed edge gathers Q[v], dO[v], ld[v].
// -------------------------------------------------------------------------------------------------
template <class Tr_>
struct Bwd2Op {
    using Tr = Tr_;
    using T = typename Tr::T;
    static constexpr int NHL = Tr::NHL, NS = 2 * Tr::NE, NS1 = NS;
    struct Params {
        const T *Q, *K, *V, *dO;
        const int32_t* t_dst;
        const float2* ld;
        T *dK, *dV;
        float* part;
        float scale, scale2;
    };
    struct Buf { RowReg<Tr> q, g; float2 x[NHL]; };
    const Params& p;
    LanePos<Tr> lp;
    RowReg<Tr> k, v;
    __device__ __forceinline__ Bwd2Op(const Params& p_, int lig) : p(p_), lp(lig) {}
    __device__ __forceinline__ const int32_t* idx_ptr() const { return p.t_dst; }
    __device__ __forceinline__ void load(Buf& b, int r, int) const {
        row_load(b.q, p.Q + lp.off + (size_t)r * Tr::F, lp);
        row_load(b.g, p.dO + lp.off + (size_t)r * Tr::F, lp);
#pragma unroll
        for (int j = 0; j < NHL; ++j) b.x[j] = __ldg(p.ld + (size_t)r * Tr::H + lp.head(j));
    }
    __device__ __forceinline__ void init_row(int row) {
        row_load(k, p.K + lp.off + (size_t)row * Tr::F, lp);
        row_load(v, p.V + lp.off + (size_t)row * Tr::F, lp);
    }
    __device__ __forceinline__ void init_state(float (&st)[NS]) {
#pragma unroll
        for (int i = 0; i < NS; ++i) st[i] = 0.f;
    }
    template <int UNR, bool MASK>
    __device__ __forceinline__ void compute(float (&st)[NS], const Buf (&b)[UNR], int pos0, int stride, int end) {
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            float s2[NHL], da[NHL], a[NHL], c[NHL];
            row_dot_heads(b[u].q, k, lp, s2);
            row_dot_heads(b[u].g, v, lp, da);
            const bool ok = !MASK || (pos0 + u * stride < end);
#pragma unroll
            for (int j = 0; j < NHL; ++j) {
                a[j] = ok ? tg_exp2(fmaf(s2[j], p.scale2, -b[u].x[j].x)) : 0.f;
                c[j] = a[j] * (da[j] - b[u].x[j].y);
            }
            row_axpy_heads(st, c, b[u].q, lp);
            row_axpy_heads(st + Tr::NE, a, b[u].g, lp);
        }
    }
    __device__ __forceinline__ void merge(float (&a)[NS], const float (&b)[NS]) {
#pragma unroll
        for (int i = 0; i < NS; ++i) a[i] += b[i];
    }
    __device__ __forceinline__ void write_final(int row, float (&st)[NS], bool) {
        row_store(p.dK + (size_t)row * Tr::F, lp, st, p.scale);
        row_store(p.dV + (size_t)row * Tr::F, lp, st + Tr::NE, 1.f);
    }
    __device__ __forceinline__ void write_partial(int slot, float (&st)[NS], bool) { tg_partial_store<Tr, NS>(p.part, slot, lp.lig, st); }
    __device__ __forceinline__ void load_partial(int slot, float (&st)[NS]) { tg_partial_load<Tr, NS>(p.part, slot, lp.lig, st); }
};

// -------------------------------------------------------------------------------------------------
// SDDMM: s[e,h] = scale * <A[row], B[idx[e]]> over one CSR side.  No state.
// -------------------------------------------------------------------------------------------------
template <class Tr_>
struct SddmmOp {
    using Tr = Tr_;
    using T = typename Tr::T;
    static constexpr int NHL = Tr::NHL, NS = 0, NS1 = 1;
    struct Params {
        const T *A, *B;
        const int32_t* idx;
        float* s;
        float scale;
    };
    struct Buf { RowReg<Tr> b; };
    const Params& p;
    LanePos<Tr> lp;
    RowReg<Tr> a;
    __device__ __forceinline__ SddmmOp(const Params& p_, int lig) : p(p_), lp(lig) {}
    __device__ __forceinline__ const int32_t* idx_ptr() const { return p.idx; }
    __device__ __forceinline__ void load(Buf& b, int r, int) const { row_load(b.b, p.B + lp.off + (size_t)r * Tr::F, lp); }
    __device__ __forceinline__ void init_row(int row) { row_load(a, p.A + lp.off + (size_t)row * Tr::F, lp); }
    __device__ __forceinline__ void init_state(float (&)[1]) {}
    template <int UNR, bool MASK>
    __device__ __forceinline__ void compute(float (&)[1], const Buf (&b)[UNR], int pos0, int stride, int end) {
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            float d[NHL];
            row_dot_heads(a, b[u].b, lp, d);
            const int e = pos0 + u * stride;
            if ((!MASK || e < end) && lp.head_writer()) {
#pragma unroll
                for (int j = 0; j < NHL; ++j) p.s[(size_t)e * Tr::H + lp.head(j)] = d[j] * p.scale;
            }
        }
    }
    __device__ __forceinline__ void merge(float (&)[1], const float (&)[1]) {}
    __device__ __forceinline__ void write_final(int, float (&)[1], bool) {}
    __device__ __forceinline__ void write_partial(int, float (&)[1], bool) {}
    __device__ __forceinline__ void load_partial(int, float (&)[1]) {}
};

// -------------------------------------------------------------------------------------------------
// Weighted row aggregation over one CSR side: Y[row] = sum_i w[widx ? widx[i] : i, h] * X[idx[i]].
// w == NULL: the paper's plain neighbour sum.  Forward uses (kv_row, positions),
// backward uses the transposed side (t_dst rows of dY, weights looked up through t_edge).
// -------------------------------------------------------------------------------------------------
template <class Tr_>
struct AggOp {
    using Tr = Tr_;
    using T = typename Tr::T;
    static constexpr int NHL = Tr::NHL, NS = Tr::NE, NS1 = NS;
    struct Params {
        const T* X;
        const int32_t* idx;
        const int32_t* widx;
        const float* w;
        T* Y;
        float* part;
    };
    struct Buf { RowReg<Tr> x; float w[NHL]; };
    const Params& p;
    LanePos<Tr> lp;
    __device__ __forceinline__ AggOp(const Params& p_, int lig) : p(p_), lp(lig) {}
    __device__ __forceinline__ const int32_t* idx_ptr() const { return p.idx; }
    __device__ __forceinline__ void load(Buf& b, int r, int pos) const {
        row_load(b.x, p.X + lp.off + (size_t)r * Tr::F, lp);
        if (p.w) {
            const int we = p.widx ? tg_ldg_i32(p.widx + pos) : pos;
#pragma unroll
            for (int j = 0; j < NHL; ++j) b.w[j] = tg_ldg_f32(p.w + (size_t)we * Tr::H + lp.head(j));
        } else {
#pragma unroll
            for (int j = 0; j < NHL; ++j) b.w[j] = 1.f;
        }
    }
    __device__ __forceinline__ void init_row(int) {}
    __device__ __forceinline__ void init_state(float (&st)[NS]) {
#pragma unroll
        for (int i = 0; i < NS; ++i) st[i] = 0.f;
    }
    template <int UNR, bool MASK>
    __device__ __forceinline__ void compute(float (&st)[NS], const Buf (&b)[UNR], int pos0, int stride, int end) {
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            const bool ok = !MASK || (pos0 + u * stride < end);
            float w[NHL];
#pragma unroll
            for (int j = 0; j < NHL; ++j) w[j] = ok ? b[u].w[j] : 0.f;
            row_axpy_heads(st, w, b[u].x, lp);
        }
    }
    __device__ __forceinline__ void merge(float (&a)[NS], const float (&b)[NS]) {
#pragma unroll
        for (int i = 0; i < NS; ++i) a[i] += b[i];
    }
    __device__ __forceinline__ void write_final(int row, float (&st)[NS], bool) { row_store(p.Y + (size_t)row * Tr::F, lp, st, 1.f); }
    __device__ __forceinline__ void write_partial(int slot, float (&st)[NS], bool) { tg_partial_store<Tr, NS>(p.part, slot, lp.lig, st); }
    __device__ __forceinline__ void load_partial(int slot, float (&st)[NS]) { tg_partial_load<Tr, NS>(p.part, slot, lp.lig, st); }
};
