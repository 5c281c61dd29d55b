// ops_edge.cuh -- NEXT-1: the full TGAT edge term.  Every sampled edge adds its own
// row (time encoding / edge-feature projection) to the gathered key and value, and the logits pass a
// LeakyReLU:   z = scale*<Q[v], K[r] + Ke[e]>,  s = z > 0 ? z : slope*z,  O[v] = sum alpha*(V[r] + Ve[e]).
// Ke, Ve are [E, H, D] in CSR order.  The operators plug into the same tier drivers (tiers.cuh); per edge they gather four
// rows instead of two, so the per-edge rows (the rho = 1, HBM-bound regime) dominate the traffic.
// LeakyReLU is positively homogeneous, so it commutes with the base-2 scaling of the logits.
#pragma once
#include "ops.cuh"

__device__ __forceinline__ float tg_lrelu(float z, float slope) { return z > 0.f ? z : z * slope; }

// -------------------------------------------------------------------------------------------------
// Forward.  State {m2[NHL], l[NHL], acc[NE]} as FwdOp.
// -------------------------------------------------------------------------------------------------
template <class Tr_>
struct FwdEOp {
    using Tr = Tr_;
    using T = typename Tr::T;
    static constexpr int NHL = Tr::NHL, NS = Tr::NE + 2 * NHL, NS1 = NS;
    struct Params {
        const T *Q, *K, *V, *Ke, *Ve;
        const int32_t* kv;
        T* O;
        float* lse;
        float* part;
        float scale2, slope;
    };
    struct Buf { RowReg<Tr> k, v, ke, ve; };
    const Params& p;
    LanePos<Tr> lp;
    RowReg<Tr> q;
    __device__ __forceinline__ FwdEOp(const Params& p_, int lig) : p(p_), lp(lig) {}
    __device__ __forceinline__ const int32_t* idx_ptr() const { return p.kv; }
    __device__ __forceinline__ void load(Buf& b, int r, int pos) const {
        row_load(b.k, p.K + lp.off + (size_t)r * Tr::F, lp);
        row_load(b.ke, p.Ke + lp.off + (size_t)pos * Tr::F, lp);
        row_load(b.v, p.V + lp.off + (size_t)r * Tr::F, lp);
        row_load(b.ve, p.Ve + lp.off + (size_t)pos * Tr::F, lp);
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
            float se[NHL];
            row_dot_heads(q, b[u].k, lp, s[u]);
            row_dot_heads(q, b[u].ke, lp, se);
            const bool ok = !MASK || (pos0 + u * stride < end);
#pragma unroll
            for (int j = 0; j < NHL; ++j) {
                s[u][j] = ok ? tg_lrelu((s[u][j] + se[j]) * p.scale2, p.slope) : TG_NEG_INF;
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
            row_axpy_heads(st + 2 * NHL, pr, b[u].ve, lp);
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
// Backward, destination-major pass: delta, dQ (and the {lse2, delta} table).  With w = (z > 0 ? 1 : slope):
//   dz = alpha*(dalpha - delta)*w,  dQ = scale * sum dz*(K[r] + Ke[e]).
// As in Bwd1Op, bf16 storage accumulates delta from the edges: state {A1 = sum alpha*dalpha*w*(K+Ke),
// A2 = sum alpha*w*(K+Ke), d = sum alpha*dalpha}, dQ = scale*(A1 - d*A2); fp32 storage takes delta = <dO, O> up front.
// -------------------------------------------------------------------------------------------------
template <class Tr_>
struct Bwd1EOp {
    using Tr = Tr_;
    using T = typename Tr::T;
    static constexpr bool EDGE_DELTA = Tr::BF16;
    static constexpr int NHL = Tr::NHL;
    static constexpr int NS = EDGE_DELTA ? 2 * Tr::NE + NHL : Tr::NE, NS1 = NS;
    struct Params {
        const T *Q, *K, *V, *Ke, *Ve, *O, *dO;
        const int32_t* kv;
        const float* lse;
        T* dQ;
        T *dKe, *dVe;   // fp32 storage only (delta is final before the sweep): the per-edge rows are written here, no extra pass
        float2* ld;
        float* part;
        float scale, scale2, slope;
    };
    struct Buf { RowReg<Tr> k, v, ke, ve; };
    const Params& p;
    LanePos<Tr> lp;
    RowReg<Tr> q, g;
    float lse2[NHL], delta[NHL];
    int cur;
    __device__ __forceinline__ Bwd1EOp(const Params& p_, int lig) : p(p_), lp(lig) {}
    __device__ __forceinline__ const int32_t* idx_ptr() const { return p.kv; }
    __device__ __forceinline__ void load(Buf& b, int r, int pos) const {
        row_load(b.k, p.K + lp.off + (size_t)r * Tr::F, lp);
        row_load(b.ke, p.Ke + lp.off + (size_t)pos * Tr::F, lp);
        row_load(b.v, p.V + lp.off + (size_t)r * Tr::F, lp);
        row_load(b.ve, p.Ve + lp.off + (size_t)pos * Tr::F, lp);
    }
    __device__ __forceinline__ void init_row(int row) {
        cur = row;
        row_load(q, p.Q + lp.off + (size_t)row * Tr::F, lp);
        row_load(g, p.dO + lp.off + (size_t)row * Tr::F, lp);
        if constexpr (!EDGE_DELTA) {
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
            float z[NHL], ze[NHL], da[NHL], dae[NHL], a[NHL], aw[NHL];
            row_dot_heads(q, b[u].k, lp, z);
            row_dot_heads(q, b[u].ke, lp, ze);
            row_dot_heads(g, b[u].v, lp, da);
            row_dot_heads(g, b[u].ve, lp, dae);
            const bool ok = !MASK || (pos0 + u * stride < end);
#pragma unroll
            for (int j = 0; j < NHL; ++j) {
                const float z2 = (z[j] + ze[j]) * p.scale2;
                a[j] = ok ? tg_exp2(tg_lrelu(z2, p.slope) - lse2[j]) : 0.f;
                aw[j] = z2 > 0.f ? a[j] : a[j] * p.slope;
                da[j] += dae[j];
            }
            if constexpr (EDGE_DELTA) {
                float c1[NHL];
#pragma unroll
                for (int j = 0; j < NHL; ++j) {
                    st[2 * Tr::NE + j] = fmaf(a[j], da[j], st[2 * Tr::NE + j]);
                    c1[j] = aw[j] * da[j];
                }
                row_axpy2_heads(st, st + Tr::NE, c1, aw, b[u].k, lp);
                row_axpy2_heads(st, st + Tr::NE, c1, aw, b[u].ke, lp);
            } else {
                float c[NHL];
#pragma unroll
                for (int j = 0; j < NHL; ++j) c[j] = aw[j] * (da[j] - delta[j]);
                row_axpy_heads(st, c, b[u].k, lp);
                row_axpy_heads(st, c, b[u].ke, lp);
                if (ok) {   // dKe[e] = scale*dz*Q[v], dVe[e] = alpha*dO[v]
                    const size_t e = (size_t)(pos0 + u * stride);
                    float x[Tr::NE], cs[NHL];
#pragma unroll
                    for (int j = 0; j < NHL; ++j) cs[j] = c[j] * p.scale;
                    row_to_float(q, x);
                    row_scale_heads(x, cs, lp);
                    row_store(p.dKe + e * Tr::F, lp, x, 1.f);
                    row_to_float(g, x);
                    row_scale_heads(x, a, lp);
                    row_store(p.dVe + e * Tr::F, lp, x, 1.f);
                }
            }
        }
    }
    __device__ __forceinline__ void merge(float (&a)[NS], const float (&b)[NS]) {
#pragma unroll
        for (int i = 0; i < NS; ++i) a[i] += b[i];
    }
    __device__ __forceinline__ void write_ld() {
        if (lp.head_writer()) {
#pragma unroll
            for (int j = 0; j < NHL; ++j) p.ld[(size_t)cur * Tr::H + lp.head(j)] = make_float2(lse2[j], delta[j]);
        }
    }
    __device__ __forceinline__ void write_final(int row, float (&st)[NS], bool first) {
        if constexpr (EDGE_DELTA) {
            float d[NHL];
#pragma unroll
            for (int j = 0; j < NHL; ++j) d[j] = st[2 * Tr::NE + j];
            row_fnma_heads(st, d, st + Tr::NE, lp);
            row_store(p.dQ + (size_t)row * Tr::F, lp, st, p.scale);
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
    __device__ __forceinline__ void write_partial(int slot, float (&st)[NS], bool first) {
        tg_partial_store<Tr, NS>(p.part, slot, lp.lig, st);
        if constexpr (!EDGE_DELTA) {
            if (first) write_ld();
        }
    }
    __device__ __forceinline__ void load_partial(int slot, float (&st)[NS]) { tg_partial_load<Tr, NS>(p.part, slot, lp.lig, st); }
};

// -------------------------------------------------------------------------------------------------
// Backward, per-edge pass (no state): with delta final, every edge writes its own gradient rows
//   dKe[e] = scale*dz*Q[v],  dVe[e] = alpha*dO[v].
// (dK[u], dV[u] are the sums of these rows over the transposed CSR; they are accumulated by Bwd2EOp from unrounded terms.)
// -------------------------------------------------------------------------------------------------
template <class Tr_>
struct BwdEdgeOp {
    using Tr = Tr_;
    using T = typename Tr::T;
    static constexpr int NHL = Tr::NHL, NS = 0, NS1 = 1;
    struct Params {
        const T *Q, *K, *V, *Ke, *Ve, *dO;
        const int32_t* kv;
        const float2* ld;
        T *dKe, *dVe;
        float scale, scale2, slope;
    };
    struct Buf { RowReg<Tr> k, v, ke, ve; };
    const Params& p;
    LanePos<Tr> lp;
    RowReg<Tr> q, g;
    float qf[Tr::NE], gf[Tr::NE];
    float lse2[NHL], delta[NHL];
    __device__ __forceinline__ BwdEdgeOp(const Params& p_, int lig) : p(p_), lp(lig) {}
    __device__ __forceinline__ const int32_t* idx_ptr() const { return p.kv; }
    __device__ __forceinline__ void load(Buf& b, int r, int pos) const {
        row_load(b.k, p.K + lp.off + (size_t)r * Tr::F, lp);
        row_load(b.ke, p.Ke + lp.off + (size_t)pos * Tr::F, lp);
        row_load(b.v, p.V + lp.off + (size_t)r * Tr::F, lp);
        row_load(b.ve, p.Ve + lp.off + (size_t)pos * Tr::F, lp);
    }
    __device__ __forceinline__ void init_row(int row) {
        row_load(q, p.Q + lp.off + (size_t)row * Tr::F, lp);
        row_load(g, p.dO + lp.off + (size_t)row * Tr::F, lp);
        row_to_float(q, qf);
        row_to_float(g, gf);
#pragma unroll
        for (int j = 0; j < NHL; ++j) {
            const float2 x = __ldg(p.ld + (size_t)row * Tr::H + lp.head(j));
            lse2[j] = x.x; delta[j] = x.y;
        }
    }
    __device__ __forceinline__ void init_state(float (&)[1]) {}
    template <int UNR, bool MASK>
    __device__ __forceinline__ void compute(float (&)[1], const Buf (&b)[UNR], int pos0, int stride, int end) {
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            float z[NHL], ze[NHL], da[NHL], dae[NHL], a[NHL], c[NHL];
            row_dot_heads(q, b[u].k, lp, z);
            row_dot_heads(q, b[u].ke, lp, ze);
            row_dot_heads(g, b[u].v, lp, da);
            row_dot_heads(g, b[u].ve, lp, dae);
            const int e = pos0 + u * stride;
#pragma unroll
            for (int j = 0; j < NHL; ++j) {
                const float z2 = (z[j] + ze[j]) * p.scale2;
                a[j] = tg_exp2(tg_lrelu(z2, p.slope) - lse2[j]);
                c[j] = a[j] * (da[j] + dae[j] - delta[j]) * (z2 > 0.f ? 1.f : p.slope) * p.scale;
            }
            if (!MASK || e < end) {
                float x[Tr::NE];
#pragma unroll
                for (int i = 0; i < Tr::NE; ++i) x[i] = qf[i];
                row_scale_heads(x, c, lp);
                row_store(p.dKe + (size_t)e * Tr::F, lp, x, 1.f);
#pragma unroll
                for (int i = 0; i < Tr::NE; ++i) x[i] = gf[i];
                row_scale_heads(x, a, lp);
                row_store(p.dVe + (size_t)e * Tr::F, lp, x, 1.f);
            }
        }
    }
    __device__ __forceinline__ void merge(float (&)[1], const float (&)[1]) {}
    __device__ __forceinline__ void write_final(int, float (&)[1], bool) {}
    __device__ __forceinline__ void write_partial(int, float (&)[1], bool) {}
    __device__ __forceinline__ void load_partial(int, float (&)[1]) {}
};

// -------------------------------------------------------------------------------------------------
// Backward, source-major pass over the transposed CSR: dK[u] = sum_{r(e)=u} scale*dz*Q[v], dV[u] = sum alpha*dO[v],
// accumulated in fp32 from recomputed terms (summing the stored, storage-rounded dKe / dVe rows instead would
// stack one bf16 rounding per edge under the sum: measured outside the bf16 bound on cancelling rows).
// Row u keeps K[u], V[u]; each transposed edge j gathers Q[v], dO[v], ld[v] (v = t_dst[j]) and Ke[e], Ve[e] (e = t_edge[j]).
// -------------------------------------------------------------------------------------------------
template <class Tr_>
struct Bwd2EOp {
    using Tr = Tr_;
    using T = typename Tr::T;
    static constexpr int NHL = Tr::NHL, NS = 2 * Tr::NE, NS1 = NS;
    struct Params {
        const T *Q, *K, *V, *Ke, *Ve, *dO;
        const int32_t *t_dst, *t_edge;
        const float2* ld;
        T *dK, *dV;
        float* part;
        float scale, scale2, slope;
    };
    struct Buf { RowReg<Tr> q, g, ke, ve; float2 x[NHL]; };
    const Params& p;
    LanePos<Tr> lp;
    RowReg<Tr> k, v;
    __device__ __forceinline__ Bwd2EOp(const Params& p_, int lig) : p(p_), lp(lig) {}
    __device__ __forceinline__ const int32_t* idx_ptr() const { return p.t_dst; }
    __device__ __forceinline__ void load(Buf& b, int r, int pos) const {
        const int e = tg_ldg_i32(p.t_edge + pos);
        row_load(b.q, p.Q + lp.off + (size_t)r * Tr::F, lp);
        row_load(b.g, p.dO + lp.off + (size_t)r * Tr::F, lp);
#pragma unroll
        for (int j = 0; j < NHL; ++j) b.x[j] = __ldg(p.ld + (size_t)r * Tr::H + lp.head(j));
        row_load(b.ke, p.Ke + lp.off + (size_t)e * Tr::F, lp);
        row_load(b.ve, p.Ve + lp.off + (size_t)e * Tr::F, lp);
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
            float z[NHL], ze[NHL], da[NHL], dae[NHL], a[NHL], c[NHL];
            row_dot_heads(b[u].q, k, lp, z);
            row_dot_heads(b[u].q, b[u].ke, lp, ze);
            row_dot_heads(b[u].g, v, lp, da);
            row_dot_heads(b[u].g, b[u].ve, lp, dae);
            const bool ok = !MASK || (pos0 + u * stride < end);
#pragma unroll
            for (int j = 0; j < NHL; ++j) {
                const float z2 = (z[j] + ze[j]) * p.scale2;
                a[j] = ok ? tg_exp2(tg_lrelu(z2, p.slope) - b[u].x[j].x) : 0.f;
                c[j] = a[j] * (da[j] + dae[j] - b[u].x[j].y) * (z2 > 0.f ? 1.f : p.slope);
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
