// ops.cuh -- the row-gather operators that plug into tiers.cuh.
//
// All softmax arithmetic is done in the base-2 domain: s2 = s*log2(e), m2 = running max of s2,
// p = exp2(s2 - m2) (one MUFU.EX2 each), LSE = (m2 + log2 l) * ln 2.
#pragma once
#include "tiers.cuh"

#define TG_NEG_INF (-__int_as_float(0x7f800000))

// -------------------------------------------------------------------------------------------------
// Fused forward: online softmax (running max m2, sum l, weighted accumulator) + aggregation.
// PAPER.md:225 (stable softmax, online normaliser ref [16]) + PAPER.md:215 (AGG).  State {m2, l, acc[NE]}.
// -------------------------------------------------------------------------------------------------
template <class Tr_, int UNR_>
struct FwdOp {
    using Tr = Tr_;
    using T = typename Tr::T;
    static constexpr int UNR = UNR_, NS = Tr::NE + 2, NS1 = NS;
    struct Params {
        const T *Q, *K, *V;
        const int32_t* kv;
        T* O;
        float* lse;
        float* part;
        float scale2;  // scale * log2(e)
    };
    const Params& p;
    LanePos<Tr> lp;
    RowReg<Tr> q;
    __device__ __forceinline__ FwdOp(const Params& p_, int lig) : p(p_), lp(lig) {}
    __device__ __forceinline__ void init_row(int row) { row_load(q, p.Q + (size_t)row * Tr::F, lp); }
    __device__ __forceinline__ void init_state(float (&st)[NS]) {
        st[0] = TG_NEG_INF;
#pragma unroll
        for (int i = 1; i < NS; ++i) st[i] = 0.f;
    }
    __device__ __forceinline__ void edges(float (&st)[NS], int i0, int end, int stride, int trips) {
        float m = st[0], l = st[1];
        for (int t = 0; t < trips; ++t) {
            bool ok[UNR];
            RowReg<Tr> k[UNR], v[UNR];
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                const int i = i0 + (t * UNR + u) * stride;
                ok[u] = i < end;
                const int r = tg_ldg_i32(p.kv + (ok[u] ? i : 0));
                row_load(k[u], p.K + (size_t)r * Tr::F, lp);
                row_load(v[u], p.V + (size_t)r * Tr::F, lp);
            }
            float s[UNR], mn = m;
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                const float d = head_sum<Tr>(row_dot(q, k[u])) * p.scale2;
                s[u] = ok[u] ? d : TG_NEG_INF;
                mn = fmaxf(mn, s[u]);
            }
            const float ms = (mn == TG_NEG_INF) ? 0.f : mn;
            const float corr = tg_exp2(m - ms);
            l *= corr;
#pragma unroll
            for (int i = 0; i < Tr::NE; ++i) st[2 + i] *= corr;
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                const float pu = tg_exp2(s[u] - ms);
                l += pu;
                row_axpy(st + 2, pu, v[u]);
            }
            m = mn;
        }
        st[0] = m; st[1] = l;
    }
    __device__ __forceinline__ void merge(float (&a)[NS], const float (&b)[NS]) {
        const float mn = fmaxf(a[0], b[0]);
        const float ms = (mn == TG_NEG_INF) ? 0.f : mn;
        const float ca = tg_exp2(a[0] - ms), cb = tg_exp2(b[0] - ms);
        a[0] = mn;
#pragma unroll
        for (int i = 1; i < NS; ++i) a[i] = a[i] * ca + b[i] * cb;
    }
    __device__ __forceinline__ void write_final(int row, float (&st)[NS], bool) {
        const float l = st[1];
        const float inv = l > 0.f ? 1.f / l : 0.f;
        row_store(p.O + (size_t)row * Tr::F, lp, st + 2, inv);
        if (lp.j == 0) p.lse[(size_t)row * Tr::H + lp.h] = (st[0] + log2f(l)) * TG_LN2;
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
template <class Tr_, int UNR_>
struct Bwd1Op {
    using Tr = Tr_;
    using T = typename Tr::T;
    static constexpr bool EDGE_DELTA = Tr::BF16;
    static constexpr int UNR = UNR_, NS = EDGE_DELTA ? 2 * Tr::NE + 1 : Tr::NE, NS1 = NS;
    struct Params {
        const T *Q, *K, *V, *O, *dO;
        const int32_t* kv;
        const float* lse;
        T* dQ;
        float2* ld;
        float* part;
        float scale, scale2;
    };
    const Params& p;
    LanePos<Tr> lp;
    RowReg<Tr> q, g;
    float lse2, delta;
    int cur;
    __device__ __forceinline__ Bwd1Op(const Params& p_, int lig) : p(p_), lp(lig) {}
    __device__ __forceinline__ void init_row(int row) {
        cur = row;
        row_load(q, p.Q + (size_t)row * Tr::F, lp);
        row_load(g, p.dO + (size_t)row * Tr::F, lp);
        delta = 0.f;
        if constexpr (!EDGE_DELTA) {
            RowReg<Tr> o;
            row_load(o, p.O + (size_t)row * Tr::F, lp);
            delta = head_sum<Tr>(row_dot(g, o));
        }
        lse2 = tg_ldg_f32(p.lse + (size_t)row * Tr::H + lp.h) * TG_LOG2E;
    }
    __device__ __forceinline__ void init_state(float (&st)[NS]) {
#pragma unroll
        for (int i = 0; i < NS; ++i) st[i] = 0.f;
    }
    __device__ __forceinline__ void edges(float (&st)[NS], int i0, int end, int stride, int trips) {
        for (int t = 0; t < trips; ++t) {
            bool ok[UNR];
            RowReg<Tr> k[UNR], v[UNR];
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                const int i = i0 + (t * UNR + u) * stride;
                ok[u] = i < end;
                const int r = tg_ldg_i32(p.kv + (ok[u] ? i : 0));
                row_load(k[u], p.K + (size_t)r * Tr::F, lp);
                row_load(v[u], p.V + (size_t)r * Tr::F, lp);
            }
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                const float s2 = head_sum<Tr>(row_dot(q, k[u])) * p.scale2;
                const float da = head_sum<Tr>(row_dot(g, v[u]));
                const float a = ok[u] ? tg_exp2(s2 - lse2) : 0.f;
                if constexpr (EDGE_DELTA) {
                    const float ada = a * da;
                    st[2 * Tr::NE] += ada;
                    row_axpy2(st, st + Tr::NE, ada, a, k[u]);
                } else {
                    row_axpy(st, a * (da - delta), k[u]);
                }
            }
        }
    }
    __device__ __forceinline__ void merge(float (&a)[NS], const float (&b)[NS]) {
#pragma unroll
        for (int i = 0; i < NS; ++i) a[i] += b[i];
    }
    __device__ __forceinline__ void write_final(int row, float (&st)[NS], bool first) {
        if constexpr (EDGE_DELTA) {
            const float d = st[2 * Tr::NE];
#pragma unroll
            for (int i = 0; i < Tr::NE; ++i) st[i] = fmaf(-d, st[Tr::NE + i], st[i]);
            row_store(p.dQ + (size_t)row * Tr::F, lp, st, p.scale);
            // `first` is false only in the hub merge, which owns the row's delta
            if (lp.j == 0) p.ld[(size_t)row * Tr::H + lp.h] = make_float2(tg_ldg_f32(p.lse + (size_t)row * Tr::H + lp.h) * TG_LOG2E, d);
        } else {
            row_store(p.dQ + (size_t)row * Tr::F, lp, st, p.scale);
            if (first && lp.j == 0) p.ld[(size_t)cur * Tr::H + lp.h] = make_float2(lse2, delta);
        }
    }
    __device__ __forceinline__ void write_partial(int slot, float (&st)[NS], bool first) {
        tg_partial_store<Tr, NS>(p.part, slot, lp.lig, st);
        if constexpr (!EDGE_DELTA) {
            if (first && lp.j == 0) p.ld[(size_t)cur * Tr::H + lp.h] = make_float2(lse2, delta);
        }
    }
    __device__ __forceinline__ void load_partial(int slot, float (&st)[NS]) { tg_partial_load<Tr, NS>(p.part, slot, lp.lig, st); }
};

// -------------------------------------------------------------------------------------------------
// Fused backward, source-major pass over the transposed CSR: dK, dV gathered, no float atomics.
// State {dk[NE], dv[NE]}.  Row u keeps K[u], V[u]; each transposed edge gathers Q[v], dO[v], ld[v].
// -------------------------------------------------------------------------------------------------
template <class Tr_, int UNR_>
struct Bwd2Op {
    using Tr = Tr_;
    using T = typename Tr::T;
    static constexpr int UNR = UNR_, NS = 2 * Tr::NE, NS1 = NS;
    struct Params {
        const T *Q, *K, *V, *dO;
        const int32_t* t_dst;
        const float2* ld;
        T *dK, *dV;
        float* part;
        float scale, scale2;
    };
    const Params& p;
    LanePos<Tr> lp;
    RowReg<Tr> k, v;
    __device__ __forceinline__ Bwd2Op(const Params& p_, int lig) : p(p_), lp(lig) {}
    __device__ __forceinline__ void init_row(int row) {
        row_load(k, p.K + (size_t)row * Tr::F, lp);
        row_load(v, p.V + (size_t)row * Tr::F, lp);
    }
    __device__ __forceinline__ void init_state(float (&st)[NS]) {
#pragma unroll
        for (int i = 0; i < NS; ++i) st[i] = 0.f;
    }
    __device__ __forceinline__ void edges(float (&st)[NS], int i0, int end, int stride, int trips) {
        for (int t = 0; t < trips; ++t) {
            bool ok[UNR];
            RowReg<Tr> q[UNR], g[UNR];
            float2 x[UNR];
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                const int i = i0 + (t * UNR + u) * stride;
                ok[u] = i < end;
                const int r = tg_ldg_i32(p.t_dst + (ok[u] ? i : 0));
                row_load(q[u], p.Q + (size_t)r * Tr::F, lp);
                row_load(g[u], p.dO + (size_t)r * Tr::F, lp);
                x[u] = __ldg(p.ld + (size_t)r * Tr::H + lp.h);
            }
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                const float s2 = head_sum<Tr>(row_dot(q[u], k)) * p.scale2;
                const float da = head_sum<Tr>(row_dot(g[u], v));
                const float a = ok[u] ? tg_exp2(s2 - x[u].x) : 0.f;
                row_axpy(st, a * (da - x[u].y), q[u]);
                row_axpy(st + Tr::NE, a, g[u]);
            }
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
template <class Tr_, int UNR_>
struct SddmmOp {
    using Tr = Tr_;
    using T = typename Tr::T;
    static constexpr int UNR = UNR_, NS = 0, NS1 = 1;
    struct Params {
        const T *A, *B;
        const int32_t* idx;
        float* s;
        float scale;
    };
    const Params& p;
    LanePos<Tr> lp;
    RowReg<Tr> a;
    __device__ __forceinline__ SddmmOp(const Params& p_, int lig) : p(p_), lp(lig) {}
    __device__ __forceinline__ void init_row(int row) { row_load(a, p.A + (size_t)row * Tr::F, lp); }
    __device__ __forceinline__ void init_state(float (&)[1]) {}
    __device__ __forceinline__ void edges(float (&)[1], int i0, int end, int stride, int trips) {
        for (int t = 0; t < trips; ++t) {
            bool ok[UNR];
            int e[UNR];
            RowReg<Tr> b[UNR];
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                e[u] = i0 + (t * UNR + u) * stride;
                ok[u] = e[u] < end;
                const int r = tg_ldg_i32(p.idx + (ok[u] ? e[u] : 0));
                row_load(b[u], p.B + (size_t)r * Tr::F, lp);
            }
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                const float d = head_sum<Tr>(row_dot(a, b[u])) * p.scale;
                if (ok[u] && lp.j == 0) p.s[(size_t)e[u] * Tr::H + lp.h] = d;
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
template <class Tr_, int UNR_>
struct AggOp {
    using Tr = Tr_;
    using T = typename Tr::T;
    static constexpr int UNR = UNR_, NS = Tr::NE, NS1 = NS;
    struct Params {
        const T* X;
        const int32_t* idx;
        const int32_t* widx;
        const float* w;
        T* Y;
        float* part;
    };
    const Params& p;
    LanePos<Tr> lp;
    __device__ __forceinline__ AggOp(const Params& p_, int lig) : p(p_), lp(lig) {}
    __device__ __forceinline__ void init_row(int) {}
    __device__ __forceinline__ void init_state(float (&st)[NS]) {
#pragma unroll
        for (int i = 0; i < NS; ++i) st[i] = 0.f;
    }
    __device__ __forceinline__ void edges(float (&st)[NS], int i0, int end, int stride, int trips) {
        for (int t = 0; t < trips; ++t) {
            float wv[UNR];
            RowReg<Tr> x[UNR];
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                const int i = i0 + (t * UNR + u) * stride;
                const bool ok = i < end;
                const int ii = ok ? i : 0;
                const int r = tg_ldg_i32(p.idx + ii);
                row_load(x[u], p.X + (size_t)r * Tr::F, lp);
                float wgt = 1.f;
                if (p.w) {
                    const int we = p.widx ? tg_ldg_i32(p.widx + ii) : ii;
                    wgt = tg_ldg_f32(p.w + (size_t)we * Tr::H + lp.h);
                }
                wv[u] = ok ? wgt : 0.f;
            }
#pragma unroll
            for (int u = 0; u < UNR; ++u) row_axpy(st, wv[u], x[u]);
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
