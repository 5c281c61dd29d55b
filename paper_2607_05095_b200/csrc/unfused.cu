// unfused.cu -- tg_sddmm, tg_aggregate_fwd, tg_aggregate_bwd.
//   SDDMM  (gSDDMM named at PAPER.md:94):  s[e,h] = scale * <A[v(e)], B[r(e)]>
//   AGG:                 Y[v] = sum_{N(v)} w[e,h] * X[r(e)],  w == NULL: plain sum
//   AGG backward:           dX[u] = sum_{r(e)=u} w[e,h] * dY[v(e)] by gather over the
//                                          transposed CSR (the paper's COO atomics, PAPER.md:219-223,
//                                          are not used);  dw[e,h] = <dY[v(e)], X[r(e)]> = SDDMM(dY, X).
#include "dispatch.cuh"

// one edge per trip, 32 resident warps in the warp tier: these operators carry little state, occupancy hides the gathers
// (unfused chain on config 4: 3.98 ms with the fused kernels' policy, 2.95 ms with this one)
using UnfPolicy = TierPolicy<1, 2, 1, 3, 1, 32, true>;

struct SddmmArgs {
    const tg_block* b;
    const void *A, *B;
    float scale;
    float* s;
    cudaStream_t stream;
};
template <class Tr>
struct SddmmFn {
    static tg_status_t run(const SddmmArgs& a) {
        using Op = SddmmOp<Tr>;
        using T = typename Tr::T;
        typename Op::Params p;
        p.A = static_cast<const T*>(a.A); p.B = static_cast<const T*>(a.B);
        p.idx = a.b->kv_row; p.s = a.s; p.scale = a.scale;
        return tg_launch_tiers<Op, UnfPolicy>(p, a.b->dst, a.stream, "tg_sddmm");
    }
};

struct AggArgs {
    const tg_side* side;
    const void* X;
    const int32_t *idx, *widx;
    const float* w;
    void* Y;
    float* part;
    cudaStream_t stream;
};
template <class Tr>
struct AggFn {
    static tg_status_t run(const AggArgs& a) {
        using Op = AggOp<Tr>;
        using T = typename Tr::T;
        typename Op::Params p;
        p.X = static_cast<const T*>(a.X); p.idx = a.idx; p.widx = a.widx; p.w = a.w;
        p.Y = static_cast<T*>(a.Y); p.part = a.part;
        return tg_launch_tiers<Op, UnfPolicy>(p, *a.side, a.stream, "tg_aggregate");
    }
};

extern "C" tg_status_t tg_sddmm(const tg_block_t* b, int H, int D, tg_dtype_t dtype, const void* A, const void* B, float scale,
                                float* s, tg_stream_t stream) {
    TG_CHECK_PTR(b);
    if (!tg_shape_supported(H, D, dtype)) TG_FAIL(TG_ERR_UNSUPPORTED, "unsupported (H=%d, D=%d, dtype=%d)", H, D, (int)dtype);
    if (b->E == 0) return TG_OK;
    TG_CHECK_ROWS(A); TG_CHECK_ROWS(B); TG_CHECK_PTR(s);
    SddmmArgs a{b, A, B, scale, s, static_cast<cudaStream_t>(stream)};
    return tg_dispatch<SddmmFn>(H, D, dtype, a);
}

extern "C" tg_status_t tg_aggregate_fwd(const tg_block_t* b, int H, int D, tg_dtype_t dtype, const float* w, const void* X,
                                        void* Y, void* ws, size_t ws_bytes, tg_stream_t stream) {
    TG_CHECK_PTR(b);
    if (!tg_shape_supported(H, D, dtype)) TG_FAIL(TG_ERR_UNSUPPORTED, "unsupported (H=%d, D=%d, dtype=%d)", H, D, (int)dtype);
    if (b->R == 0) return TG_OK;
    TG_CHECK_ROWS(Y);
    if (b->E > 0) TG_CHECK_ROWS(X);
    tg_geom g;
    TG_TRY(tg_get_geom(H, D, dtype, &g));
    const size_t need = tg_part_slots(b->dst) * g.NE * g.LPR * sizeof(float);
    if (need > 0 && (!ws || ws_bytes < need)) TG_FAIL(TG_ERR_WORKSPACE, "aggregate fwd needs %zu workspace bytes", need);
    AggArgs a{&b->dst, X, b->kv_row, nullptr, w, Y, static_cast<float*>(ws), static_cast<cudaStream_t>(stream)};
    return tg_dispatch<AggFn>(H, D, dtype, a);
}

extern "C" tg_status_t tg_aggregate_bwd(const tg_block_t* b, int H, int D, tg_dtype_t dtype, const float* w, const void* X,
                                        const void* dY, void* dX, float* dw, void* ws, size_t ws_bytes, tg_stream_t stream) {
    TG_CHECK_PTR(b);
    if (!tg_shape_supported(H, D, dtype)) TG_FAIL(TG_ERR_UNSUPPORTED, "unsupported (H=%d, D=%d, dtype=%d)", H, D, (int)dtype);
    if (b->E == 0) return TG_OK;   // U == 0: nothing to write
    TG_CHECK_ROWS(dY); TG_CHECK_ROWS(dX);
    if (dw) TG_CHECK_ROWS(X);
    tg_geom g;
    TG_TRY(tg_get_geom(H, D, dtype, &g));
    const size_t need = tg_part_slots(b->src) * g.NE * g.LPR * sizeof(float);
    if (need > 0 && (!ws || ws_bytes < need)) TG_FAIL(TG_ERR_WORKSPACE, "aggregate bwd needs %zu workspace bytes", need);
    AggArgs a{&b->src, dY, b->t_dst, b->t_edge, w, dX, static_cast<float*>(ws), static_cast<cudaStream_t>(stream)};
    TG_TRY(tg_dispatch<AggFn>(H, D, dtype, a));
    if (dw) {
        SddmmArgs sa{b, dY, X, 1.0f, dw, static_cast<cudaStream_t>(stream)};
        TG_TRY(tg_dispatch<SddmmFn>(H, D, dtype, sa));
    }
    return TG_OK;
}
