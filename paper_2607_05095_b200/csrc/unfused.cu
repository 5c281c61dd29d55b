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

// ---------------------------------------------------------------------------------------------
// The paper's own AGG partitioning, as the measured alternative: COO, edge-centric,
// "each thread handles one edge independently ... a single atomic update to global memory".
// One thread per (edge, 4-element vector): Y[scatter[e]] += X[gather[e]] with one red.global.add.v4.f32.
//   forward  (h_v = sum v_u): gather = kv_row, scatter = the edge's destination
//   backward               : gather = the edge's destination, scatter = kv_row
// Y is float32 (the accumulation target of the atomics) and is zeroed by the call.  Float atomics: the summation order,
// hence the last bits, change from run to run -- unlike tg_aggregate_fwd / _bwd.
// ---------------------------------------------------------------------------------------------
__global__ void k_coo_dst(int64_t R, const int32_t* __restrict__ indptr, int32_t* coo_dst) {
    // one warp per destination row: writes the row id over the row's edge range
    const int64_t row = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (row >= R) return;
    const int b = indptr[row], e = indptr[row + 1];
    for (int i = b + lane; i < e; i += 32) coo_dst[i] = (int32_t)row;
}

template <typename T>
__global__ void __launch_bounds__(256) k_coo_scatter_add(int64_t E, int F4, const int32_t* __restrict__ gather,
                                                         const int32_t* __restrict__ scatter, const T* __restrict__ X, float* Y) {
    const int64_t n = E * F4;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t e = i / F4;
        const int j = (int)(i - e * F4);
        const int64_t src = (int64_t)gather[e] * F4 + j, dst = (int64_t)scatter[e] * F4 + j;
        float4 x;
        if constexpr (sizeof(T) == 4) {
            x = reinterpret_cast<const float4*>(X)[src];
        } else {
            const uint2 w = reinterpret_cast<const uint2*>(X)[src];
            x = make_float4(tg_bf16lo(w.x), tg_bf16hi(w.x), tg_bf16lo(w.y), tg_bf16hi(w.y));
        }
        asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(Y + dst * 4), "f"(x.x), "f"(x.y), "f"(x.z), "f"(x.w) : "memory");
    }
}

extern "C" tg_status_t tg_block_coo_dst(const tg_block_t* b, int32_t* coo_dst, tg_stream_t stream_) {
    TG_CHECK_PTR(b);
    if (b->E == 0) return TG_OK;
    TG_CHECK_PTR(coo_dst);
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const int64_t threads = b->R * 32;
    k_coo_dst<<<(unsigned)((threads + 255) / 256), 256, 0, stream>>>(b->R, b->indptr, coo_dst);
    TG_LAUNCH_CHECK("tg_block_coo_dst");
    return TG_OK;
}

extern "C" tg_status_t tg_aggregate_coo(const tg_block_t* b, int H, int D, tg_dtype_t dtype, int backward, const int32_t* coo_dst,
                                        const void* X, float* Y, tg_stream_t stream_) {
    TG_CHECK_PTR(b);
    if (dtype != TG_F32 && dtype != TG_BF16) TG_FAIL(TG_ERR_UNSUPPORTED, "dtype %d", (int)dtype);
    const int F = H * D;
    if (H < 1 || D < 1 || F % 4 != 0) TG_FAIL(TG_ERR_UNSUPPORTED, "tg_aggregate_coo needs H*D to be a multiple of 4 (H=%d, D=%d)", H, D);
    const int64_t out_rows = backward ? b->U : b->R;
    if (out_rows == 0) return TG_OK;
    TG_CHECK_ROWS(Y);
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    TG_CUDA(cudaMemsetAsync(Y, 0, (size_t)out_rows * F * sizeof(float), stream));
    if (b->E == 0) return TG_OK;
    TG_CHECK_ROWS(X); TG_CHECK_PTR(coo_dst);
    const int32_t* gather = backward ? coo_dst : b->kv_row;
    const int32_t* scatter = backward ? b->kv_row : coo_dst;
    const int64_t n = b->E * (F / 4);
    const unsigned grid = (unsigned)((n + 255) / 256 < 148 * 64 ? (n + 255) / 256 : 148 * 64);
    if (dtype == TG_F32) k_coo_scatter_add<float><<<grid, 256, 0, stream>>>(b->E, F / 4, gather, scatter, static_cast<const float*>(X), Y);
    else k_coo_scatter_add<__nv_bfloat16><<<grid, 256, 0, stream>>>(b->E, F / 4, gather, scatter, static_cast<const __nv_bfloat16*>(X), Y);
    TG_LAUNCH_CHECK("tg_aggregate_coo");
    return TG_OK;
}
