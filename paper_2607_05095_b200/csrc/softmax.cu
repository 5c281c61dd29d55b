// softmax.cu -- tg_edge_softmax_fwd / tg_edge_softmax_bwd on [E, H] float32 edge tensors.
// ESM: max reduction, sum reduction, element-wise division per destination; backward
// ds = alpha*(dalpha - sum alpha*dalpha).  Tiers follow the destination-side schedule:
//   deg <= 8  : one thread per (row, head) looping over the row's edges -- the paper's CSR "thread-loop"
//               partitioning, which keeps every lane busy at small degree;
//   deg <= 64 : one warp per row, lanes stride over the flat (edge, head) range, shuffle reduction;
//   larger    : one CTA per row (launched on the row's first chunk item), shared-memory reduction.
// H must be a power of two <= 16 so that a lane / thread keeps one head for all its elements.
#include "dispatch.cuh"

template <bool BWD>
struct EsmArgs {
    const float* a;   // fwd: s        bwd: alpha
    const float* b;   // fwd: unused   bwd: dalpha
    float* out;       // fwd: alpha    bwd: ds
};

// reduce over the lanes with equal (lane % H)
template <bool MAX>
__device__ __forceinline__ float esm_lane_reduce(float x, int H) {
    for (int o = H; o < 32; o <<= 1) {
        const float y = __shfl_xor_sync(0xffffffffu, x, o);
        x = MAX ? fmaxf(x, y) : x + y;
    }
    return x;
}

template <bool MAX>
__device__ __forceinline__ float esm_cta_reduce(float x, int H, float* sm, int warp, int lane) {
    x = esm_lane_reduce<MAX>(x, H);
    __syncthreads();
    if (lane < H) sm[warp * 16 + lane] = x;
    __syncthreads();
    float r = sm[lane % H];
    for (int w = 1; w < TG_CTA_WARPS; ++w) {
        const float y = sm[w * 16 + lane % H];
        r = MAX ? fmaxf(r, y) : r + y;
    }
    return r;
}

// tier: 0 = warp-tier rows (one CTA per row, launched on every chunk item, only the first one works),
//       1 = group-tier rows of the classes > 8 (one warp per row), 2 = classes <= 8 (one thread per (row, head))
template <bool BWD>
__global__ void __launch_bounds__(TG_CTA_THREADS) tg_esm_kernel(EsmArgs<BWD> a, const int4* __restrict__ recs,
                                                                const int32_t* __restrict__ indptr, int n, int H, int tier) {
    __shared__ float sm[TG_CTA_WARPS * 16];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (tier == 0) {
        const int4 it = recs[blockIdx.x];
        const int b = indptr[it.x], e = indptr[it.x + 1];
        if (it.y != b) return;  // only the row's first chunk item works (CTA-uniform)
        const size_t lo = (size_t)b * H, hi = (size_t)e * H;
        if (!BWD) {
            float m = TG_NEG_INF;
            for (size_t i = lo + threadIdx.x; i < hi; i += TG_CTA_THREADS) m = fmaxf(m, a.a[i]);
            m = esm_cta_reduce<true>(m, H, sm, warp, lane);
            float l = 0.f;
            for (size_t i = lo + threadIdx.x; i < hi; i += TG_CTA_THREADS) l += tg_exp2((a.a[i] - m) * TG_LOG2E);
            l = esm_cta_reduce<false>(l, H, sm, warp, lane);
            const float inv = 1.f / l;
            for (size_t i = lo + threadIdx.x; i < hi; i += TG_CTA_THREADS) a.out[i] = tg_exp2((a.a[i] - m) * TG_LOG2E) * inv;
        } else {
            float d = 0.f;
            for (size_t i = lo + threadIdx.x; i < hi; i += TG_CTA_THREADS) d = fmaf(a.a[i], a.b[i], d);
            d = esm_cta_reduce<false>(d, H, sm, warp, lane);
            for (size_t i = lo + threadIdx.x; i < hi; i += TG_CTA_THREADS) a.out[i] = a.a[i] * (a.b[i] - d);
        }
    } else if (tier == 1) {
        const int idx = blockIdx.x * TG_CTA_WARPS + warp;
        if (idx >= n) return;
        const int4 it = recs[idx];
        const size_t lo = (size_t)it.y * H, hi = (size_t)it.z * H;
        if (!BWD) {
            float m = TG_NEG_INF;
            for (size_t i = lo + lane; i < hi; i += 32) m = fmaxf(m, a.a[i]);
            m = esm_lane_reduce<true>(m, H);
            float l = 0.f;
            for (size_t i = lo + lane; i < hi; i += 32) l += tg_exp2((a.a[i] - m) * TG_LOG2E);
            l = esm_lane_reduce<false>(l, H);
            const float inv = 1.f / l;
            for (size_t i = lo + lane; i < hi; i += 32) a.out[i] = tg_exp2((a.a[i] - m) * TG_LOG2E) * inv;
        } else {
            float d = 0.f;
            for (size_t i = lo + lane; i < hi; i += 32) d = fmaf(a.a[i], a.b[i], d);
            d = esm_lane_reduce<false>(d, H);
            for (size_t i = lo + lane; i < hi; i += 32) a.out[i] = a.a[i] * (a.b[i] - d);
        }
    } else {
        const int rows_per_cta = TG_CTA_THREADS / H;
        const int idx = blockIdx.x * rows_per_cta + threadIdx.x / H;
        const int h = threadIdx.x % H;
        if (idx >= n) return;
        const int4 it = recs[idx];
        const int b = it.y, e = it.z;
        if (!BWD) {
            float m = TG_NEG_INF, l = 0.f;
            for (int i = b; i < e; ++i) m = fmaxf(m, a.a[(size_t)i * H + h]);
            for (int i = b; i < e; ++i) l += tg_exp2((a.a[(size_t)i * H + h] - m) * TG_LOG2E);
            const float inv = 1.f / l;
            for (int i = b; i < e; ++i) a.out[(size_t)i * H + h] = tg_exp2((a.a[(size_t)i * H + h] - m) * TG_LOG2E) * inv;
        } else {
            float d = 0.f;
            for (int i = b; i < e; ++i) d = fmaf(a.a[(size_t)i * H + h], a.b[(size_t)i * H + h], d);
            for (int i = b; i < e; ++i) a.out[(size_t)i * H + h] = a.a[(size_t)i * H + h] * (a.b[(size_t)i * H + h] - d);
        }
    }
}

template <bool BWD>
static tg_status_t esm_launch(const tg_block* b, int H, const float* x, const float* y, float* out, cudaStream_t stream,
                              const char* name) {
    if (H < 1 || H > 16 || (H & (H - 1)) != 0) TG_FAIL(TG_ERR_UNSUPPORTED, "%s: H=%d must be a power of two <= 16", name, H);
    if (b->E == 0) return TG_OK;
    const tg_side& s = b->dst;
    EsmArgs<BWD> a{x, y, out};
    if (s.n_items > 0) {
        tg_esm_kernel<BWD><<<(unsigned)s.n_items, TG_CTA_THREADS, 0, stream>>>(a, s.items, s.indptr, s.n_items, H, 0);
        TG_LAUNCH_CHECK(name);
    }
    const int n_big = s.n_group_big(), n_small = s.n_group_small();
    if (n_big > 0) {
        tg_esm_kernel<BWD><<<(unsigned)((n_big + TG_CTA_WARPS - 1) / TG_CTA_WARPS), TG_CTA_THREADS, 0, stream>>>(a, s.rows, s.indptr, n_big, H, 1);
        TG_LAUNCH_CHECK(name);
    }
    if (n_small > 0) {
        const int rpc = TG_CTA_THREADS / H;
        tg_esm_kernel<BWD><<<(unsigned)((n_small + rpc - 1) / rpc), TG_CTA_THREADS, 0, stream>>>(a, s.rows + n_big, s.indptr, n_small, H, 2);
        TG_LAUNCH_CHECK(name);
    }
    return TG_OK;
}

extern "C" tg_status_t tg_edge_softmax_fwd(const tg_block_t* b, int H, const float* s, float* alpha, tg_stream_t stream) {
    TG_CHECK_PTR(b);
    if (b->E > 0) { TG_CHECK_PTR(s); TG_CHECK_PTR(alpha); }
    return esm_launch<false>(b, H, s, nullptr, alpha, static_cast<cudaStream_t>(stream), "tg_edge_softmax_fwd");
}

extern "C" tg_status_t tg_edge_softmax_bwd(const tg_block_t* b, int H, const float* alpha, const float* dalpha, float* ds,
                                           tg_stream_t stream) {
    TG_CHECK_PTR(b);
    if (b->E > 0) { TG_CHECK_PTR(alpha); TG_CHECK_PTR(dalpha); TG_CHECK_PTR(ds); }
    return esm_launch<true>(b, H, alpha, dalpha, ds, static_cast<cudaStream_t>(stream), "tg_edge_softmax_bwd");
}
