// softmax.cu -- tg_edge_softmax_fwd / tg_edge_softmax_bwd on [E, H] float32 edge tensors.
// ESM: max reduction, sum reduction, element-wise division per destination; backward
// ds = alpha*(dalpha - sum alpha*dalpha).  Tiers follow the destination-side schedule:
//   small rows: one thread per (row, head) looping over the row's edges -- the paper's CSR "thread-loop"
//               partitioning, which keeps every lane busy at degree <= 8;
//   warp rows : one warp per row, lanes stride over the flat (edge, head) range, shuffle reduction;
//   cta rows  : one CTA per row (launched on the row's first chunk item), shared-memory reduction.
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

template <bool BWD>
__global__ void __launch_bounds__(TG_CTA_THREADS) tg_esm_kernel(EsmArgs<BWD> a, SideDev sd, int H, int nb_warp) {
    __shared__ float sm[TG_CTA_WARPS * 16];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int bid = blockIdx.x;
    if (bid < sd.n_items) {
        const int4 it = sd.items[bid];
        const int b = sd.indptr[it.x], e = sd.indptr[it.x + 1];
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
    } else if ((bid -= sd.n_items) < nb_warp) {
        const int idx = bid * TG_CTA_WARPS + warp;
        if (idx >= sd.n_warp) return;
        const int row = sd.order[sd.n_small + idx];
        const size_t lo = (size_t)sd.indptr[row] * H, hi = (size_t)sd.indptr[row + 1] * H;
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
        bid -= nb_warp;
        const int rows_per_cta = TG_CTA_THREADS / H;
        const int idx = bid * rows_per_cta + threadIdx.x / H;
        const int h = threadIdx.x % H;
        if (idx >= sd.n_small) return;
        const int row = sd.order[idx];
        const int b = sd.indptr[row], e = sd.indptr[row + 1];
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
    SideDev sd = tg_side_dev(s);
    const int nb_warp = (s.n_warp + TG_CTA_WARPS - 1) / TG_CTA_WARPS;
    const int rpc = TG_CTA_THREADS / H;
    const int nb_small = (s.n_small + rpc - 1) / rpc;
    const long long grid = (long long)s.n_items + nb_warp + nb_small;
    EsmArgs<BWD> a{x, y, out};
    if (grid > 0) {
        tg_esm_kernel<BWD><<<(unsigned)grid, TG_CTA_THREADS, 0, stream>>>(a, sd, H, nb_warp);
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
