// scan.cuh -- exclusive prefix sum of K-component int vectors with fused input / output functors.
// Three launches: per-tile reduce, single-CTA spine, per-tile scan + output.  Integer, exact.
//   In  : IVec<K> operator()(int64_t i)
//   Out : void operator()(int64_t i, const IVec<K>& exclusive_prefix, const IVec<K>& value, const IVec<K>& total)
#pragma once
#include "common.cuh"

template <int K>
struct IVec {
    int v[K];
};

constexpr int TG_SCAN_THREADS = 256;
constexpr int TG_SCAN_ITEMS = 4;
constexpr int TG_SCAN_TILE = TG_SCAN_THREADS * TG_SCAN_ITEMS;

template <int K>
__device__ __forceinline__ void ivec_add(IVec<K>& a, const IVec<K>& b) {
#pragma unroll
    for (int k = 0; k < K; ++k) a.v[k] += b.v[k];
}
template <int K>
__device__ __forceinline__ IVec<K> ivec_zero() {
    IVec<K> z;
#pragma unroll
    for (int k = 0; k < K; ++k) z.v[k] = 0;
    return z;
}

// CTA-wide exclusive scan of one IVec per thread; returns the exclusive prefix, `total` = CTA sum.
template <int K, int THREADS>
__device__ __forceinline__ IVec<K> cta_exclusive_scan(IVec<K> x, IVec<K>& total, IVec<K>* sm /*[THREADS/32]*/) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    IVec<K> inc = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const int y = __shfl_up_sync(0xffffffffu, inc.v[k], o);
            if (lane >= o) inc.v[k] += y;
        }
    }
    __syncthreads();
    if (lane == 31) sm[warp] = inc;
    __syncthreads();
    IVec<K> base = ivec_zero<K>();
    total = ivec_zero<K>();
    for (int w = 0; w < THREADS / 32; ++w) {
        if (w < warp) ivec_add(base, sm[w]);
        ivec_add(total, sm[w]);
    }
    IVec<K> ex;
#pragma unroll
    for (int k = 0; k < K; ++k) ex.v[k] = base.v[k] + inc.v[k] - x.v[k];
    return ex;
}

template <int K, class In>
__global__ void __launch_bounds__(TG_SCAN_THREADS) tg_scan_reduce(int64_t n, const int* __restrict__ n_dev, In in, IVec<K>* tile_sums) {
    __shared__ IVec<K> sm[TG_SCAN_THREADS / 32];
    if (n_dev) n = min(n, (int64_t)*n_dev);   // the launch was sized for the bound n; tiles past the real end sum to zero
    if ((int64_t)blockIdx.x * TG_SCAN_TILE >= n) return;   // whole CTA; the spine stops at the real end too
    const int64_t base = (int64_t)blockIdx.x * TG_SCAN_TILE + (int64_t)threadIdx.x * TG_SCAN_ITEMS;
    IVec<K> s = ivec_zero<K>();
#pragma unroll
    for (int i = 0; i < TG_SCAN_ITEMS; ++i)
        if (base + i < n) ivec_add(s, in(base + i));
    IVec<K> total;
    cta_exclusive_scan<K, TG_SCAN_THREADS>(s, total, sm);
    if (threadIdx.x == 0) tile_sums[blockIdx.x] = total;
}

template <int K>
__global__ void __launch_bounds__(1024) tg_scan_spine(int64_t n_tiles, const int* __restrict__ n_dev, IVec<K>* tile_sums, IVec<K>* total_out) {
    __shared__ IVec<K> sm[32];
    if (n_dev) n_tiles = min(n_tiles, ((int64_t)*n_dev + TG_SCAN_TILE - 1) / TG_SCAN_TILE);   // tiles past the real end are not read by anyone
    IVec<K> carry = ivec_zero<K>();
    for (int64_t base = 0; base < n_tiles; base += 1024) {
        const int64_t i = base + threadIdx.x;
        IVec<K> x = (i < n_tiles) ? tile_sums[i] : ivec_zero<K>();
        IVec<K> total;
        IVec<K> ex = cta_exclusive_scan<K, 1024>(x, total, sm);
        ivec_add(ex, carry);
        if (i < n_tiles) tile_sums[i] = ex;
        ivec_add(carry, total);
        __syncthreads();
    }
    if (threadIdx.x == 0) *total_out = carry;
}

template <int K, class In, class Out>
__global__ void __launch_bounds__(TG_SCAN_THREADS) tg_scan_down(int64_t n, const int* __restrict__ n_dev, In in, const IVec<K>* tile_sums, const IVec<K>* total_in, Out out) {
    __shared__ IVec<K> sm[TG_SCAN_THREADS / 32];
    if (n_dev) n = min(n, (int64_t)*n_dev);
    if ((int64_t)blockIdx.x * TG_SCAN_TILE >= n) return;   // whole CTA: no barrier is skipped by a part of it
    const int64_t base = (int64_t)blockIdx.x * TG_SCAN_TILE + (int64_t)threadIdx.x * TG_SCAN_ITEMS;
    IVec<K> x[TG_SCAN_ITEMS];
    IVec<K> s = ivec_zero<K>();
#pragma unroll
    for (int i = 0; i < TG_SCAN_ITEMS; ++i) {
        x[i] = (base + i < n) ? in(base + i) : ivec_zero<K>();
        ivec_add(s, x[i]);
    }
    IVec<K> cta_total;
    IVec<K> ex = cta_exclusive_scan<K, TG_SCAN_THREADS>(s, cta_total, sm);
    ivec_add(ex, tile_sums[blockIdx.x]);
    const IVec<K> total = *total_in;
#pragma unroll
    for (int i = 0; i < TG_SCAN_ITEMS; ++i) {
        if (base + i < n) out(base + i, ex, x[i], total);
        ivec_add(ex, x[i]);
    }
}

template <int K>
static inline size_t tg_scan_bytes(int64_t n) {
    const int64_t tiles = (n + TG_SCAN_TILE - 1) / TG_SCAN_TILE;
    return tg_align_up((size_t)(tiles + 1) * sizeof(IVec<K>)) + 256;
}

// `tmp` holds tg_scan_bytes<K>(n); the grand total is left at `total_dev` (device).  n_dev (nullable): the real length
// lives on the device (<= n, the bound the launches are sized for) -- lets a caller chain scans without a host round trip.
template <int K, class In, class Out>
static tg_status_t tg_scan(int64_t n, In in, Out out, void* tmp, IVec<K>* total_dev, cudaStream_t stream, const int* n_dev = nullptr) {
    const int64_t tiles = (n + TG_SCAN_TILE - 1) / TG_SCAN_TILE;
    IVec<K>* sums = static_cast<IVec<K>*>(tmp);
    if (tiles > 0x7fffffffLL) TG_FAIL(TG_ERR_INTERNAL, "scan too large");
    if (tiles > 0) {
        tg_scan_reduce<K, In><<<(unsigned)tiles, TG_SCAN_THREADS, 0, stream>>>(n, n_dev, in, sums);
        TG_LAUNCH_CHECK("tg_scan_reduce");
    }
    tg_scan_spine<K><<<1, 1024, 0, stream>>>(tiles, n_dev, sums, total_dev);
    TG_LAUNCH_CHECK("tg_scan_spine");
    if (tiles > 0) {
        tg_scan_down<K, In, Out><<<(unsigned)tiles, TG_SCAN_THREADS, 0, stream>>>(n, n_dev, in, sums, total_dev, out);
        TG_LAUNCH_CHECK("tg_scan_down");
    }
    return TG_OK;
}

// ---------------------------------------------------------------------------------------------
// Boundary fill of a CSR indptr from sorted keys.  The single-pass builders (block.cu k_scan_lists, sampler.cu
// k_tcsr_emit) let the thread that sees a key boundary write indptr for the rows in between: fine for the few empty
// rows of a dense batch, a serial loop of up to n_rows stores when one long run of rows is empty (n_rows >> n, or an
// empty tail).  They therefore fill only gaps shorter than TG_FILL_CAP and raise a flag otherwise; this kernel, launched
// behind them, returns at once unless the flag is set and then writes every row by binary search:
// indptr[x] = number of keys below x, x in [0, n_rows].  Unsorted keys give in-range garbage, never a stray write.
// ---------------------------------------------------------------------------------------------
constexpr int TG_FILL_CAP = 32;
template <class KeyT, class PtrT>
__global__ void __launch_bounds__(256) tg_fill_indptr_by_search(int64_t n, int64_t n_rows, const KeyT* __restrict__ keys,
                                                                PtrT* __restrict__ indptr, const int* __restrict__ enable) {
    if (*enable == 0) return;
    for (int64_t x = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; x <= n_rows; x += (int64_t)gridDim.x * blockDim.x) {
        int64_t lo = 0, hi = n;   // first position whose key is >= x
        while (lo < hi) {
            const int64_t mid = (lo + hi) >> 1;
            if ((int64_t)keys[mid] < x) lo = mid + 1; else hi = mid;
        }
        indptr[x] = (PtrT)lo;
    }
}
