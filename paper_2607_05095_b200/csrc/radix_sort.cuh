// radix_sort.cuh -- stable LSD radix sort of (key, int32 value) pairs, 8 bits per pass, written for the block build
// (group-by-destination, sorted-unique of neighbour ids, transposed CSR) and the T-CSR build of the
// sampler.  Integer work, exactly one correct result: a stable sort.
//
// One pass = three steps:
//   tg_rs_hist     per-tile digit counts              counts[digit * n_tiles + tile]
//   tg_scan<1>     exclusive scan of that array (digit-major): the global base of every (digit, tile)
//   tg_rs_scatter  per tile: stable rank of every key among the keys of its digit, tile reordered in shared memory,
//                  written out in runs (one run per digit), so the global stores are coalesced
// Stable rank inside a tile: the tile is cut into per-warp segments; a warp walks its segment 32 keys at a time in index
// order and ranks equal digits with __match_any_sync; per-warp digit counters live in shared memory; segment order =
// warp order, so rank = (keys of that digit in earlier warps) + (warp-local rank).
// The first pass can synthesise the values (value = position: iota) instead of reading them.
#pragma once
#include "scan.cuh"

constexpr int TG_RS_BITS = 8;
constexpr int TG_RS_BINS = 1 << TG_RS_BITS;
constexpr int TG_RS_THREADS = 256;
constexpr int TG_RS_WARPS = TG_RS_THREADS / 32;
#ifndef TG_RS_ITEMS32
#define TG_RS_ITEMS32 8
#endif
#ifndef TG_RS_MINB
#define TG_RS_MINB 4
#endif
template <class K> struct RsTile { static constexpr int ITEMS = sizeof(K) == 4 ? TG_RS_ITEMS32 : 12; static constexpr int TILE = TG_RS_THREADS * ITEMS; };

template <class K>
__device__ __forceinline__ int tg_rs_digit(K key, int shift) { return (int)((key >> shift) & (K)(TG_RS_BINS - 1)); }

template <class K>
__global__ void __launch_bounds__(TG_RS_THREADS) tg_rs_hist(int64_t n, const K* __restrict__ keys, int shift, int n_tiles, int32_t* __restrict__ counts) {
    __shared__ int h[TG_RS_BINS];
    constexpr int TILE = RsTile<K>::TILE;
    h[threadIdx.x] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * TILE;
    // plain shared-memory atomics: warp-aggregating them with __match_any_sync was measured slower (41.7 vs 27.6 us per pass on
    // config 4), even with a key that holds 18 % of the edges
    for (int i = threadIdx.x; i < TILE; i += TG_RS_THREADS) {
        const int64_t g = base + i;
        if (g < n) atomicAdd(&h[tg_rs_digit(keys[g], shift)], 1);
    }
    __syncthreads();
    counts[(int64_t)threadIdx.x * n_tiles + blockIdx.x] = h[threadIdx.x];
}

struct RsCntIn {
    const int32_t* c;
    __device__ __forceinline__ IVec<1> operator()(int64_t i) const { IVec<1> x; x.v[0] = c[i]; return x; }
};
struct RsBaseOut {
    int32_t* b;
    __device__ __forceinline__ void operator()(int64_t i, const IVec<1>& ex, const IVec<1>&, const IVec<1>&) const { b[i] = ex.v[0]; }
};

template <class K, bool IOTA>
__global__ void __launch_bounds__(TG_RS_THREADS, TG_RS_MINB) tg_rs_scatter(int64_t n, const K* __restrict__ keys_in, const int32_t* __restrict__ vals_in,
                                                               K* __restrict__ keys_out, int32_t* __restrict__ vals_out, int shift, int n_tiles,
                                                               const int32_t* __restrict__ base) {
    constexpr int ITEMS = RsTile<K>::ITEMS, TILE = RsTile<K>::TILE;
    __shared__ int wcnt[TG_RS_WARPS][TG_RS_BINS];     // per-warp digit counts, then exclusive prefix over warps
    __shared__ int dbase[TG_RS_BINS];                 // tile-local start of every digit's run
    __shared__ int gbase[TG_RS_BINS];                 // global start of this tile's run of every digit
    __shared__ K skey[TILE];
    __shared__ int32_t sval[TILE];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t tile0 = (int64_t)blockIdx.x * TILE;
    for (int i = threadIdx.x; i < TG_RS_WARPS * TG_RS_BINS; i += TG_RS_THREADS) (&wcnt[0][0])[i] = 0;
    gbase[threadIdx.x] = base[(int64_t)threadIdx.x * n_tiles + blockIdx.x];
    __syncthreads();
    // warp `warp` owns tile positions [warp*32*ITEMS, (warp+1)*32*ITEMS); step k covers 32 consecutive positions
    K key[ITEMS];
    int32_t val[ITEMS];
    int rank[ITEMS];
    const unsigned lt = (1u << lane) - 1u;
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        const int64_t g = tile0 + (warp * ITEMS + k) * 32 + lane;
        const bool ok = g < n;
        key[k] = ok ? keys_in[g] : (K)0;
        val[k] = ok ? (IOTA ? (int32_t)g : vals_in[g]) : 0;
    }
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        const int64_t g = tile0 + (warp * ITEMS + k) * 32 + lane;
        const bool ok = g < n;
        const int d = tg_rs_digit(key[k], shift);
        // positions past the end only occur at the tail of the last tile: they get a private pseudo-digit and are dropped
        const unsigned peers = __match_any_sync(0xffffffffu, ok ? d : (TG_RS_BINS + lane));
        const int leader = __ffs(peers) - 1;
        int old = 0;
        if (ok && lane == leader) { old = wcnt[warp][d]; wcnt[warp][d] = old + __popc(peers); }
        old = __shfl_sync(0xffffffffu, old, leader);
        rank[k] = ok ? old + __popc(peers & lt) : -1;
        __syncwarp();
    }
    __syncthreads();
    {   // thread d: prefix over the warps for digit d, then the tile-local start of every digit
        const int d = threadIdx.x;
        int run = 0;
#pragma unroll
        for (int w = 0; w < TG_RS_WARPS; ++w) { const int c = wcnt[w][d]; wcnt[w][d] = run; run += c; }
        __shared__ IVec<1> sm[TG_RS_THREADS / 32];
        IVec<1> x, tot;
        x.v[0] = run;
        const IVec<1> ex = cta_exclusive_scan<1, TG_RS_THREADS>(x, tot, sm);
        dbase[d] = ex.v[0];
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        if (rank[k] >= 0) {
            const int d = tg_rs_digit(key[k], shift);
            const int p = dbase[d] + wcnt[warp][d] + rank[k];
            skey[p] = key[k];
            sval[p] = val[k];
        }
    }
    __syncthreads();
    const int n_here = (int)min((int64_t)TILE, n - tile0);
    for (int i = threadIdx.x; i < n_here; i += TG_RS_THREADS) {
        const K kk = skey[i];
        const int d = tg_rs_digit(kk, shift);
        const int64_t o = (int64_t)gbase[d] + (i - dbase[d]);
        keys_out[o] = kk;
        vals_out[o] = sval[i];
    }
}

template <class K>
static inline int64_t tg_rs_tiles(int64_t n) { return (n + RsTile<K>::TILE - 1) / RsTile<K>::TILE; }

// scratch of one sort: counts + bases [256 * tiles] each, the scan's own scratch
template <class K>
static inline size_t tg_rs_bytes(int64_t n) {
    const int64_t t = tg_rs_tiles<K>(n);
    return 2 * tg_align_up((size_t)TG_RS_BINS * (size_t)(t + 1) * 4) + tg_scan_bytes<1>(TG_RS_BINS * (t + 1)) + 512;
}

// Sorts n pairs by the key bits [0, bits).  keys_a / vals_a hold the input (iota: the values are the positions and
// vals_a is only scratch); the passes ping-pong between (keys_a, vals_a) and (keys_b, vals_b); the result lands in
// (*keys_res, *vals_res): the b buffers after an odd number of passes (tg_rs_passes), the a buffers after an even one.
// All four buffers hold n elements and are overwritten.  bits <= 0 sorts nothing.
static inline int tg_rs_passes(int bits) { return bits <= 0 ? 0 : (bits + TG_RS_BITS - 1) / TG_RS_BITS; }

template <class K>
static tg_status_t tg_radix_sort(int64_t n, int bits, K* keys_a, int32_t* vals_a, bool iota, K* keys_b, int32_t* vals_b,
                                 K** keys_res, int32_t** vals_res, void* scratch, cudaStream_t stream) {
    K* kin = keys_a; K* kout = keys_b;
    int32_t* vin = vals_a; int32_t* vout = vals_b;
    if (n > 0 && bits > 0) {
        const int64_t tiles = tg_rs_tiles<K>(n);
        if (tiles * TG_RS_BINS > 0x7fffffffLL) TG_FAIL(TG_ERR_INTERNAL, "radix sort too large");
        tg_carver c(scratch, (size_t)-1);
        int32_t* counts = static_cast<int32_t*>(c.take((size_t)TG_RS_BINS * (size_t)(tiles + 1) * 4));
        int32_t* base = static_cast<int32_t*>(c.take((size_t)TG_RS_BINS * (size_t)(tiles + 1) * 4));
        void* scan_tmp = c.take(tg_scan_bytes<1>(TG_RS_BINS * (tiles + 1)));
        IVec<1>* total = static_cast<IVec<1>*>(c.take(256));
        const int passes = (bits + TG_RS_BITS - 1) / TG_RS_BITS;
        for (int p = 0; p < passes; ++p) {
            const int shift = p * TG_RS_BITS;
            tg_rs_hist<K><<<(unsigned)tiles, TG_RS_THREADS, 0, stream>>>(n, kin, shift, (int)tiles, counts);
            TG_LAUNCH_CHECK("tg_rs_hist");
            TG_TRY((tg_scan<1>(TG_RS_BINS * tiles, RsCntIn{counts}, RsBaseOut{base}, scan_tmp, total, stream)));
            if (p == 0 && iota)
                tg_rs_scatter<K, true><<<(unsigned)tiles, TG_RS_THREADS, 0, stream>>>(n, kin, nullptr, kout, vout, shift, (int)tiles, base);
            else
                tg_rs_scatter<K, false><<<(unsigned)tiles, TG_RS_THREADS, 0, stream>>>(n, kin, vin, kout, vout, shift, (int)tiles, base);
            TG_LAUNCH_CHECK("tg_rs_scatter");
            K* tk = kin; kin = kout; kout = tk;
            int32_t* tv = vin;
            vin = vout; vout = tv;
        }
    }
    *keys_res = kin;
    *vals_res = vin;
    return TG_OK;
}
