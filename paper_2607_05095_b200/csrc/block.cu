// block.cu -- tg_block_build: the compression engine's triple uni_ID / inv_Idx / CSR ind_ptr
// (§4.2, §5), the transposed CSR for the backward gather, and the internal
// degree-tier schedules.  All integer work, exactly one correct result (readings R7-R10).
//
// Device pipeline, no library sort, ONE host synchronisation (to return U):
//   1. one pass over the sampler lists: range / sortedness flags, min / max of the neighbour ids, the 32- or 64-bit
//      sort keys, and -- for destination-sorted input (what a sampler emits) -- indptr by boundary fill and perm = iota;
//      unsorted input: integer-atomic histogram + scan for indptr, stable radix sort of (root_idx, position) for perm,
//      then the CSR-order gathers
//   2. dedup: stable radix sort (radix_sort.cuh) of (neighbour key, CSR position) over exactly the bits the ids need
//      -> t_edge; head flags -> scan with fused emit -> kv_row, uniq_node, t_indptr, t_dst     (identity mode: iota)
//   3. schedules for both CSR sides (scan with fused classification / list emission); the source side's row count U is
//      still on the device then: its launches are sized for the bound E and read U from device memory
//   4. one D2H of {flags, U, both schedules' totals}, one cudaStreamSynchronize
// What the host cannot know before step 4 (is the input sorted? how many bits do the ids need?) is SPECULATED from the
// previous call of this thread and verified in step 4; a wrong guess re-runs the build once with the measured values.
#include <atomic>
#include "dispatch.cuh"
#include "scan.cuh"
#include "radix_sort.cuh"

// ---------------------------------------------------------------------------------------------
// Schedules
// ---------------------------------------------------------------------------------------------
// scan vector: [0, TG_NCLS) group-tier class counts, then warp items per length class (TG_NICLS), partial slots, hubs.
// Warp items are stored by length class, longest first -- class 0: chunks of multi-chunk rows (chunk/2 < len <= chunk),
// then single-chunk rows in classes of a factor sqrt(2) in length -- so that the 8 warps of a CTA finish together (the CTA's registers are
// held until its slowest warp ends: unsorted items left 30 % of the resident warp slots idle on config 4).
constexpr int TG_NICLS = 7;
constexpr int TG_SK = TG_NCLS + TG_NICLS + 3;   // ... partial slots, hubs, big hubs (> TG_HUB_DIRECT chunks)
__host__ __device__ constexpr int tg_item_class(int deg, int chunk) {
    if (deg > chunk) return 0;
    int c = 1;   // single-chunk rows: one class per factor sqrt(2) of length (181/256 ~ 1/sqrt 2)
    for (int t = chunk; c < TG_NICLS - 1; ++c) {
        t = (c & 1) ? (chunk >> (c >> 1)) * 181 >> 8 : chunk >> (c >> 1);
        if (deg > t) break;
    }
    return c;
}

struct SchedIn {
    const int32_t* indptr;
    int chunk;
    int n_edges;
    int group_max;   // rows up to this degree go to the group tier (tg_side::group_max)
    __device__ __forceinline__ IVec<TG_SK> operator()(int64_t i) const {
        int deg = indptr[i + 1] - indptr[i];
        if (deg < 0 || deg > n_edges) deg = 0;   // only a speculative build on unsorted input sees such an indptr (block.cu header)
        IVec<TG_SK> x = ivec_zero<TG_SK>();
        if (deg <= group_max) {
            x.v[tg_degree_class(deg)] = 1;
        } else {
            const int chunks = (deg + chunk - 1) / chunk;
            x.v[TG_NCLS + tg_item_class(deg, chunk)] = chunks;
            x.v[TG_NCLS + TG_NICLS] = chunks > 1 ? chunks : 0;
            x.v[TG_NCLS + TG_NICLS + 1] = chunks > 1;
            x.v[TG_NCLS + TG_NICLS + 2] = chunks > TG_HUB_DIRECT;
        }
        return x;
    }
};
struct SchedOut {
    const int32_t* indptr;
    int chunk;
    int4* rows;
    int4* items;
    int4* hubs;
    int4* bighubs;
    int* max_deg;
    int n_edges;
    int group_max;
    int64_t rows_cap, items_cap, hubs_cap, bighubs_cap;   // a speculative build may scan a garbage indptr: never write past the lists
    __device__ __forceinline__ void operator()(int64_t i, const IVec<TG_SK>& ex, const IVec<TG_SK>& x, const IVec<TG_SK>& tot) const {
        const int row = (int)i;
        const int b = indptr[i];
        int e = indptr[i + 1];
        if (e < b || e - b > n_edges) e = b;
        const int ic = tg_item_class(e - b, chunk);
        const int chunks = (e - b > group_max) ? x.v[TG_NCLS + ic] : 0;
        if (chunks == 0) {
            const int c = tg_degree_class(e - b);
            int pos = ex.v[c];
            for (int cc = c + 1; cc < TG_NCLS; ++cc) pos += tot.v[cc];  // larger classes come first
            if (pos >= 0 && pos < rows_cap) rows[pos] = make_int4(row, b, e, 0);
        } else {
            const int len = (e - b + chunks - 1) / chunks;
            int base = ex.v[TG_NCLS + ic];
            for (int cc = 0; cc < ic; ++cc) base += tot.v[TG_NCLS + cc];  // longer classes come first
            for (int c = 0; c < chunks; ++c) {
                const int cb = min(b + c * len, e), ce = min(cb + len, e);
                if (base + c >= 0 && base + c < items_cap) items[base + c] = make_int4(row, cb, ce, chunks > 1 ? ex.v[TG_NCLS + TG_NICLS] + c : -1);
            }
            const int hi = ex.v[TG_NCLS + TG_NICLS + 1], bi = ex.v[TG_NCLS + TG_NICLS + 2];
            if (chunks > 1 && hi >= 0 && hi < hubs_cap) hubs[hi] = make_int4(row, ex.v[TG_NCLS + TG_NICLS], chunks, 0);
            if (chunks > TG_HUB_DIRECT && bi >= 0 && bi < bighubs_cap) bighubs[bi] = make_int4(row, ex.v[TG_NCLS + TG_NICLS], chunks, 0);
        }
        if (e - b > 8) atomicMax(max_deg, e - b);
    }
};

// a warp-tier row (deg > group_max >= TG_GROUP_MAX_SMALL) has ceil(deg / chunk) <= deg / TG_CHUNK_MIN + 1 items
static inline int64_t side_items_bound(int64_t n_edges) { return n_edges / TG_CHUNK_MIN + n_edges / TG_GROUP_MAX_SMALL + 2; }
static inline int64_t side_hubs_bound(int64_t n_edges) { return n_edges / TG_CHUNK_MIN + 1; }
static inline int64_t side_bighubs_bound(int64_t n_edges) { return n_edges / (TG_CHUNK_MIN * TG_HUB_DIRECT) + 1; }

size_t tg_side_bytes(int64_t n_rows_bound, int64_t n_edges) {
    return tg_align_up((size_t)(n_rows_bound + 1) * sizeof(int4)) + tg_align_up((size_t)side_items_bound(n_edges) * sizeof(int4)) +
           tg_align_up((size_t)side_hubs_bound(n_edges) * sizeof(int4)) + tg_align_up((size_t)side_bighubs_bound(n_edges) * sizeof(int4)) +
           tg_scan_bytes<TG_SK>(n_rows_bound) + 512;
}

// Launch half: enqueues the schedule scan of one side; totals (IVec<TG_SK> + max_deg) land at `totals_dev` (TG_SK + 1 ints,
// zeroed by the caller).  n_rows is the bound the launches are sized for; n_rows_dev (nullable) the real count on the device.
static tg_status_t tg_side_launch(tg_side* s, int64_t n_rows, const int* n_rows_dev, int64_t n_edges, const int32_t* indptr, void* ws,
                                  size_t ws_bytes, int* totals_dev, cudaStream_t stream) {
    *s = tg_side();
    s->n_rows = n_rows; s->n_edges = n_edges; s->indptr = indptr;
    if (n_rows == 0) return TG_OK;
    tg_carver c(ws, ws_bytes);
    s->rows = static_cast<int4*>(c.take((size_t)(n_rows + 1) * sizeof(int4)));
    s->items = static_cast<int4*>(c.take((size_t)side_items_bound(n_edges) * sizeof(int4)));
    s->hubs = static_cast<int4*>(c.take((size_t)side_hubs_bound(n_edges) * sizeof(int4)));
    s->bighubs = static_cast<int4*>(c.take((size_t)side_bighubs_bound(n_edges) * sizeof(int4)));
    void* scan_tmp = c.take(tg_scan_bytes<TG_SK>(n_rows));
    if (!c.ok()) TG_FAIL(TG_ERR_WORKSPACE, "schedule workspace too small: need %zu, have %zu", c.off, ws_bytes);
    // about 4 warp items per resident warp slot (148 SMs x 16 warps) when the side is small, TG_CHUNK_MAX beyond
    int chunk = TG_CHUNK_MIN;
    while (chunk < TG_CHUNK_MAX && n_edges / chunk > 148 * 16 * 4) chunk *= 2;
    s->chunk = chunk;
    // A launch-bound small side is limited by its longest single-group chain (one edge per trip, one gather latency per
    // trip): rows above 32 edges go to the warp tier there (config 3: 62 -> 55 us per step, config 2: 113 -> 100 us; 16 costs the destination side more than it saves), where the four groups of a warp share the row.
    s->group_max = n_edges < TG_FORK_MIN_EDGES ? TG_GROUP_MAX_SMALL : TG_GROUP_MAX;
    SchedIn in{indptr, chunk, (int)n_edges, s->group_max};
    SchedOut out{indptr, chunk, s->rows, s->items, s->hubs, s->bighubs, totals_dev + TG_SK, (int)n_edges, s->group_max,
                 n_rows + 1, side_items_bound(n_edges), side_hubs_bound(n_edges), side_bighubs_bound(n_edges)};
    TG_TRY((tg_scan<TG_SK>(n_rows, in, out, scan_tmp, reinterpret_cast<IVec<TG_SK>*>(totals_dev), stream, n_rows_dev)));
    return TG_OK;
}
// Host half: the totals have arrived.
static void tg_side_finish(tg_side* s, int64_t n_rows, const int* h) {
    s->n_rows = n_rows;
    s->n_group = 0;
    for (int k = 0; k < TG_NCLS; ++k) { s->n_cls[k] = h[k]; s->n_group += h[k]; }
    s->n_items = 0;
    for (int k = 0; k < TG_NICLS; ++k) s->n_items += h[TG_NCLS + k];
    s->n_slots = h[TG_NCLS + TG_NICLS]; s->n_hubs = h[TG_NCLS + TG_NICLS + 1]; s->n_bighubs = h[TG_NCLS + TG_NICLS + 2];
    s->max_deg = h[TG_SK];
}

tg_status_t tg_side_build(tg_side* s, int64_t n_rows, int64_t n_edges, const int32_t* indptr, void* ws, size_t ws_bytes,
                          cudaStream_t stream) {
    *s = tg_side();
    s->n_rows = n_rows; s->n_edges = n_edges; s->indptr = indptr;
    if (n_rows == 0) return TG_OK;
    tg_carver c(ws, ws_bytes);
    int* totals = static_cast<int*>(c.take(256));  // IVec<TG_SK> + max_deg at [TG_SK]
    if (!c.ok()) TG_FAIL(TG_ERR_WORKSPACE, "schedule workspace too small");
    TG_CUDA(cudaMemsetAsync(totals, 0, 256, stream));
    TG_TRY(tg_side_launch(s, n_rows, nullptr, n_edges, indptr, static_cast<char*>(ws) + c.off, ws_bytes - c.off, totals, stream));
    int h[TG_SK + 1];
    TG_CUDA(cudaMemcpyAsync(h, totals, sizeof(h), cudaMemcpyDeviceToHost, stream));
    TG_CUDA(cudaStreamSynchronize(stream));
    tg_side_finish(s, n_rows, h);
    return TG_OK;
}

// ---------------------------------------------------------------------------------------------
// Build kernels
// ---------------------------------------------------------------------------------------------
// Everything the host learns from a build, fetched by the single D2H copy at its end.
struct BuildFlags {
    int bad_root;     // some root_idx outside [0, R)
    int unsorted;     // root_idx is not non-decreasing
    long long nbr_min, nbr_max;
    int U;            // unique source rows (IVec<1> total of the dedup scan)
    int pad;
    int dst_tot[TG_SK + 1];   // schedule totals of the destination side (+ max_deg)
    int src_tot[TG_SK + 1];   // ... of the source side
    int long_gap;     // sorted input with a run of >= TG_FILL_CAP empty rows: indptr comes from tg_fill_indptr_by_search
};

// sort key of a neighbour id: 32-bit when all ids fit [0, 2^32), else 64-bit with the sign bit flipped (signed order)
template <class K> __device__ __forceinline__ K tg_make_key(long long id);
template <> __device__ __forceinline__ uint32_t tg_make_key<uint32_t>(long long id) { return (uint32_t)id; }
template <> __device__ __forceinline__ uint64_t tg_make_key<uint64_t>(long long id) { return (uint64_t)id ^ 0x8000000000000000ULL; }
template <class K> __device__ __forceinline__ long long tg_key_id(K k);
template <> __device__ __forceinline__ long long tg_key_id<uint32_t>(uint32_t k) { return (long long)k; }
template <> __device__ __forceinline__ long long tg_key_id<uint64_t>(uint64_t k) { return (long long)(k ^ 0x8000000000000000ULL); }

// One pass over the sampler lists: flags, min / max of the ids and, if SORTED (root_idx non-decreasing -- verified by the
// flags), the whole CSR: indptr by boundary fill (indptr[v] = e for every v in (root[e-1], root[e]]), perm = iota, the
// pass-through arrays, the dedup sort keys.  !SORTED: flags only (the CSR comes from the root sort).
template <class K, bool SORTED>
__global__ void k_scan_lists(int64_t R, int64_t E, const int32_t* __restrict__ root, const int64_t* __restrict__ nbr,
                             const int64_t* __restrict__ eid, const float* __restrict__ ts, BuildFlags* f, int32_t* indptr,
                             int32_t* perm, K* keys, int64_t* eid_csr, float* ts_csr) {
    int bad = 0, uns = 0;
    long long mn = 0x7fffffffffffffffLL, mx = -0x7fffffffffffffffLL - 1;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e <= E; e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t prev = (e == 0) ? -1 : (int64_t)root[e - 1];
        const int64_t cur = (e == E) ? R : (int64_t)root[e];
        if (e < E) {
            bad |= (cur < 0 || cur >= R);
            uns |= (prev > cur);
            const long long x = nbr[e];
            mn = min(mn, x); mx = max(mx, x);
            if (SORTED) {
                perm[e] = (int32_t)e;
                if (keys) keys[e] = tg_make_key<K>(x);
                if (eid_csr) eid_csr[e] = eid[e];
                if (ts_csr) ts_csr[e] = ts[e];
            }
        }
        if (SORTED) {   // garbage in, nothing out: an out-of-range or unsorted input writes no indptr entry out of bounds
            const int64_t lo = max(prev + 1, (int64_t)0), hi = min(cur, R);
            if (hi - lo >= TG_FILL_CAP) f->long_gap = 1;   // a long run of empty rows: left to the search kernel (all rows)
            else for (int64_t v = lo; v <= hi; ++v) indptr[v] = (int32_t)e;
        }
    }
    bad = __reduce_or_sync(0xffffffffu, bad);
    uns = __reduce_or_sync(0xffffffffu, uns);
    for (int o = 16; o > 0; o >>= 1) {
        mn = min(mn, __shfl_xor_sync(0xffffffffu, mn, o));
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if ((threadIdx.x & 31) == 0) {
        if (bad) atomicOr(&f->bad_root, 1);
        if (uns) atomicOr(&f->unsorted, 1);
        atomicMin(&f->nbr_min, mn);
        atomicMax(&f->nbr_max, mx);
    }
}

__global__ void k_hist(int64_t R, int64_t E, const int32_t* __restrict__ root, int32_t* cnt, uint32_t* root_keys) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < E; e += (int64_t)gridDim.x * blockDim.x) {
        const int r = root[e];
        if (r >= 0 && r < R) atomicAdd(&cnt[r], 1);
        root_keys[e] = (uint32_t)r;
    }
}

// unsorted input: CSR-order gathers through perm
template <class K>
__global__ void k_gather_csr(int64_t E, const int32_t* __restrict__ perm, const int32_t* __restrict__ root,
                             const int64_t* __restrict__ nbr, const int64_t* __restrict__ eid, const float* __restrict__ ts,
                             K* keys, int64_t* nbr_csr, int32_t* edge_dst, int64_t* eid_csr, float* ts_csr) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < E; e += (int64_t)gridDim.x * blockDim.x) {
        const int p = perm[e];
        const long long x = nbr[p];
        if (keys) keys[e] = tg_make_key<K>(x);
        if (nbr_csr) nbr_csr[e] = x;
        edge_dst[e] = root[p];
        if (eid_csr) eid_csr[e] = eid[p];
        if (ts_csr) ts_csr[e] = ts[p];
    }
}

// identity mode: K/V are per-edge rows
__global__ void k_identity(int64_t E, const int32_t* __restrict__ perm, const int32_t* __restrict__ root, const int64_t* __restrict__ nbr,
                           int32_t* kv_row, int64_t* uniq, int32_t* t_indptr, int32_t* t_edge, int32_t* t_dst) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e <= E; e += (int64_t)gridDim.x * blockDim.x) {
        t_indptr[e] = (int32_t)e;
        if (e < E) {
            const int p = perm[e];
            kv_row[e] = (int32_t)e; t_edge[e] = (int32_t)e; t_dst[e] = root[p]; uniq[e] = nbr[p];
        }
    }
}

struct CntIn {
    const int32_t* cnt;
    __device__ __forceinline__ IVec<1> operator()(int64_t i) const { IVec<1> x; x.v[0] = cnt[i]; return x; }
};
struct IndptrOut {
    int32_t* indptr;
    int64_t R;
    __device__ __forceinline__ void operator()(int64_t i, const IVec<1>& ex, const IVec<1>& x, const IVec<1>& tot) const {
        indptr[i] = ex.v[0];
        if (i == R - 1) indptr[R] = tot.v[0];
    }
};

template <class K>
struct HeadIn {
    const K* skeys;
    __device__ __forceinline__ IVec<1> operator()(int64_t j) const {
        IVec<1> x;
        x.v[0] = (j == 0) || (skeys[j] != skeys[j - 1]);
        return x;
    }
};
template <class K>
struct DedupOut {
    const K* skeys;
    const int32_t* t_edge;
    const int32_t* edge_dst;   // destination of CSR edge e
    int32_t* kv_row;
    int64_t* uniq;
    int32_t* t_indptr;
    int32_t* t_dst;
    int64_t E;
    __device__ __forceinline__ void operator()(int64_t j, const IVec<1>& ex, const IVec<1>& x, const IVec<1>& tot) const {
        const int row = ex.v[0] + x.v[0] - 1;
        const int e = t_edge[j];
        kv_row[e] = row;
        t_dst[j] = edge_dst[e];
        if (x.v[0]) { uniq[row] = tg_key_id<K>(skeys[j]); t_indptr[row] = (int32_t)j; }
        if (j == E - 1) t_indptr[tot.v[0]] = (int32_t)E;
    }
};

static inline int grid_for(int64_t n) {
    int64_t g = (n + 255) / 256;
    if (g < 1) g = 1;
    if (g > 148 * 16) g = 148 * 16;
    return (int)g;
}

static inline int bits_for(uint64_t x) {
    int b = 0;
    while (x) { ++b; x >>= 1; }
    return b < 1 ? 1 : b;
}

struct BuildWs {
    BuildFlags* flags;
    int32_t* cnt;       // [R+1]              unsorted input only
    void* keys_a;       // [E] x 8 bytes      sort keys (32- or 64-bit)
    void* keys_b;       // [E] x 8 bytes
    int32_t* vals_a;    // [E]
    int32_t* vals_b;    // [E]
    int32_t* edge_dst;  // [E]                unsorted input only (sorted input: root_idx itself)
    void* scan_tmp;
    void* rs_tmp;
    void* side_dst;
    size_t side_dst_bytes;
    void* side_src;
    size_t side_src_bytes;
};

static tg_status_t build_ws_layout(int64_t R, int64_t E, int dedup_mode, tg_carver& c, BuildWs* w) {
    // schedules first: they persist for the lifetime of the block
    w->side_dst_bytes = tg_side_bytes(R, E);
    w->side_dst = c.take(w->side_dst_bytes);
    w->side_src_bytes = tg_side_bytes(E, E);
    w->side_src = c.take(w->side_src_bytes);
    w->flags = static_cast<BuildFlags*>(c.take(sizeof(BuildFlags)));
    w->cnt = static_cast<int32_t*>(c.take((size_t)(R + 1) * 4));
    w->keys_a = c.take((size_t)E * 8);
    w->keys_b = c.take((size_t)E * 8);
    w->vals_a = static_cast<int32_t*>(c.take((size_t)E * 4));
    w->vals_b = static_cast<int32_t*>(c.take((size_t)E * 4));
    w->edge_dst = static_cast<int32_t*>(c.take((size_t)E * 4));
    w->scan_tmp = c.take(tg_scan_bytes<1>(E > R ? E : R));
    const size_t r32 = tg_rs_bytes<uint32_t>(E), r64 = tg_rs_bytes<uint64_t>(E);
    w->rs_tmp = c.take(r32 > r64 ? r32 : r64);
    (void)dedup_mode;
    return TG_OK;
}

extern "C" tg_status_t tg_block_workspace_bytes(int64_t R, int64_t E, int dedup_mode, size_t* bytes) {
    if (!bytes) TG_FAIL(TG_ERR_INVALID_ARG, "bytes is null");
    if (R < 0 || E < 0 || R > TG_MAX_INDEX || E > TG_MAX_INDEX) TG_FAIL(TG_ERR_INVALID_ARG, "R=%lld E=%lld out of range", (long long)R, (long long)E);
    tg_carver c(nullptr, 0);
    BuildWs w;
    TG_TRY(build_ws_layout(R, E, dedup_mode, c, &w));
    *bytes = c.off + 256;
    return TG_OK;
}

extern "C" tg_status_t tg_sched_workspace_bytes(int64_t R, int64_t E, int64_t U, size_t* bytes) {
    if (!bytes) TG_FAIL(TG_ERR_INVALID_ARG, "bytes is null");
    if (R < 0 || E < 0 || U < 0) TG_FAIL(TG_ERR_INVALID_ARG, "negative size");
    *bytes = tg_align_up(tg_side_bytes(R, E)) + tg_align_up(tg_side_bytes(U, E)) + 256;
    return TG_OK;
}

extern "C" tg_status_t tg_block_from_csr(int64_t R, int64_t E, int64_t U, const int32_t* indptr, const int32_t* kv_row,
                                         const int32_t* t_indptr, const int32_t* t_edge, const int32_t* t_dst, void* workspace,
                                         size_t workspace_bytes, tg_stream_t stream_, tg_block_t** out) {
    if (!out) TG_FAIL(TG_ERR_INVALID_ARG, "out is null");
    *out = nullptr;
    if (R < 0 || E < 0 || U < 0 || U > E || R > TG_MAX_INDEX || E > TG_MAX_INDEX)
        TG_FAIL(TG_ERR_INVALID_ARG, "bad sizes R=%lld E=%lld U=%lld", (long long)R, (long long)E, (long long)U);
    if (!indptr) TG_FAIL(TG_ERR_INVALID_ARG, "indptr is null");
    if (E > 0 && (!kv_row || !t_indptr || !t_edge || !t_dst)) TG_FAIL(TG_ERR_INVALID_ARG, "null index array");
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    tg_carver c(workspace, workspace_bytes);
    const size_t bd = tg_side_bytes(R, E), bs = tg_side_bytes(U, E);
    void* wd = c.take(bd);
    void* wsrc = c.take(bs);
    if (!c.ok()) TG_FAIL(TG_ERR_WORKSPACE, "schedule workspace: need %zu bytes, have %zu", c.off, workspace_bytes);
    tg_block* b = new tg_block();
    b->R = R; b->E = E; b->U = U;
    b->indptr = indptr; b->kv_row = kv_row; b->t_indptr = t_indptr; b->t_edge = t_edge; b->t_dst = t_dst;
    tg_status_t st = tg_side_build(&b->dst, R, E, indptr, wd, bd, stream);
    if (st == TG_OK && U > 0) st = tg_side_build(&b->src, U, E, t_indptr, wsrc, bs, stream);
    if (st != TG_OK) { delete b; return st; }
    *out = b;
    return TG_OK;
}

struct BuildArgs {
    int64_t R, E;
    const int32_t* root_idx; const int64_t* nbr_node; const int64_t* edge_id; const float* ts;
    int dedup_mode;
    int32_t *indptr, *perm, *kv_row; int64_t* uniq_node; int32_t *t_indptr, *t_edge, *t_dst;
    int64_t* eid_csr; float* ts_csr;
};

// One attempt under the assumptions (unsorted?, key width K, key bits); every launch is enqueued, then ONE D2H + sync.
template <class K>
static tg_status_t build_attempt(const BuildArgs& a, const BuildWs& w, bool assume_unsorted, int bits, tg_block* b, BuildFlags* fh,
                                 cudaStream_t stream) {
    const int64_t R = a.R, E = a.E;
    BuildFlags f0;
    memset(&f0, 0, sizeof(f0));
    f0.nbr_min = 0x7fffffffffffffffLL; f0.nbr_max = -0x7fffffffffffffffLL - 1;
    TG_CUDA(cudaMemcpyAsync(w.flags, &f0, sizeof(f0), cudaMemcpyHostToDevice, stream));
    K* keys_a = static_cast<K*>(w.keys_a);
    K* keys_b = static_cast<K*>(w.keys_b);
    const int32_t* edge_dst = a.root_idx;   // destination of CSR edge e (sorted input: the root list itself)
    // 1. lists -> CSR
    if (!assume_unsorted) {
        k_scan_lists<K, true><<<grid_for(E + 1), 256, 0, stream>>>(R, E, a.root_idx, a.nbr_node, a.edge_id, a.ts, w.flags, a.indptr, a.perm,
                                                                    a.dedup_mode ? keys_a : nullptr, a.eid_csr, a.ts_csr);
        TG_LAUNCH_CHECK("k_scan_lists");
        tg_fill_indptr_by_search<int32_t, int32_t><<<grid_for(R + 1), 256, 0, stream>>>(E, R, a.root_idx, a.indptr, &w.flags->long_gap);
        TG_LAUNCH_CHECK("tg_fill_indptr_by_search");
    } else {
        k_scan_lists<K, false><<<grid_for(E + 1), 256, 0, stream>>>(R, E, a.root_idx, a.nbr_node, a.edge_id, a.ts, w.flags, nullptr, nullptr,
                                                                     nullptr, nullptr, nullptr);
        TG_LAUNCH_CHECK("k_scan_lists");
        TG_CUDA(cudaMemsetAsync(w.cnt, 0, (size_t)(R + 1) * 4, stream));
        uint32_t* rk_a = static_cast<uint32_t*>(w.keys_a);
        uint32_t* rk_b = static_cast<uint32_t*>(w.keys_b);
        k_hist<<<grid_for(E), 256, 0, stream>>>(R, E, a.root_idx, w.cnt, rk_a);
        TG_LAUNCH_CHECK("k_hist");
        TG_TRY((tg_scan<1>(R, CntIn{w.cnt}, IndptrOut{a.indptr, R}, w.scan_tmp, reinterpret_cast<IVec<1>*>(&w.flags->pad), stream)));
        const int rbits = bits_for((uint64_t)(R - 1));
        const bool odd = tg_rs_passes(rbits) & 1;     // the last pass must write perm
        uint32_t* kres; int32_t* vres;
        TG_TRY((tg_radix_sort<uint32_t>(E, rbits, rk_a, odd ? w.vals_a : a.perm, true, rk_b, odd ? a.perm : w.vals_b, &kres, &vres, w.rs_tmp, stream)));
        if (vres != a.perm) TG_FAIL(TG_ERR_INTERNAL, "root sort landed in the wrong buffer");
        k_gather_csr<K><<<grid_for(E), 256, 0, stream>>>(E, a.perm, a.root_idx, a.nbr_node, a.edge_id, a.ts, a.dedup_mode ? keys_a : nullptr,
                                                         nullptr, w.edge_dst, a.eid_csr, a.ts_csr);
        TG_LAUNCH_CHECK("k_gather_csr");
        edge_dst = w.edge_dst;
    }
    // The destination side's schedule only needs indptr: on a large block it runs on an auxiliary stream beside the dedup sort
    // (plain event fork / join, as in tiers.cuh; 0.83 -> 0.79 ms per build on config 4).
    b->R = R; b->E = E;
    b->indptr = a.indptr; b->kv_row = a.kv_row; b->t_indptr = a.t_indptr; b->t_edge = a.t_edge; b->t_dst = a.t_dst;
    tg_aux_streams* aux = (E >= TG_FORK_MIN_EDGES && a.dedup_mode) ? tg_get_aux_streams() : nullptr;
    if (aux) {
        TG_CUDA(cudaEventRecord(aux->fork, stream));
        TG_CUDA(cudaStreamWaitEvent(aux->s[0], aux->fork, 0));
    }
    tg_status_t st_dst = tg_side_launch(&b->dst, R, nullptr, E, a.indptr, w.side_dst, w.side_dst_bytes, w.flags->dst_tot, aux ? aux->s[0] : stream);
    // steps 2 and 3 run on `stream` meanwhile; the auxiliary stream is joined whatever they return
    const tg_status_t st_main = [&]() -> tg_status_t {
        // 2. unique rows + transposed CSR
        if (a.dedup_mode == 0) {
            k_identity<<<grid_for(E + 1), 256, 0, stream>>>(E, a.perm, a.root_idx, a.nbr_node, a.kv_row, a.uniq_node, a.t_indptr, a.t_edge, a.t_dst);
            TG_LAUNCH_CHECK("k_identity");
        } else {
            const bool odd = tg_rs_passes(bits) & 1;      // the last pass must write t_edge
            K* kres; int32_t* vres;
            TG_TRY((tg_radix_sort<K>(E, bits, keys_a, odd ? w.vals_a : a.t_edge, true, keys_b, odd ? a.t_edge : w.vals_b, &kres, &vres, w.rs_tmp, stream)));
            if (vres != a.t_edge) TG_FAIL(TG_ERR_INTERNAL, "dedup sort landed in the wrong buffer");
            DedupOut<K> dout{kres, a.t_edge, edge_dst, a.kv_row, a.uniq_node, a.t_indptr, a.t_dst, E};
            TG_TRY((tg_scan<1>(E, HeadIn<K>{kres}, dout, w.scan_tmp, reinterpret_cast<IVec<1>*>(&w.flags->U), stream)));
        }
        // 3. the source side's schedule (its row count is still on the device)
        return tg_side_launch(&b->src, E, a.dedup_mode ? &w.flags->U : nullptr, E, a.t_indptr, w.side_src, w.side_src_bytes, w.flags->src_tot, stream);
    }();
    if (aux) {
        const bool ok = cudaEventRecord(aux->join[0], aux->s[0]) == cudaSuccess && cudaStreamWaitEvent(stream, aux->join[0], 0) == cudaSuccess;
        if (!ok && st_dst == TG_OK) { tg_set_error("tg_block_build: joining the auxiliary stream failed"); st_dst = TG_ERR_CUDA; }
    }
    TG_TRY(st_dst);
    TG_TRY(st_main);
    // 4. the one round trip
    TG_CUDA(cudaMemcpyAsync(fh, w.flags, sizeof(BuildFlags), cudaMemcpyDeviceToHost, stream));
    TG_CUDA(cudaStreamSynchronize(stream));
    b->U = a.dedup_mode ? fh->U : E;
    tg_side_finish(&b->dst, R, fh->dst_tot);
    tg_side_finish(&b->src, b->U, fh->src_tot);
    return TG_OK;
}

// What the recent builds of this thread found: the speculation of the next one.  The hint is sticky: it keeps the
// largest key width seen recently (in whole 8-bit radix passes) and "unsorted" from any recent build, and gives them up
// only after TG_HINT_PATIENCE consecutive builds that needed less.  A thread that alternates between blocks with
// different needs (16- and 17-bit node ids, sorted and shuffled lists) then pays one unneeded radix pass, or a sort of
// sorted input, on the smaller ones instead of building the larger ones twice.  tg_block_build_retries() counts the
// builds that were repeated because the speculation was too optimistic.
constexpr int TG_HINT_PATIENCE = 8;
struct BuildHint {
    int bits = 24;
    bool unsorted = false;
    int narrower_streak = 0, narrower_max = 0;   // consecutive builds that needed fewer passes, and the most they needed
    int sorted_streak = 0;
    void observe(int need_bits /* < 0: this build sorted no neighbour keys */, bool was_unsorted) {
        const int need = need_bits >= 64 ? 64 : (need_bits + 7) / 8 * 8;
        if (need_bits < 0) {}
        else if (need >= bits) { bits = need; narrower_streak = 0; narrower_max = 0; }
        else {
            narrower_max = need > narrower_max ? need : narrower_max;
            if (++narrower_streak >= TG_HINT_PATIENCE) { bits = narrower_max; narrower_streak = 0; narrower_max = 0; }
        }
        if (was_unsorted) { unsorted = true; sorted_streak = 0; }
        else if (unsorted && ++sorted_streak >= TG_HINT_PATIENCE) { unsorted = false; sorted_streak = 0; }
    }
};
static thread_local BuildHint g_hint;
static std::atomic<unsigned long long> g_build_retries{0};
extern "C" unsigned long long tg_block_build_retries(void) { return g_build_retries.load(std::memory_order_relaxed); }

extern "C" tg_status_t tg_block_build(int64_t R, int64_t E, const int32_t* root_idx, const int64_t* nbr_node,
                                      const int64_t* edge_id, const float* ts, int dedup_mode, int32_t* indptr, int32_t* perm,
                                      int32_t* kv_row, int64_t* uniq_node, int32_t* t_indptr, int32_t* t_edge, int32_t* t_dst,
                                      int64_t* eid_csr, float* ts_csr, int64_t* U_host, void* workspace, size_t workspace_bytes,
                                      tg_stream_t stream_, tg_block_t** out) {
    if (!out || !U_host) TG_FAIL(TG_ERR_INVALID_ARG, "out / U_host is null");
    *out = nullptr;
    *U_host = 0;
    if (R < 0 || E < 0 || R > TG_MAX_INDEX || E > TG_MAX_INDEX) TG_FAIL(TG_ERR_INVALID_ARG, "R=%lld E=%lld out of range", (long long)R, (long long)E);
    if (dedup_mode != 0 && dedup_mode != 1) TG_FAIL(TG_ERR_INVALID_ARG, "dedup_mode must be 0 or 1");
    if (!indptr || !t_indptr) TG_FAIL(TG_ERR_INVALID_ARG, "indptr / t_indptr is null");
    if (E > 0 && (!root_idx || !nbr_node || !perm || !kv_row || !uniq_node || !t_edge || !t_dst)) TG_FAIL(TG_ERR_INVALID_ARG, "null index array");
    if (E > 0 && R == 0) TG_FAIL(TG_ERR_INVALID_ARG, "E > 0 with R == 0");
    if ((eid_csr && !edge_id) || (ts_csr && !ts)) TG_FAIL(TG_ERR_INVALID_ARG, "eid_csr / ts_csr need edge_id / ts");
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    tg_carver c(workspace, workspace_bytes);
    BuildWs w;
    TG_TRY(build_ws_layout(R, E, dedup_mode, c, &w));
    if (!c.ok()) TG_FAIL(TG_ERR_WORKSPACE, "block workspace: need %zu bytes, have %zu", c.off, workspace_bytes);

    tg_block* b = new tg_block();
    tg_status_t st = TG_OK;
    if (E == 0) {
        b->R = R; b->E = 0; b->U = 0;
        b->indptr = indptr; b->kv_row = kv_row; b->t_indptr = t_indptr; b->t_edge = t_edge; b->t_dst = t_dst;
        cudaError_t e = cudaMemsetAsync(indptr, 0, (size_t)(R + 1) * 4, stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(t_indptr, 0, 4, stream);
        if (e != cudaSuccess) { tg_set_error("tg_block_build: %s", cudaGetErrorString(e)); st = TG_ERR_CUDA; }
        if (st == TG_OK) st = tg_side_build(&b->dst, R, 0, indptr, w.side_dst, w.side_dst_bytes, stream);   // all rows are degree 0
    } else {
        BuildArgs a{R, E, root_idx, nbr_node, edge_id, ts, dedup_mode, indptr, perm, kv_row, uniq_node, t_indptr, t_edge, t_dst, eid_csr, ts_csr};
        bool unsorted = g_hint.unsorted;
        int bits = g_hint.bits;
        for (int attempt = 0; attempt < 3; ++attempt) {
            BuildFlags fh;
            st = (bits <= 32) ? build_attempt<uint32_t>(a, w, unsorted, bits, b, &fh, stream)
                              : build_attempt<uint64_t>(a, w, unsorted, bits, b, &fh, stream);
            if (st != TG_OK) break;
            if (fh.bad_root) { tg_set_error("root_idx has an entry outside [0, R)"); st = TG_ERR_INVALID_ARG; break; }
            const bool wide = fh.nbr_min < 0 || fh.nbr_max > 0xffffffffLL;
            const int need = wide ? 64 : bits_for((uint64_t)fh.nbr_max);
            const bool ok = (unsorted || !fh.unsorted) && (dedup_mode == 0 || bits >= need);
            g_hint.observe(dedup_mode ? need : -1, fh.unsorted != 0);   // identity rows sort no neighbour keys: no evidence on the width
            if (ok) break;
            // the speculation was wrong: once more with what this pass measured (never less than was speculated)
            g_build_retries.fetch_add(1, std::memory_order_relaxed);
            unsorted = unsorted || fh.unsorted != 0;
            bits = need > bits ? need : bits;
            if (attempt == 2) { tg_set_error("tg_block_build: speculation did not converge"); st = TG_ERR_INTERNAL; }
        }
    }
    if (st != TG_OK) { delete b; return st; }
    *U_host = b->U;
    *out = b;
    return TG_OK;
}

extern "C" tg_status_t tg_block_destroy(tg_block_t* b) {
    delete b;
    return TG_OK;
}

extern "C" tg_status_t tg_block_sched_info(const tg_block_t* b, int64_t out[8]) {
    TG_CHECK_PTR(b);
    if (!out) TG_FAIL(TG_ERR_INVALID_ARG, "tg_block_sched_info: out is null");
    const tg_side* sides[2] = {&b->dst, &b->src};
    for (int i = 0; i < 2; ++i) {
        out[4 * i + 0] = sides[i]->group_max; out[4 * i + 1] = sides[i]->chunk;
        out[4 * i + 2] = sides[i]->n_hubs;    out[4 * i + 3] = sides[i]->max_deg;
    }
    return TG_OK;
}

extern "C" tg_status_t tg_block_info(const tg_block_t* b, int64_t* R, int64_t* E, int64_t* U, int64_t stats[8]) {
    TG_CHECK_PTR(b);
    if (R) *R = b->R;
    if (E) *E = b->E;
    if (U) *U = b->U;
    if (stats) {
        stats[0] = b->dst.n_group_small(); stats[1] = b->dst.n_group_big(); stats[2] = b->dst.n_items; stats[3] = b->dst.n_slots;
        stats[4] = b->src.n_group_small(); stats[5] = b->src.n_group_big(); stats[6] = b->src.n_items; stats[7] = b->src.n_slots;
    }
    return TG_OK;
}
