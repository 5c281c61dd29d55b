// block.cu -- tg_block_build: the compression engine's triple uni_ID / inv_Idx / CSR ind_ptr
// (§4.2, §5), the transposed CSR for the backward gather, and the internal
// degree-tier schedules.  All integer work, exactly one correct result (readings R7-R10).
//
// Device pipeline:
//   1. check root_idx range + sortedness, min/max of neighbour ids            (1 launch, tiny D2H)
//   2. indptr: sorted input -> boundary fill; else integer-atomic histogram + scan
//   3. perm:   sorted input -> iota; else stable LSD radix sort of (root_idx, position)
//   4. gather nbr/edge_id/ts into CSR order
//   5. dedup:  stable radix sort of (nbr_csr, CSR position) -> t_edge; head flags -> scan ->
//              kv_row, uniq_node, t_indptr, t_dst                             (identity mode: iota)
//   6. schedules for both CSR sides (scan with fused classification / list emission)
// The radix sort is cub::DeviceRadixSort (ships with the CUDA toolkit; compiled into this library).
#include <cub/device/device_radix_sort.cuh>

#include "dispatch.cuh"
#include "scan.cuh"

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
    __device__ __forceinline__ IVec<TG_SK> operator()(int64_t i) const {
        const int deg = indptr[i + 1] - indptr[i];
        IVec<TG_SK> x = ivec_zero<TG_SK>();
        if (deg <= TG_GROUP_MAX) {
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
    __device__ __forceinline__ void operator()(int64_t i, const IVec<TG_SK>& ex, const IVec<TG_SK>& x, const IVec<TG_SK>& tot) const {
        const int row = (int)i;
        const int b = indptr[i], e = indptr[i + 1];
        const int ic = tg_item_class(e - b, chunk);
        const int chunks = (e - b > TG_GROUP_MAX) ? x.v[TG_NCLS + ic] : 0;
        if (chunks == 0) {
            const int c = tg_degree_class(e - b);
            int pos = ex.v[c];
            for (int cc = c + 1; cc < TG_NCLS; ++cc) pos += tot.v[cc];  // larger classes come first
            rows[pos] = make_int4(row, b, e, 0);
        } else {
            const int len = (e - b + chunks - 1) / chunks;
            int base = ex.v[TG_NCLS + ic];
            for (int cc = 0; cc < ic; ++cc) base += tot.v[TG_NCLS + cc];  // longer classes come first
            for (int c = 0; c < chunks; ++c) {
                const int cb = min(b + c * len, e), ce = min(cb + len, e);
                items[base + c] = make_int4(row, cb, ce, chunks > 1 ? ex.v[TG_NCLS + TG_NICLS] + c : -1);
            }
            if (chunks > 1) hubs[ex.v[TG_NCLS + TG_NICLS + 1]] = make_int4(row, ex.v[TG_NCLS + TG_NICLS], chunks, 0);
            if (chunks > TG_HUB_DIRECT) bighubs[ex.v[TG_NCLS + TG_NICLS + 2]] = make_int4(row, ex.v[TG_NCLS + TG_NICLS], chunks, 0);
        }
        if (e - b > 8) atomicMax(max_deg, e - b);
    }
};

// a warp-tier row (deg > TG_GROUP_MAX) has ceil(deg / chunk) <= deg / TG_CHUNK_MIN + 1 <= 2 * deg / TG_GROUP_MAX items
static inline int64_t side_items_bound(int64_t n_edges) { return 2 * (n_edges / TG_GROUP_MAX) + 2; }
static inline int64_t side_hubs_bound(int64_t n_edges) { return n_edges / TG_CHUNK_MIN + 1; }
static inline int64_t side_bighubs_bound(int64_t n_edges) { return n_edges / (TG_CHUNK_MIN * TG_HUB_DIRECT) + 1; }

size_t tg_side_bytes(int64_t n_rows_bound, int64_t n_edges) {
    return tg_align_up((size_t)(n_rows_bound + 1) * sizeof(int4)) + tg_align_up((size_t)side_items_bound(n_edges) * sizeof(int4)) +
           tg_align_up((size_t)side_hubs_bound(n_edges) * sizeof(int4)) + tg_align_up((size_t)side_bighubs_bound(n_edges) * sizeof(int4)) +
           tg_scan_bytes<TG_SK>(n_rows_bound) + 512;
}

tg_status_t tg_side_build(tg_side* s, int64_t n_rows, int64_t n_edges, const int32_t* indptr, void* ws, size_t ws_bytes,
                          cudaStream_t stream) {
    *s = tg_side();
    s->n_rows = n_rows; s->n_edges = n_edges; s->indptr = indptr;
    if (n_rows == 0) return TG_OK;
    tg_carver c(ws, ws_bytes);
    s->rows = static_cast<int4*>(c.take((size_t)(n_rows + 1) * sizeof(int4)));
    s->items = static_cast<int4*>(c.take((size_t)side_items_bound(n_edges) * sizeof(int4)));
    s->hubs = static_cast<int4*>(c.take((size_t)side_hubs_bound(n_edges) * sizeof(int4)));
    s->bighubs = static_cast<int4*>(c.take((size_t)side_bighubs_bound(n_edges) * sizeof(int4)));
    void* scan_tmp = c.take(tg_scan_bytes<TG_SK>(n_rows));
    int* totals = static_cast<int*>(c.take(256));  // IVec<TG_SK> + max_deg at [TG_SK]
    if (!c.ok()) TG_FAIL(TG_ERR_WORKSPACE, "schedule workspace too small: need %zu, have %zu", c.off, ws_bytes);
    TG_CUDA(cudaMemsetAsync(totals, 0, 256, stream));
    // about 4 warp items per resident warp slot (148 SMs x 16 warps) when the side is small, TG_CHUNK_MAX beyond
    int chunk = TG_CHUNK_MIN;
    while (chunk < TG_CHUNK_MAX && n_edges / chunk > 148 * 16 * 4) chunk *= 2;
    s->chunk = chunk;
    SchedIn in{indptr, chunk};
    SchedOut out{indptr, chunk, s->rows, s->items, s->hubs, s->bighubs, totals + TG_SK};
    TG_TRY((tg_scan<TG_SK>(n_rows, in, out, scan_tmp, reinterpret_cast<IVec<TG_SK>*>(totals), stream)));
    int h[TG_SK + 1];
    TG_CUDA(cudaMemcpyAsync(h, totals, sizeof(h), cudaMemcpyDeviceToHost, stream));
    TG_CUDA(cudaStreamSynchronize(stream));
    s->n_group = 0;
    for (int k = 0; k < TG_NCLS; ++k) { s->n_cls[k] = h[k]; s->n_group += h[k]; }
    s->n_items = 0;
    for (int k = 0; k < TG_NICLS; ++k) s->n_items += h[TG_NCLS + k];
    s->n_slots = h[TG_NCLS + TG_NICLS]; s->n_hubs = h[TG_NCLS + TG_NICLS + 1]; s->n_bighubs = h[TG_NCLS + TG_NICLS + 2];
    s->max_deg = h[TG_SK];
    return TG_OK;
}

// ---------------------------------------------------------------------------------------------
// Build kernels
// ---------------------------------------------------------------------------------------------
struct BuildFlags {
    int bad_root;     // some root_idx outside [0, R)
    int unsorted;     // root_idx is not non-decreasing
    long long nbr_min, nbr_max;
};

__global__ void k_check(int64_t R, int64_t E, const int32_t* __restrict__ root, const int64_t* __restrict__ nbr, BuildFlags* f) {
    int bad = 0, uns = 0;
    long long mn = 0x7fffffffffffffffLL, mx = -0x7fffffffffffffffLL - 1;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < E; e += (int64_t)gridDim.x * blockDim.x) {
        const int r = root[e];
        bad |= (r < 0 || r >= R);
        if (e > 0) uns |= (root[e - 1] > r);
        const long long x = nbr[e];
        mn = min(mn, x); mx = max(mx, x);
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

// sorted roots: indptr[v] = e for every v in (root[e-1], root[e]]  (root[-1] = -1, root[E] = R)
__global__ void k_indptr_sorted(int64_t R, int64_t E, const int32_t* __restrict__ root, int32_t* indptr) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e <= E; e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t lo = (e == 0) ? 0 : (int64_t)root[e - 1] + 1;
        const int64_t hi = (e == E) ? R : (int64_t)root[e];
        for (int64_t v = lo; v <= hi; ++v) indptr[v] = (int32_t)e;
    }
}

__global__ void k_hist(int64_t E, const int32_t* __restrict__ root, int32_t* cnt) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < E; e += (int64_t)gridDim.x * blockDim.x)
        atomicAdd(&cnt[root[e]], 1);
}

__global__ void k_iota(int64_t n, int32_t* a) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) a[i] = (int32_t)i;
}

__global__ void k_gather_csr(int64_t E, const int32_t* __restrict__ perm, const int32_t* __restrict__ root,
                             const int64_t* __restrict__ nbr, const int64_t* __restrict__ eid, const float* __restrict__ ts,
                             int64_t* nbr_csr, int32_t* edge_dst, int64_t* eid_csr, float* ts_csr) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < E; e += (int64_t)gridDim.x * blockDim.x) {
        const int p = perm[e];
        nbr_csr[e] = nbr[p];
        edge_dst[e] = root[p];
        if (eid_csr) eid_csr[e] = eid[p];
        if (ts_csr) ts_csr[e] = ts[p];
    }
}

__global__ void k_identity(int64_t E, const int32_t* __restrict__ edge_dst, int32_t* kv_row, int32_t* t_indptr,
                           int32_t* t_edge, int32_t* t_dst) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e <= E; e += (int64_t)gridDim.x * blockDim.x) {
        t_indptr[e] = (int32_t)e;
        if (e < E) { kv_row[e] = (int32_t)e; t_edge[e] = (int32_t)e; t_dst[e] = edge_dst[e]; }
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

struct HeadIn {
    const int64_t* skeys;
    __device__ __forceinline__ IVec<1> operator()(int64_t j) const {
        IVec<1> x;
        x.v[0] = (j == 0) || (skeys[j] != skeys[j - 1]);
        return x;
    }
};
struct DedupOut {
    const int64_t* skeys;
    const int32_t* t_edge;
    const int32_t* edge_dst;
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
        if (x.v[0]) { uniq[row] = skeys[j]; t_indptr[row] = (int32_t)j; }
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
    int32_t* cnt;       // [R+1]
    int64_t* nbr_csr;   // [E]
    int64_t* keys_out;  // [E]
    int32_t* iota;      // [E]
    int32_t* root_out;  // [E]
    int32_t* edge_dst;  // [E]
    void* scan_tmp;
    int* scan_total;
    void* cub_tmp;
    size_t cub_bytes;
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
    w->nbr_csr = static_cast<int64_t*>(c.take((size_t)E * 8));
    w->keys_out = static_cast<int64_t*>(c.take((size_t)E * 8));
    w->iota = static_cast<int32_t*>(c.take((size_t)E * 4));
    w->root_out = static_cast<int32_t*>(c.take((size_t)E * 4));
    w->edge_dst = static_cast<int32_t*>(c.take((size_t)E * 4));
    w->scan_tmp = c.take(tg_scan_bytes<1>(E > R ? E : R));
    w->scan_total = static_cast<int*>(c.take(256));
    size_t b1 = 0, b2 = 0;
    if (E > 0) {
        TG_CUDA((cub::DeviceRadixSort::SortPairs<int32_t, int32_t>(nullptr, b1, nullptr, nullptr, nullptr, nullptr, (int)E, 0, 32)));
        if (dedup_mode)
            TG_CUDA((cub::DeviceRadixSort::SortPairs<int64_t, int32_t>(nullptr, b2, nullptr, nullptr, nullptr, nullptr, (int)E, 0, 64)));
    }
    w->cub_bytes = b1 > b2 ? b1 : b2;
    w->cub_tmp = c.take(w->cub_bytes);
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

    int64_t U = 0;
    if (E == 0) {
        TG_CUDA(cudaMemsetAsync(indptr, 0, (size_t)(R + 1) * 4, stream));
        TG_CUDA(cudaMemsetAsync(t_indptr, 0, 4, stream));
    } else {
        // 1. checks
        BuildFlags f0{0, 0, 0x7fffffffffffffffLL, -0x7fffffffffffffffLL - 1};
        TG_CUDA(cudaMemcpyAsync(w.flags, &f0, sizeof(f0), cudaMemcpyHostToDevice, stream));
        k_check<<<grid_for(E), 256, 0, stream>>>(R, E, root_idx, nbr_node, w.flags);
        TG_LAUNCH_CHECK("k_check");
        BuildFlags f;
        TG_CUDA(cudaMemcpyAsync(&f, w.flags, sizeof(f), cudaMemcpyDeviceToHost, stream));
        TG_CUDA(cudaStreamSynchronize(stream));
        if (f.bad_root) TG_FAIL(TG_ERR_INVALID_ARG, "root_idx has an entry outside [0, R)");
        // 2-3. indptr, perm
        if (!f.unsorted) {
            k_indptr_sorted<<<grid_for(E + 1), 256, 0, stream>>>(R, E, root_idx, indptr);
            TG_LAUNCH_CHECK("k_indptr_sorted");
            k_iota<<<grid_for(E), 256, 0, stream>>>(E, perm);
            TG_LAUNCH_CHECK("k_iota");
        } else {
            TG_CUDA(cudaMemsetAsync(w.cnt, 0, (size_t)(R + 1) * 4, stream));
            k_hist<<<grid_for(E), 256, 0, stream>>>(E, root_idx, w.cnt);
            TG_LAUNCH_CHECK("k_hist");
            TG_TRY((tg_scan<1>(R, CntIn{w.cnt}, IndptrOut{indptr, R}, w.scan_tmp, reinterpret_cast<IVec<1>*>(w.scan_total), stream)));
            k_iota<<<grid_for(E), 256, 0, stream>>>(E, w.iota);
            TG_LAUNCH_CHECK("k_iota");
            size_t tb = w.cub_bytes;
            TG_CUDA((cub::DeviceRadixSort::SortPairs<int32_t, int32_t>(w.cub_tmp, tb, root_idx, w.root_out, w.iota, perm, (int)E, 0,
                                                                        bits_for((uint64_t)(R - 1)), stream)));
        }
        // 4. CSR-order gathers
        k_gather_csr<<<grid_for(E), 256, 0, stream>>>(E, perm, root_idx, nbr_node, edge_id, ts, w.nbr_csr, w.edge_dst,
                                                       eid_csr, ts_csr);
        TG_LAUNCH_CHECK("k_gather_csr");
        // 5. unique rows + transposed CSR
        if (dedup_mode == 0) {
            U = E;
            TG_CUDA(cudaMemcpyAsync(uniq_node, w.nbr_csr, (size_t)E * 8, cudaMemcpyDeviceToDevice, stream));
            k_identity<<<grid_for(E + 1), 256, 0, stream>>>(E, w.edge_dst, kv_row, t_indptr, t_edge, t_dst);
            TG_LAUNCH_CHECK("k_identity");
        } else {
            k_iota<<<grid_for(E), 256, 0, stream>>>(E, w.iota);
            TG_LAUNCH_CHECK("k_iota");
            const int end_bit = (f.nbr_min >= 0) ? bits_for((uint64_t)f.nbr_max) : 64;
            size_t tb = w.cub_bytes;
            TG_CUDA((cub::DeviceRadixSort::SortPairs<int64_t, int32_t>(w.cub_tmp, tb, w.nbr_csr, w.keys_out, w.iota, t_edge, (int)E, 0,
                                                                        end_bit, stream)));
            DedupOut dout{w.keys_out, t_edge, w.edge_dst, kv_row, uniq_node, t_indptr, t_dst, E};
            TG_TRY((tg_scan<1>(E, HeadIn{w.keys_out}, dout, w.scan_tmp, reinterpret_cast<IVec<1>*>(w.scan_total), stream)));
            int u32 = 0;
            TG_CUDA(cudaMemcpyAsync(&u32, w.scan_total, 4, cudaMemcpyDeviceToHost, stream));
            TG_CUDA(cudaStreamSynchronize(stream));
            U = u32;
        }
    }
    // 6. schedules
    tg_block* b = new tg_block();
    b->R = R; b->E = E; b->U = U;
    b->indptr = indptr; b->kv_row = kv_row; b->t_indptr = t_indptr; b->t_edge = t_edge; b->t_dst = t_dst;
    tg_status_t st = tg_side_build(&b->dst, R, E, indptr, w.side_dst, w.side_dst_bytes, stream);
    if (st == TG_OK && U > 0) st = tg_side_build(&b->src, U, E, t_indptr, w.side_src, w.side_src_bytes, stream);
    if (st == TG_OK) {
        cudaError_t e = cudaStreamSynchronize(stream);
        if (e != cudaSuccess) { tg_set_error("tg_block_build: %s", cudaGetErrorString(e)); st = TG_ERR_CUDA; }
    }
    if (st != TG_OK) { delete b; return st; }
    *U_host = U;
    *out = b;
    return TG_OK;
}

extern "C" tg_status_t tg_block_destroy(tg_block_t* b) {
    delete b;
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
