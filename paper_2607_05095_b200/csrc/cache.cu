// cache.cu -- NEXT-2 of SURVEY.md §8(f): SlimCache (§4.2).
//   tg_cache_greedy_select  Algorithm 1: greedy hot-node / hot-edge selection under a budget.  HOST.
//   tg_cache_lookup         runtime stage: which of the batch's unique ids are resident, which rows must be
//                           transferred; builds the map the reconstruction uses.  DEVICE (one scan with a fused emit).
//   tg_feature_reconstruct  X[i] = row of occurrence i, through the inverse index, from the transferred rows or the resident
//                           cache.  DEVICE, a pure HBM gather/copy: 16-byte vectors, consecutive lanes on consecutive vectors.
#include <algorithm>
#include <mutex>
#include <numeric>
#include <vector>

#include "dispatch.cuh"
#include "scan.cuh"

// ---------------------------------------------------------------------------------------------
// Algorithm 1.  Readings: descending frequency, ties by ascending id; a tie between the node and the
// edge candidate goes to the edge (strict > in line 9); an exhausted list hands over to the other one.
// ---------------------------------------------------------------------------------------------
static void count_and_order(int64_t n, int64_t n_batches, const int64_t* ptr, const int64_t* ids, std::vector<int64_t>& f,
                            std::vector<int64_t>& order, bool* bad) {
    f.assign((size_t)n, 0);
    std::vector<int64_t> last((size_t)n, -1);   // a batch counts an id once (the batches are id sets)
    for (int64_t k = 0; k < n_batches; ++k)
        for (int64_t i = ptr[k]; i < ptr[k + 1]; ++i) {
            const int64_t x = ids[i];
            if (x < 0 || x >= n) { *bad = true; continue; }
            if (last[(size_t)x] != k) { last[(size_t)x] = k; f[(size_t)x] += 1; }
        }
    order.resize((size_t)n);
    std::iota(order.begin(), order.end(), (int64_t)0);
    std::stable_sort(order.begin(), order.end(), [&](int64_t a, int64_t b) { return f[(size_t)a] > f[(size_t)b]; });
}

extern "C" tg_status_t tg_cache_greedy_select(double alpha, int64_t n_batches, const int64_t* node_ptr, const int64_t* node_ids,
                                              const int64_t* edge_ptr, const int64_t* edge_ids, int64_t n_nodes, int64_t n_edges,
                                              int64_t* hot_nodes, int64_t* n_hot_nodes, int64_t* hot_edges, int64_t* n_hot_edges) {
    if (n_batches < 0 || n_nodes < 0 || n_edges < 0 || !(alpha >= 0.0) || !n_hot_nodes || !n_hot_edges)
        TG_FAIL(TG_ERR_INVALID_ARG, "tg_cache_greedy_select: bad argument");
    if (n_batches > 0 && (!node_ptr || !edge_ptr)) TG_FAIL(TG_ERR_INVALID_ARG, "tg_cache_greedy_select: null batch pointers");
    if ((n_nodes > 0 && !hot_nodes) || (n_edges > 0 && !hot_edges)) TG_FAIL(TG_ERR_INVALID_ARG, "tg_cache_greedy_select: null output");
    std::vector<int64_t> fv, fe, sv, se;
    bool bad = false;
    count_and_order(n_nodes, n_batches, node_ptr, node_ids, fv, sv, &bad);     // lines 1-6
    count_and_order(n_edges, n_batches, edge_ptr, edge_ids, fe, se, &bad);
    if (bad) TG_FAIL(TG_ERR_INVALID_ARG, "tg_cache_greedy_select: id outside [0, n)");
    int64_t i = 0, j = 0;                                                       // line 7
    const double budget = alpha * (double)(n_nodes + n_edges);
    while ((double)(i + j) < budget && (i < n_nodes || j < n_edges)) {          // line 8
        if (i < n_nodes && (j >= n_edges || fv[(size_t)sv[(size_t)i]] > fe[(size_t)se[(size_t)j]])) {   // line 9
            hot_nodes[i] = sv[(size_t)i]; ++i;                                  // lines 10-11
        } else {
            hot_edges[j] = se[(size_t)j]; ++j;                                  // lines 13-14
        }
    }
    *n_hot_nodes = i; *n_hot_edges = j;
    return TG_OK;
}

// ---------------------------------------------------------------------------------------------
// Lookup: map[u] = slot >= 0 ? -slot - 1 : (number of uncached ids before u); fresh_ids = the uncached ids, in order.
// ---------------------------------------------------------------------------------------------
struct MissIn {
    const int64_t* uniq;
    const int32_t* slot_of_id;
    __device__ __forceinline__ IVec<1> operator()(int64_t u) const {
        IVec<1> x;
        x.v[0] = slot_of_id[uniq[u]] < 0;
        return x;
    }
};
struct MissOut {
    const int64_t* uniq;
    const int32_t* slot_of_id;
    int32_t* map;
    int64_t* fresh_ids;
    __device__ __forceinline__ void operator()(int64_t u, const IVec<1>& ex, const IVec<1>& x, const IVec<1>&) const {
        if (x.v[0]) { map[u] = ex.v[0]; fresh_ids[ex.v[0]] = uniq[u]; }
        else map[u] = -slot_of_id[uniq[u]] - 1;
    }
};

extern "C" tg_status_t tg_cache_lookup_workspace_bytes(int64_t U, size_t* bytes) {
    if (!bytes || U < 0) TG_FAIL(TG_ERR_INVALID_ARG, "tg_cache_lookup_workspace_bytes: bad argument");
    *bytes = tg_scan_bytes<1>(U) + 512;
    return TG_OK;
}

extern "C" tg_status_t tg_cache_lookup(int64_t U, const int64_t* uniq_ids, const int32_t* slot_of_id, int32_t* map, int64_t* fresh_ids,
                                       int64_t* n_fresh_host, void* ws, size_t ws_bytes, tg_stream_t stream_) {
    if (U < 0 || U > TG_MAX_INDEX || !n_fresh_host) TG_FAIL(TG_ERR_INVALID_ARG, "tg_cache_lookup: bad argument");
    *n_fresh_host = 0;
    if (U == 0) return TG_OK;
    if (!uniq_ids || !slot_of_id || !map || !fresh_ids) TG_FAIL(TG_ERR_INVALID_ARG, "tg_cache_lookup: null array");
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    tg_carver c(ws, ws_bytes);
    void* tmp = c.take(tg_scan_bytes<1>(U));
    int* total = static_cast<int*>(c.take(256));
    if (!c.ok()) TG_FAIL(TG_ERR_WORKSPACE, "tg_cache_lookup needs %zu workspace bytes", c.off);
    TG_TRY((tg_scan<1>(U, MissIn{uniq_ids, slot_of_id}, MissOut{uniq_ids, slot_of_id, map, fresh_ids}, tmp,
                       reinterpret_cast<IVec<1>*>(total), stream)));
    int n = 0;
    TG_CUDA(cudaMemcpyAsync(&n, total, 4, cudaMemcpyDeviceToHost, stream));
    TG_CUDA(cudaStreamSynchronize(stream));
    *n_fresh_host = n;
    return TG_OK;
}

// ---------------------------------------------------------------------------------------------
// Reconstruction: one 16-byte (or 4-byte) vector per thread and step, VPR vectors per row.
// ---------------------------------------------------------------------------------------------
template <class V>
__global__ void __launch_bounds__(256) k_reconstruct(int64_t n, int vpr, const int32_t* __restrict__ inv, const int32_t* __restrict__ map,
                                                     const V* __restrict__ fresh, const V* __restrict__ cache, V* __restrict__ out) {
    constexpr int UN = 4;   // independent gathers in flight per thread: index -> map -> row is a three-deep dependent chain
    const int64_t total = n * vpr, stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t t0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t0 < total; t0 += UN * stride) {
        int m[UN], k[UN];
        V x[UN];
#pragma unroll
        for (int u = 0; u < UN; ++u) {
            const int64_t t = t0 + u * stride;
            const int64_t i = min(t, total - 1) / vpr;
            k[u] = (int)(min(t, total - 1) - i * vpr);
            m[u] = inv ? inv[i] : (int)i;
        }
#pragma unroll
        for (int u = 0; u < UN; ++u) m[u] = map[m[u]];
#pragma unroll
        for (int u = 0; u < UN; ++u) x[u] = (m[u] >= 0 ? fresh + (int64_t)m[u] * vpr : cache + (int64_t)(-m[u] - 1) * vpr)[k[u]];
#pragma unroll
        for (int u = 0; u < UN; ++u)
            if (t0 + u * stride < total) out[t0 + u * stride] = x[u];
    }
}

extern "C" tg_status_t tg_feature_reconstruct(int64_t n, int64_t row_bytes, const int32_t* inv_idx, const int32_t* map,
                                              const void* fresh_rows, const void* cache_rows, void* out, tg_stream_t stream_) {
    if (n < 0 || row_bytes <= 0 || (row_bytes & 3) != 0) TG_FAIL(TG_ERR_INVALID_ARG, "tg_feature_reconstruct: row_bytes must be a positive multiple of 4");
    if (n == 0) return TG_OK;
    if (!map || !out) TG_FAIL(TG_ERR_INVALID_ARG, "tg_feature_reconstruct: null array");
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const bool v16 = (row_bytes & 15) == 0 && ((reinterpret_cast<uintptr_t>(fresh_rows) | reinterpret_cast<uintptr_t>(cache_rows) |
                                                reinterpret_cast<uintptr_t>(out)) & 15) == 0;
    const int vpr = (int)(row_bytes / (v16 ? 16 : 4));
    int64_t grid = (n * vpr + 1023) / 1024;
    if (grid > 148 * 16) grid = 148 * 16;
    if (grid < 1) grid = 1;
    if (v16)
        k_reconstruct<uint4><<<(unsigned)grid, 256, 0, stream>>>(n, vpr, inv_idx, map, static_cast<const uint4*>(fresh_rows),
                                                                  static_cast<const uint4*>(cache_rows), static_cast<uint4*>(out));
    else
        k_reconstruct<uint32_t><<<(unsigned)grid, 256, 0, stream>>>(n, vpr, inv_idx, map, static_cast<const uint32_t*>(fresh_rows),
                                                                     static_cast<const uint32_t*>(cache_rows), static_cast<uint32_t*>(out));
    TG_LAUNCH_CHECK("tg_feature_reconstruct");
    return TG_OK;
}

// ---------------------------------------------------------------------------------------------
// tg_cache_lookup_static: the lookup above for callers that have no way to hand over a workspace.
//
// Who that is: code that runs where device allocation is forbidden or impossible -- a serving loop whose memory pool was
// sized once and is now full by design, a plug-in that is handed tensors by a host framework but owns no allocator, a
// real-time thread that must not take the driver's allocation lock (cudaMalloc synchronises the whole device).  For them
// the scan's scratch (one partial sum per tile of 1024 ids plus the grand total) lives in the array below: it is part of
// the library image, so every GPU on which the library is used holds these ~17 KB from the first use until the process
// exits, and no call ever asks the driver for memory.
//
// `g_lookup_scratch` is a DEVICE object.  In host code the name only identifies the symbol -- it is not an address a
// kernel can use -- so the address on each device is asked for once (cudaGetSymbolAddress, with that device current) and
// cached per device ordinal.
// ---------------------------------------------------------------------------------------------
constexpr size_t TG_LOOKUP_SCRATCH_TOTAL_OFF = (((size_t)(TG_CACHE_STATIC_MAX_IDS / TG_SCAN_TILE) + 1) * sizeof(IVec<1>) + 255) / 256 * 256 + 256;
constexpr size_t TG_LOOKUP_SCRATCH_BYTES = TG_LOOKUP_SCRATCH_TOTAL_OFF + 256;   // tile sums (tg_scan_bytes<1>(max)) + the total
static_assert(TG_CACHE_STATIC_MAX_IDS % TG_SCAN_TILE == 0, "the scratch is sized in whole scan tiles");

static __device__ __align__(256) unsigned char g_lookup_scratch[TG_LOOKUP_SCRATCH_BYTES];

constexpr int TG_MAX_DEVICES = 64;
static void* g_lookup_scratch_ptr[TG_MAX_DEVICES];   // device address of g_lookup_scratch, per device ordinal (0 = not asked yet)
static std::mutex g_lookup_scratch_mutex;

// Device address of the scratch on the CURRENT device; the first call per device asks the runtime (this may load the
// library's device code onto that GPU, which is why it should not happen for the first time inside a stream capture).
static tg_status_t lookup_scratch_on_current_device(unsigned char** out) {
    int dev = -1;
    TG_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= TG_MAX_DEVICES) TG_FAIL(TG_ERR_UNSUPPORTED, "tg_cache_lookup_static: device ordinal %d outside [0, %d)", dev, TG_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_lookup_scratch_mutex);
    if (!g_lookup_scratch_ptr[dev]) {
        void* p = nullptr;
        TG_CUDA(cudaGetSymbolAddress(&p, g_lookup_scratch));
        if (!p) TG_FAIL(TG_ERR_INTERNAL, "tg_cache_lookup_static: the runtime returned a null address for the scratch symbol");
        g_lookup_scratch_ptr[dev] = p;
    }
    *out = static_cast<unsigned char*>(g_lookup_scratch_ptr[dev]);
    return TG_OK;
}

extern "C" tg_status_t tg_cache_lookup_static(int64_t U, const int64_t* uniq_ids, const int32_t* slot_of_id, int32_t* map,
                                              int64_t* fresh_ids, int64_t* n_fresh_host, tg_stream_t stream_) {
    if (U < 0 || !n_fresh_host) TG_FAIL(TG_ERR_INVALID_ARG, "tg_cache_lookup_static: bad argument");
    *n_fresh_host = 0;
    if (U > (int64_t)TG_CACHE_STATIC_MAX_IDS)
        TG_FAIL(TG_ERR_WORKSPACE, "tg_cache_lookup_static: U = %lld exceeds the built-in scratch (TG_CACHE_STATIC_MAX_IDS = %lld ids); "
                                  "use tg_cache_lookup with a caller workspace", (long long)U, (long long)TG_CACHE_STATIC_MAX_IDS);
    if (U == 0) return TG_OK;
    if (!uniq_ids || !slot_of_id || !map || !fresh_ids) TG_FAIL(TG_ERR_INVALID_ARG, "tg_cache_lookup_static: null array");
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    unsigned char* scratch = nullptr;
    TG_TRY(lookup_scratch_on_current_device(&scratch));
    // Nothing in the scratch has to start at zero: the reduce launch writes every tile sum the spine reads, and the spine
    // writes the total before anyone reads it, so whatever the previous call left behind is overwritten first.
    void* tmp = scratch;
    int* total = reinterpret_cast<int*>(scratch + TG_LOOKUP_SCRATCH_TOTAL_OFF);
    TG_TRY((tg_scan<1>(U, MissIn{uniq_ids, slot_of_id}, MissOut{uniq_ids, slot_of_id, map, fresh_ids}, tmp,
                       reinterpret_cast<IVec<1>*>(total), stream)));
    int n = 0;
    TG_CUDA(cudaMemcpyAsync(&n, total, 4, cudaMemcpyDeviceToHost, stream));
    TG_CUDA(cudaStreamSynchronize(stream));
    *n_fresh_host = n;
    return TG_OK;
}
