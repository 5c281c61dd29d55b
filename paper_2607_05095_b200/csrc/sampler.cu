// sampler.cu -- device-side temporal neighbour sampler.
//
// The paper samples on the CPU (TGL's OpenMP sampler over T-CSR, with FAST's topology-aware core binding,
// PAPER.md:233-247) and ships the sampled lists over PCIe; here the time-sorted per-node incidence lists (T-CSR) live in
// HBM and the "top-k recent neighbor sampling with k = 10" of PAPER.md:311 (and the uniform-in-time variant of
// BASELINE.json configs[2]) runs on the device, emitting tg_block_build's inputs directly.
//
//   tg_tcsr_build       event stream (u, v, t) -> T-CSR {indptr, nbr, eid, ts}: every event is listed under both endpoints
//                       (a self-loop once), inside a node in ascending event index (readings R20, R27).  One stable radix
//                       sort of (node, entry position) + boundary fill + gather.  Integer work, bit-exact.
//   tg_sample_neighbors per root (node, cutoff): binary search of the cutoff in the node's list, then the k most recent
//                       prior entries or k of them uniformly without replacement -- Floyd's algorithm driven by the
//                       counter-based SplitMix64 stream (seed, root, draw) (reading R28).  One scan whose input functor
//                       counts and whose output functor emits at the exclusive offset; one D2H of the total.
#include "dispatch.cuh"
#include "scan.cuh"
#include "radix_sort.cuh"

// ---------------------------------------------------------------------------------------------
// T-CSR build
// ---------------------------------------------------------------------------------------------
// entry 2i = (u_i -> v_i), entry 2i+1 = (v_i -> u_i); the second entry of a self-loop gets the sentinel key n_nodes
__global__ void k_tcsr_keys(int64_t M, int64_t n_nodes, const int64_t* __restrict__ u, const int64_t* __restrict__ v, uint32_t* keys,
                            int* bad) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < M; i += (int64_t)gridDim.x * blockDim.x) {
        const long long a = u[i], b = v[i];
        if (a < 0 || a >= n_nodes || b < 0 || b >= n_nodes) atomicOr(bad, 1);
        keys[2 * i] = (uint32_t)a;
        keys[2 * i + 1] = (a == b) ? (uint32_t)n_nodes : (uint32_t)b;
    }
}

// sorted keys -> indptr (boundary fill: indptr[x] = first position whose key >= x) and the entry arrays
__global__ void k_tcsr_emit(int64_t M2b, int64_t n_nodes, const uint32_t* __restrict__ skeys, const int32_t* __restrict__ sent,
                            const int64_t* __restrict__ u, const int64_t* __restrict__ v, const float* __restrict__ t,
                            int64_t* indptr, int64_t* nbr, int64_t* eid, float* ts, int* long_gap) {
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p <= M2b; p += (int64_t)gridDim.x * blockDim.x) {
        const int64_t prev = (p == 0) ? -1 : (int64_t)skeys[p - 1];
        const int64_t cur = (p == M2b) ? n_nodes : (int64_t)skeys[p];
        const int64_t hi = min(cur, n_nodes);
        if (hi - prev > TG_FILL_CAP) *long_gap = 1;   // a long run of nodes without events: tg_fill_indptr_by_search writes all rows
        else for (int64_t x = prev + 1; x <= hi; ++x) indptr[x] = p;
        if (p < M2b && cur < n_nodes) {
            const int ent = sent[p];
            const int64_t i = ent >> 1;
            nbr[p] = (ent & 1) ? u[i] : v[i];
            eid[p] = i;
            ts[p] = t[i];
        }
    }
}

static inline int smp_grid(int64_t n) {
    int64_t g = (n + 255) / 256;
    return (int)(g < 1 ? 1 : (g > 148 * 16 ? 148 * 16 : g));
}
static inline int smp_bits(uint64_t x) {
    int b = 0;
    while (x) { ++b; x >>= 1; }
    return b < 1 ? 1 : b;
}

extern "C" tg_status_t tg_tcsr_workspace_bytes(int64_t n_nodes, int64_t M, size_t* bytes) {
    if (!bytes) TG_FAIL(TG_ERR_INVALID_ARG, "bytes is null");
    if (n_nodes < 0 || M < 0 || n_nodes >= 0xffffffffLL || 2 * M > TG_MAX_INDEX) TG_FAIL(TG_ERR_INVALID_ARG, "n_nodes=%lld M=%lld out of range", (long long)n_nodes, (long long)M);
    *bytes = 2 * tg_align_up((size_t)(2 * M) * 4) * 2 + tg_rs_bytes<uint32_t>(2 * M) + 1024;
    return TG_OK;
}

extern "C" tg_status_t tg_tcsr_build(int64_t n_nodes, int64_t M, const int64_t* u, const int64_t* v, const float* t, int64_t* tc_indptr,
                                     int64_t* tc_nbr, int64_t* tc_eid, float* tc_ts, void* workspace, size_t workspace_bytes,
                                     tg_stream_t stream_) {
    if (n_nodes < 0 || M < 0 || n_nodes >= 0xffffffffLL || 2 * M > TG_MAX_INDEX) TG_FAIL(TG_ERR_INVALID_ARG, "n_nodes=%lld M=%lld out of range", (long long)n_nodes, (long long)M);
    if (!tc_indptr) TG_FAIL(TG_ERR_INVALID_ARG, "tc_indptr is null");
    if (M > 0 && (!u || !v || !t || !tc_nbr || !tc_eid || !tc_ts)) TG_FAIL(TG_ERR_INVALID_ARG, "null stream / output array");
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    if (M == 0) {
        TG_CUDA(cudaMemsetAsync(tc_indptr, 0, (size_t)(n_nodes + 1) * 8, stream));
        return TG_OK;
    }
    tg_carver c(workspace, workspace_bytes);
    const int64_t n = 2 * M;
    uint32_t* ka = static_cast<uint32_t*>(c.take((size_t)n * 4));
    uint32_t* kb = static_cast<uint32_t*>(c.take((size_t)n * 4));
    int32_t* va = static_cast<int32_t*>(c.take((size_t)n * 4));
    int32_t* vb = static_cast<int32_t*>(c.take((size_t)n * 4));
    void* rs = c.take(tg_rs_bytes<uint32_t>(n));
    int* bad = static_cast<int*>(c.take(256));
    if (!c.ok()) TG_FAIL(TG_ERR_WORKSPACE, "T-CSR workspace: need %zu bytes, have %zu", c.off, workspace_bytes);
    TG_CUDA(cudaMemsetAsync(bad, 0, 8, stream));   // bad[0]: endpoint out of range; bad[1]: a long run of empty rows
    k_tcsr_keys<<<smp_grid(M), 256, 0, stream>>>(M, n_nodes, u, v, ka, bad);
    TG_LAUNCH_CHECK("k_tcsr_keys");
    uint32_t* kres; int32_t* vres;
    TG_TRY((tg_radix_sort<uint32_t>(n, smp_bits((uint64_t)n_nodes), ka, va, true, kb, vb, &kres, &vres, rs, stream)));
    k_tcsr_emit<<<smp_grid(n + 1), 256, 0, stream>>>(n, n_nodes, kres, vres, u, v, t, tc_indptr, tc_nbr, tc_eid, tc_ts, bad + 1);
    TG_LAUNCH_CHECK("k_tcsr_emit");
    // keys equal to n_nodes are the self-loop sentinels: "number of keys below x" for x <= n_nodes never counts them
    tg_fill_indptr_by_search<uint32_t, int64_t><<<smp_grid(n_nodes + 1), 256, 0, stream>>>(n, n_nodes, kres, tc_indptr, bad + 1);
    TG_LAUNCH_CHECK("tg_fill_indptr_by_search");
    int hbad = 0;
    TG_CUDA(cudaMemcpyAsync(&hbad, bad, 4, cudaMemcpyDeviceToHost, stream));
    TG_CUDA(cudaStreamSynchronize(stream));
    if (hbad) TG_FAIL(TG_ERR_INVALID_ARG, "an event endpoint is outside [0, n_nodes)");
    return TG_OK;
}

// ---------------------------------------------------------------------------------------------
// Sampling
// ---------------------------------------------------------------------------------------------
constexpr int TG_SAMPLE_MAX_K = 64;

// n-th output (n >= 1) of SplitMix64 seeded with `seed`: state_n = seed + n * golden, output = finaliser(state_n)
__device__ __forceinline__ unsigned long long tg_splitmix64(unsigned long long seed, unsigned long long n) {
    unsigned long long z = seed + n * 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

struct SampleParams {
    const int64_t* root_node; const int64_t* root_cutoff;
    const int64_t* tc_indptr; const int64_t* tc_nbr; const int64_t* tc_eid; const float* tc_ts;
    int64_t n_nodes;
    int k, mode;
    unsigned long long seed;
    int32_t* root_idx; int64_t* nbr_node; int64_t* edge_id; float* ts;
};

// [s, p): the root's entries with event index strictly below its cutoff
__device__ __forceinline__ void tg_prior_range(const SampleParams& P, int64_t i, int64_t& s, int64_t& p) {
    const int64_t x = P.root_node[i];
    if (x < 0 || x >= P.n_nodes) { s = p = 0; return; }     // unknown node: no prior events
    s = P.tc_indptr[x];
    int64_t lo = s, hi = P.tc_indptr[x + 1];
    const int64_t c = P.root_cutoff[i];
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (P.tc_eid[mid] < c) lo = mid + 1; else hi = mid;
    }
    p = lo;
}

struct SampleIn {
    SampleParams P;
    __device__ __forceinline__ IVec<1> operator()(int64_t i) const {
        int64_t s, p;
        tg_prior_range(P, i, s, p);
        IVec<1> x;
        x.v[0] = (int)min((int64_t)P.k, p - s);
        return x;
    }
};
struct SampleOut {
    SampleParams P;
    __device__ __forceinline__ void emit(int64_t o, int64_t i, int64_t pos) const {
        P.root_idx[o] = (int32_t)i;
        P.nbr_node[o] = P.tc_nbr[pos];
        P.edge_id[o] = P.tc_eid[pos];
        P.ts[o] = P.tc_ts[pos];
    }
    __device__ __forceinline__ void operator()(int64_t i, const IVec<1>& ex, const IVec<1>& x, const IVec<1>&) const {
        const int take = x.v[0];
        if (take == 0) return;
        int64_t s, p;
        tg_prior_range(P, i, s, p);
        const int64_t n = p - s, o = ex.v[0];
        if (P.mode == 0 || n <= P.k) {            // most recent (oldest first); fewer candidates than k: all of them
            for (int j = 0; j < take; ++j) emit(o + j, i, p - take + j);
            return;
        }
        // Floyd: for j = n-k .. n-1 draw t in [0, j]; take t unless taken, else j.  Kept sorted by insertion.
        int64_t pick[TG_SAMPLE_MAX_K];
        int m = 0;
        for (int d = 0; d < P.k; ++d) {
            const int64_t j = n - P.k + d;
            const unsigned long long r = tg_splitmix64(P.seed, (unsigned long long)TG_SAMPLE_MAX_K * (unsigned long long)i + d + 1);
            int64_t t = (int64_t)__umul64hi(r, (unsigned long long)(j + 1));
            bool taken = false;
            for (int q = 0; q < m; ++q) taken |= (pick[q] == t);
            if (taken) t = j;
            int q = m++;
            while (q > 0 && pick[q - 1] > t) { pick[q] = pick[q - 1]; --q; }
            pick[q] = t;
        }
        for (int j = 0; j < P.k; ++j) emit(o + j, i, s + pick[j]);
    }
};

extern "C" tg_status_t tg_sample_workspace_bytes(int64_t n_roots, size_t* bytes) {
    if (!bytes) TG_FAIL(TG_ERR_INVALID_ARG, "bytes is null");
    if (n_roots < 0 || n_roots > TG_MAX_INDEX) TG_FAIL(TG_ERR_INVALID_ARG, "n_roots out of range");
    *bytes = tg_scan_bytes<1>(n_roots) + 512;
    return TG_OK;
}

extern "C" tg_status_t tg_sample_neighbors(int mode, int k, uint64_t seed, int64_t n_roots, const int64_t* root_node,
                                           const int64_t* root_cutoff, int64_t n_nodes, const int64_t* tc_indptr, const int64_t* tc_nbr,
                                           const int64_t* tc_eid, const float* tc_ts, int32_t* root_idx, int64_t* nbr_node,
                                           int64_t* edge_id, float* ts, int64_t* E_host, void* workspace, size_t workspace_bytes,
                                           tg_stream_t stream_) {
    if (!E_host) TG_FAIL(TG_ERR_INVALID_ARG, "E_host is null");
    *E_host = 0;
    if (mode != 0 && mode != 1) TG_FAIL(TG_ERR_INVALID_ARG, "mode must be 0 (most recent) or 1 (uniform)");
    if (k < 1 || k > TG_SAMPLE_MAX_K) TG_FAIL(TG_ERR_INVALID_ARG, "k must be in [1, %d]", TG_SAMPLE_MAX_K);
    if (n_roots < 0 || n_roots > TG_MAX_INDEX || n_roots * (int64_t)k > TG_MAX_INDEX) TG_FAIL(TG_ERR_INVALID_ARG, "n_roots * k out of range");
    if (n_roots == 0) return TG_OK;
    if (!root_node || !root_cutoff || !tc_indptr || !root_idx || !nbr_node || !edge_id || !ts) TG_FAIL(TG_ERR_INVALID_ARG, "null array");
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    tg_carver c(workspace, workspace_bytes);
    void* scan_tmp = c.take(tg_scan_bytes<1>(n_roots));
    IVec<1>* total = static_cast<IVec<1>*>(c.take(256));
    if (!c.ok()) TG_FAIL(TG_ERR_WORKSPACE, "sampler workspace: need %zu bytes, have %zu", c.off, workspace_bytes);
    SampleParams P{root_node, root_cutoff, tc_indptr, tc_nbr, tc_eid, tc_ts, n_nodes, k, mode, (unsigned long long)seed, root_idx, nbr_node, edge_id, ts};
    TG_TRY((tg_scan<1>(n_roots, SampleIn{P}, SampleOut{P}, scan_tmp, total, stream)));
    int e = 0;
    TG_CUDA(cudaMemcpyAsync(&e, total, 4, cudaMemcpyDeviceToHost, stream));
    TG_CUDA(cudaStreamSynchronize(stream));
    *E_host = e;
    return TG_OK;
}
