/*
 * fasttg.h -- C ABI of libfasttg: temporal-attention message passing over one mini-batch's
 * sampled temporal subgraph, hand-written for NVIDIA B200 (sm_100a).
 *
 * What the library computes (reference = PAPER.md, FAST, arxiv/paper_2607_05095):
 *   - the compression engine's index triple uni_ID / inv_Idx / CSR ind_ptr (§4.2,
 *     PAPER.md:287 §5) plus a transposed CSR for the backward gather          -> tg_block_build
 *   - AGG, h_v = sum_{u in N_in(v)} v_u (§4.3 "Balanced Aggregate", Eq.(1)),
 *     optionally alpha-weighted                                              -> tg_aggregate_fwd/bwd
 *   - ESM, the numerically stable edge softmax: max reduction, sum reduction, element-wise division
 *     per destination (§4.3 "Edge Softmax")                      -> tg_edge_softmax_fwd/bwd
 *   - per-edge attention logits (DGL gSDDMM, only named at PAPER.md:94)       -> tg_sddmm
 *   - the three fused into one pass, "forward and backward" -> tg_attn_fused_fwd/bwd
 *
 * Conventions shared by every call
 *   Memory.    Every pointer is a DEVICE pointer unless its comment says HOST.  The library never
 *              allocates or frees device memory: inputs, outputs, workspaces and the block's index
 *              arrays belong to the caller and must stay alive until the work enqueued on `stream`
 *              has finished (block arrays and the block workspace: until tg_block_destroy).
 *   Layout.    Row-major, contiguous.  Row tensors are [rows, H, D] in the storage dtype (TG_F32 or
 *              TG_BF16); edge-level tensors are [E, H] float32; all accumulation is float32.
 *              Base pointers of row tensors must be 16-byte aligned (else TG_ERR_ALIGNMENT).
 *   Notation.  R destinations (roots), E sampled edges in destination-grouped CSR order, U unique
 *              source rows, v(e) destination of CSR edge e, r(e) = kv_row[e], N(v) = CSR edges of v.
 *   Streams.   `stream` is a cudaStream_t passed as void*.  Calls enqueue and return; only
 *              tg_block_build synchronises the stream (it returns U to the host).
 *   Errors.    Every call returns a tg_status_t; nothing throws or aborts across the ABI.  Arguments
 *              are validated before any launch.  tg_last_error() gives thread-local detail text.
 *   Edge cases. R == 0 or E == 0 is TG_OK.  A zero-degree destination gives O = 0, LSE = -inf,
 *              dQ = 0 (reading R5).  Inputs must be finite.  Multi-edges are distinct edges.
 *   Supported (H, D): (2,50) (4,32) (8,16) (2,64) (1,128) (2,32) (4,16) (2,128), each in TG_F32 and TG_BF16;
 *              tg_supported() answers for a given (H, D, dtype); anything else is TG_ERR_UNSUPPORTED.
 *   There is no CPU fallback: without a CUDA device every compute call returns TG_ERR_CUDA.
 */
#ifndef FASTTG_H_
#define FASTTG_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(_WIN32)
#define TG_API
#else
#define TG_API __attribute__((visibility("default")))
#endif

typedef enum {
    TG_OK = 0,
    TG_ERR_INVALID_ARG = 1,  /* null pointer, negative size, out-of-range scalar */
    TG_ERR_UNSUPPORTED = 2,  /* (H, D, dtype) outside the supported set */
    TG_ERR_ALIGNMENT = 3,    /* a row tensor's base pointer is not 16-byte aligned */
    TG_ERR_WORKSPACE = 4,    /* workspace pointer null or too small */
    TG_ERR_CUDA = 5,         /* a CUDA runtime call failed; text in tg_last_error() */
    TG_ERR_INTERNAL = 6
} tg_status_t;

typedef enum { TG_F32 = 0, TG_BF16 = 1 } tg_dtype_t;

typedef void* tg_stream_t; /* cudaStream_t */

/* Host-side handle.  Holds sizes, pointers into caller memory and the internal schedules (which
 * live in the block workspace).  Created by tg_block_build / tg_block_from_csr. */
typedef struct tg_block tg_block_t;

TG_API const char* tg_status_string(tg_status_t s);
TG_API const char* tg_last_error(void);
TG_API int tg_version(void);
/* Number of kernels this library has launched in the process so far (all threads, all streams):
 * the difference across a timed region is the library's launch count for it. */
TG_API unsigned long long tg_launch_count(void);
/* 1 if (H, D, dtype) has a compiled kernel path, else 0. */
TG_API int tg_supported(int H, int D, tg_dtype_t dtype);

/* ------------------------------------------------------------------------------------------------
 * Block build: the compression engine's triple + transposed CSR (R7-R10)
 *
 * Input: the sampler's COO lists, in any order (E entries):
 *   root_idx[e]  int32, destination slot in [0,R)       nbr_node[e]  int64, neighbour (source) node id
 *   edge_id[e]   int64, nullable                        ts[e]        float32, nullable
 * Output (all caller-allocated, device):
 *   indptr[R+1]  int32  exclusive prefix sum of bincount(root_idx)            (CSR ind_ptr)
 *   perm[E]      int32  stable argsort of root_idx: CSR position -> input position
 *   kv_row[E]    int32  rank of nbr_node[perm[e]] in uniq_node                 (inv_Idx)
 *   uniq_node[>=E] int64 ascending distinct neighbour ids, U valid entries     (uni_ID)
 *   t_indptr[>=E+1] int32, t_edge[E] int32, t_dst[E] int32: transposed CSR; row u lists the CSR
 *                positions e with kv_row[e] == u in ascending order, t_dst[j] = v(t_edge[j])
 *   eid_csr[E] int64 = edge_id[perm], ts_csr[E] float32 = ts[perm]   (nullable, need their inputs)
 *   U_host       HOST int64*, written before return
 * dedup_mode 0: identity rows (U = E, kv_row[e] = e, uniq_node[e] = nbr_node[perm[e]]; K/V are per-edge
 *               rows [E,H,D]);  dedup_mode 1: dedup by neighbour node id.
 * All index results are exact integers with exactly one correct value (bit-exact against the oracle).
 * Errors: TG_ERR_INVALID_ARG (null, R < 0, E < 0, E or R > 2^31 - 4096, root_idx out of range ->
 *         detected on device, reported after the sync), TG_ERR_WORKSPACE, TG_ERR_CUDA.
 * The workspace must stay alive (and untouched) until tg_block_destroy: the schedules live in it.
 * Synchronisation: every launch of the build is enqueued first, then ONE device-to-host copy (flags, U, the
 * schedules' sizes) and ONE cudaStreamSynchronize.  What the host cannot know beforehand (is root_idx sorted? how
 * many bits do the neighbour ids need?) is speculated from the calling thread's previous build and verified after
 * the sync; a wrong guess repeats the build once with the measured values (first call of a thread, or a workload
 * whose id range grows).  No library sort: csrc/radix_sort.cuh.
 * ---------------------------------------------------------------------------------------------- */
TG_API tg_status_t tg_block_workspace_bytes(int64_t R, int64_t E, int dedup_mode, size_t* bytes /*HOST*/);

TG_API tg_status_t tg_block_build(int64_t R, int64_t E,
                                  const int32_t* root_idx, const int64_t* nbr_node,
                                  const int64_t* edge_id, const float* ts, int dedup_mode,
                                  int32_t* indptr, int32_t* perm, int32_t* kv_row, int64_t* uniq_node,
                                  int32_t* t_indptr, int32_t* t_edge, int32_t* t_dst,
                                  int64_t* eid_csr, float* ts_csr,
                                  int64_t* U_host /*HOST*/,
                                  void* workspace, size_t workspace_bytes, tg_stream_t stream,
                                  tg_block_t** out /*HOST*/);

/* Wrap index arrays that already exist on the device (e.g. a previous build, or a caller's own
 * CSR) and build only the internal schedules.  Same ownership rules.  Synchronises the stream.
 * tg_sched_workspace_bytes gives the workspace size. */
TG_API tg_status_t tg_sched_workspace_bytes(int64_t R, int64_t E, int64_t U, size_t* bytes /*HOST*/);
TG_API tg_status_t tg_block_from_csr(int64_t R, int64_t E, int64_t U,
                                     const int32_t* indptr, const int32_t* kv_row,
                                     const int32_t* t_indptr, const int32_t* t_edge, const int32_t* t_dst,
                                     void* workspace, size_t workspace_bytes, tg_stream_t stream,
                                     tg_block_t** out /*HOST*/);

TG_API tg_status_t tg_block_destroy(tg_block_t* b);

/* Sizes and schedule statistics of a block (HOST outputs; any may be null).
 * stats[0..7] = dst side {group-tier rows with degree <= 8, group-tier rows with degree 9..64, warp-tier
 * chunk items (rows above the side's group_max, one per `chunk` edges: tg_block_sched_info), partial slots of multi-chunk rows}, src side the same. */
TG_API tg_status_t tg_block_info(const tg_block_t* b, int64_t* R, int64_t* E, int64_t* U, int64_t stats[8]);

/* Schedule parameters of a block (HOST output): out[0..3] = destination side {group_max: rows of up to this many edges
 * are group-tier rows, chunk: edges per warp-tier item, number of hub rows (rows split over several items), largest
 * degree (0 unless some row has more than 8 edges)}, out[4..7] = the source side likewise. */
TG_API tg_status_t tg_block_sched_info(const tg_block_t* b, int64_t out[8]);
/* Number of block builds in this process that ran twice because the calling thread's speculation (sorted input, key
 * width) was too optimistic.  The speculation is sticky (it follows the largest recent need and relaxes after eight
 * consecutive smaller builds), so a steady workload shows at most one retry per thread and change of regime. */
TG_API unsigned long long tg_block_build_retries(void);

/* ------------------------------------------------------------------------------------------------
 * Temporal neighbour sampler on the device
 *
 * PAPER.md:311 "top-k recent neighbor sampling [18] with k=10" over TGL's T-CSR.  The paper samples on
 * the CPU (section 4.4) and ships the lists over PCIe; here the lists are produced in HBM, in the
 * form tg_block_build consumes.
 *
 * tg_tcsr_build: event stream -> per-node, time-ordered incidence lists.
 *   in : u[M], v[M] int64 endpoints in [0, n_nodes), t[M] float32 event times; event i has stream index i, the stream
 *        is in time order (ties broken by the index, readings R20, R27)
 *   out: tc_indptr[n_nodes+1] int64; tc_nbr / tc_eid [2M] int64, tc_ts [2M] float32 (tc_indptr[n_nodes] valid entries):
 *        node x's entries tc_indptr[x] .. tc_indptr[x+1]-1 list, in ascending event index, every event incident to x
 *        (either direction, a self-loop once) as {other endpoint, event index, event time}
 *   Exact integer work (one stable radix sort).  Synchronises the stream (reports out-of-range endpoints).
 *
 * tg_sample_neighbors: per root i = (root_node[i], root_cutoff[i]) the prior events of its node -- event index
 *   strictly below the cutoff -- at most k of them:
 *     mode 0: the k most recent;  mode 1: k uniformly without replacement (all if there are <= k).
 *   Mode 1 is Floyd's algorithm (draw d = 0..k-1: t uniform in [0, n-k+d], take t unless taken, else n-k+d) on the
 *   counter-based stream  r(seed, i, d) = SplitMix64 output number 64*i + d + 1 of `seed`,  t = high 64 bits of r * (n-k+d+1):
 *   reproducible, the same draw for any launch shape (reading R28).
 *   out (capacity n_roots * k each): root_idx int32 (= i), nbr_node int64, edge_id int64, ts float32 -- roots in order,
 *   inside a root oldest first; E_host (HOST) = number of sampled edges.  A root whose node is outside [0, n_nodes)
 *   or has no prior event contributes nothing.  1 <= k <= 64.  Synchronises the stream (returns E).
 * ---------------------------------------------------------------------------------------------- */
TG_API tg_status_t tg_tcsr_workspace_bytes(int64_t n_nodes, int64_t M, size_t* bytes /*HOST*/);
TG_API tg_status_t tg_tcsr_build(int64_t n_nodes, int64_t M, const int64_t* u, const int64_t* v, const float* t,
                                 int64_t* tc_indptr, int64_t* tc_nbr, int64_t* tc_eid, float* tc_ts,
                                 void* workspace, size_t workspace_bytes, tg_stream_t stream);
TG_API tg_status_t tg_sample_workspace_bytes(int64_t n_roots, size_t* bytes /*HOST*/);
TG_API tg_status_t tg_sample_neighbors(int mode, int k, uint64_t seed, int64_t n_roots,
                                       const int64_t* root_node, const int64_t* root_cutoff,
                                       int64_t n_nodes, const int64_t* tc_indptr, const int64_t* tc_nbr,
                                       const int64_t* tc_eid, const float* tc_ts,
                                       int32_t* root_idx, int64_t* nbr_node, int64_t* edge_id, float* ts,
                                       int64_t* E_host /*HOST*/, void* workspace, size_t workspace_bytes, tg_stream_t stream);

/* ------------------------------------------------------------------------------------------------
 * Unfused operators
 * ---------------------------------------------------------------------------------------------- */

/* SDDMM (gSDDMM named at PAPER.md:94; R1): s[e,h] = scale * <A[v(e),h,:], B[r(e),h,:]>.
 * A [R,H,D], B [U,H,D] in `dtype`; s [E,H] float32. */
TG_API tg_status_t tg_sddmm(const tg_block_t* b, int H, int D, tg_dtype_t dtype,
                            const void* A, const void* B, float scale, float* s, tg_stream_t stream);

/* ESM forward: alpha[e,h] = exp(s[e,h] - m[v,h]) / l[v,h], m = max over N(v),
 * l = sum over N(v) of exp(s - m).  s, alpha [E,H] float32; alpha may alias s. */
TG_API tg_status_t tg_edge_softmax_fwd(const tg_block_t* b, int H, const float* s, float* alpha,
                                       tg_stream_t stream);

/* ESM backward: ds[e,h] = alpha[e,h] * (dalpha[e,h] - sum_{e' in N(v)} alpha[e',h]*dalpha[e',h]). */
TG_API tg_status_t tg_edge_softmax_bwd(const tg_block_t* b, int H, const float* alpha, const float* dalpha,
                                       float* ds, tg_stream_t stream);

/* AGG forward: Y[v,h,:] = sum_{e in N(v)} w[e,h] * X[r(e),h,:]; w == NULL is the paper's
 * plain neighbour sum.  X [U,H,D], Y [R,H,D] in `dtype`; w [E,H] float32.
 * ws: tg_attn_workspace_bytes(...).fwd_bytes is sufficient. */
TG_API tg_status_t tg_aggregate_fwd(const tg_block_t* b, int H, int D, tg_dtype_t dtype,
                                    const float* w, const void* X, void* Y,
                                    void* ws, size_t ws_bytes, tg_stream_t stream);

/* AGG backward (the paper scatters with atomics, PAPER.md:219-223 -- here a gather
 * through the transposed CSR, no float atomics):
 *   dX[u,h,:] = sum_{e: r(e)=u} w[e,h] * dY[v(e),h,:]          (w == NULL: plain sum)
 *   dw[e,h]   = <dY[v(e),h,:], X[r(e),h,:]>                    (only if dw != NULL; needs X)
 * ws: tg_attn_workspace_bytes(...).bwd_bytes is sufficient. */
TG_API tg_status_t tg_aggregate_bwd(const tg_block_t* b, int H, int D, tg_dtype_t dtype,
                                    const float* w, const void* X, const void* dY,
                                    void* dX, float* dw, void* ws, size_t ws_bytes, tg_stream_t stream);

/* The paper's own AGG partitioning as the measured alternative (Fig. 6(b)-III): COO, one thread per
 * (edge, 4-element vector), one red.global.add.v4.f32 per thread.  Plain sum only (w == NULL of the calls above).
 *   tg_block_coo_dst : coo_dst[e] = v(e), the destination of CSR edge e (int32 [E]) -- the COO row array.
 *   tg_aggregate_coo : backward == 0:  Y[v(e)] += X[r(e)]   (X [U,H,D] in `dtype`, Y [R,H,D] float32)
 *                      backward != 0:  Y[r(e)] += X[v(e)]   (X [R,H,D] in `dtype`, Y [U,H,D] float32)
 *   Y is zeroed by the call and accumulated with float atomics: the result is NOT bitwise reproducible (the CSR calls
 *   above are).  H*D must be a multiple of 4.  DESIGN.md section 15 has the measured comparison. */
TG_API tg_status_t tg_block_coo_dst(const tg_block_t* b, int32_t* coo_dst, tg_stream_t stream);
TG_API tg_status_t tg_aggregate_coo(const tg_block_t* b, int H, int D, tg_dtype_t dtype, int backward,
                                    const int32_t* coo_dst, const void* X, float* Y, tg_stream_t stream);

/* ------------------------------------------------------------------------------------------------
 * Fused attention (SDDMM -> ESM -> alpha-weighted AGG without materialising s or alpha)
 * ---------------------------------------------------------------------------------------------- */
TG_API tg_status_t tg_attn_workspace_bytes(const tg_block_t* b, int H, int D, tg_dtype_t dtype,
                                           size_t* fwd_bytes /*HOST*/, size_t* bwd_bytes /*HOST*/);

/* Forward:  s = scale*<Q[v(e)],K[r(e)]>, alpha = softmax over N(v), O[v] = sum alpha*V[r(e)],
 *           LSE[v,h] = m + ln l (natural log).  Q,O [R,H,D]; K,V [U,H,D]; LSE [R,H] float32.
 * o_f32 (nullable, [R,H,D] float32, 16-byte aligned): an unrounded copy of O for the backward.  Meant for TG_BF16
 *           storage, where it lets the backward take delta = <dO, O> up front instead of accumulating it from the
 *           edges; R*H*D*4 extra bytes written here and read there, not part of the compulsory bytes. */
TG_API tg_status_t tg_attn_fused_fwd(const tg_block_t* b, int H, int D, tg_dtype_t dtype,
                                     const void* Q, const void* K, const void* V, float scale,
                                     void* O, float* lse, float* o_f32, void* ws, size_t ws_bytes, tg_stream_t stream);

/* Backward for upstream gradient dO:
 *   delta[v,h] = <dO[v,h,:], O[v,h,:]>;  alpha = exp(s - LSE);  dalpha = <dO[v(e)], V[r(e)]>;
 *   ds = alpha*(dalpha - delta);  dQ[v] = scale * sum_{N(v)} ds*K[r(e)];
 *   dK[u] = scale * sum_{r(e)=u} ds*Q[v(e)];  dV[u] = sum_{r(e)=u} alpha*dO[v(e)].
 * O and lse are the forward's outputs.  dQ [R,H,D]; dK,dV [U,H,D].
 * TG_BF16 storage: the bf16 rounding of O would leak into dQ through delta, so delta comes either from
 * o_f32 (the forward's float32 copy of O, if given) or, with o_f32 == NULL, from the edges (sum alpha*dalpha in fp32,
 * one more accumulator per lane); O itself is then only validated, not read.  TG_F32 storage ignores o_f32. */
TG_API tg_status_t tg_attn_fused_bwd(const tg_block_t* b, int H, int D, tg_dtype_t dtype,
                                     const void* Q, const void* K, const void* V, const void* O, const float* o_f32,
                                     const float* lse, const void* dO, float scale,
                                     void* dQ, void* dK, void* dV,
                                     void* ws, size_t ws_bytes, tg_stream_t stream);

/* Streams.  Every attention call only enqueues work.  On a block side with >= 2^20 edges part of the work is put on
 * two library-owned auxiliary streams that are forked from `stream` and joined back into it with events before the
 * call returns, so for the caller the call is ordered on `stream` like a single kernel, and it can be captured into a
 * CUDA graph (stream capture follows the fork / join).  The auxiliary streams are per calling thread and device. */

/* The two passes of tg_attn_fused_bwd as separate calls (tg_attn_fused_bwd = _dst then _src on one stream),
 * for callers that want to time or overlap them.  _dst: destination-major, writes dQ and the internal
 * {LSE, delta} table into `ws`; _src: source-major over the transposed CSR, reads that table from the
 * SAME `ws`, writes dK and dV.  Arguments as in tg_attn_fused_bwd. */
TG_API tg_status_t tg_attn_fused_bwd_dst(const tg_block_t* b, int H, int D, tg_dtype_t dtype,
                                         const void* Q, const void* K, const void* V, const void* O, const float* o_f32,
                                         const float* lse, const void* dO, float scale, void* dQ,
                                         void* ws, size_t ws_bytes, tg_stream_t stream);
TG_API tg_status_t tg_attn_fused_bwd_src(const tg_block_t* b, int H, int D, tg_dtype_t dtype,
                                         const void* Q, const void* K, const void* V, const void* dO,
                                         float scale, void* dK, void* dV,
                                         void* ws, size_t ws_bytes, tg_stream_t stream);

/* ------------------------------------------------------------------------------------------------
 * NEXT-1: the full TGAT edge term -- "temporal and edge information during message
 * passing".  Every sampled edge adds its own row (time encoding / edge-feature projection)
 * to the gathered key and value, and the logits pass a LeakyReLU (slope = 1: none):
 *     z[e,h] = scale * <Q[v(e),h,:], K[r(e),h,:] + Ke[e,h,:]>,   s = z > 0 ? z : slope*z,
 *     alpha  = per-(destination, head) softmax of s,   O[v,h,:] = sum alpha * (V[r(e),h,:] + Ve[e,h,:]).
 * Ke, Ve [E, H, D] DEVICE rows in CSR order (storage dtype, 16-byte aligned, required when E > 0).
 * Backward writes dQ [R,H,D], dK, dV [U,H,D] and the per-edge dKe, dVe [E,H,D] (dK[u], dV[u] are their sums over the
 * edges that reference row u).  Workspaces: the sizes tg_attn_workspace_bytes returns.  Same conventions as
 * tg_attn_fused_fwd / _bwd (async on `stream`, zero-degree destinations, error codes).
 * ---------------------------------------------------------------------------------------------- */
TG_API tg_status_t tg_attn_edge_fused_fwd(const tg_block_t* b, int H, int D, tg_dtype_t dtype,
                                          const void* Q, const void* K, const void* V, const void* Ke, const void* Ve,
                                          float scale, float slope, void* O, float* lse,
                                          void* ws, size_t ws_bytes, tg_stream_t stream);
TG_API tg_status_t tg_attn_edge_fused_bwd(const tg_block_t* b, int H, int D, tg_dtype_t dtype,
                                          const void* Q, const void* K, const void* V, const void* Ke, const void* Ve,
                                          const void* O, const float* lse, const void* dO, float scale, float slope,
                                          void* dQ, void* dK, void* dV, void* dKe, void* dVe,
                                          void* ws, size_t ws_bytes, tg_stream_t stream);

/* ------------------------------------------------------------------------------------------------
 * NEXT-2: SlimCache (section 4.2).
 *
 * tg_cache_greedy_select -- Algorithm 1, HOST only.  `n_batches` pre-sampled mini-batches, batch k's
 *   node ids node_ids[node_ptr[k] .. node_ptr[k+1]) and edge ids likewise (a batch counts an id once).  Picks, by
 *   descending access frequency (ties: ascending id; node vs edge tie: the edge), ids until i + j >= alpha*(n_nodes+n_edges).
 *   hot_nodes [>= n_nodes], hot_edges [>= n_edges] HOST outputs in selection order, counts in n_hot_nodes / n_hot_edges.
 * tg_cache_lookup -- runtime stage: uniq_ids[U] DEVICE int64 (a block's uniq_node, or unique edge ids),
 *   slot_of_id DEVICE int32 indexed by id (>= 0: row of the resident cache, < 0: not cached).  Writes map[U] DEVICE int32
 *   (>= 0: position among the rows to transfer; < 0: -(cache slot) - 1) and fresh_ids [>= U] DEVICE int64, the ids to
 *   transfer in the order of uniq_ids; *n_fresh_host = their number.  Synchronises the stream.
 * tg_feature_reconstruct -- out[i, :] = row of occurrence i: m = map[inv_idx ? inv_idx[i] : i];
 *   m >= 0 ? fresh_rows[m] : cache_rows[-m-1].  Rows of row_bytes bytes (multiple of 4; 16-byte vectors when the
 *   pointers and row_bytes allow), all DEVICE.  Async on `stream`.
 * ---------------------------------------------------------------------------------------------- */
TG_API tg_status_t tg_cache_greedy_select(double alpha, int64_t n_batches, const int64_t* node_ptr, const int64_t* node_ids,
                                          const int64_t* edge_ptr, const int64_t* edge_ids, int64_t n_nodes, int64_t n_edges,
                                          int64_t* hot_nodes, int64_t* n_hot_nodes, int64_t* hot_edges, int64_t* n_hot_edges);
TG_API tg_status_t tg_cache_lookup_workspace_bytes(int64_t U, size_t* bytes /*HOST*/);
TG_API tg_status_t tg_cache_lookup(int64_t U, const int64_t* uniq_ids, const int32_t* slot_of_id, int32_t* map, int64_t* fresh_ids,
                                   int64_t* n_fresh_host /*HOST*/, void* ws, size_t ws_bytes, tg_stream_t stream);
TG_API tg_status_t tg_feature_reconstruct(int64_t n, int64_t row_bytes, const int32_t* inv_idx, const int32_t* map,
                                          const void* fresh_rows, const void* cache_rows, void* out, tg_stream_t stream);

/* tg_cache_lookup for callers that cannot provide a workspace because they cannot allocate device memory at this point:
 * a serving process whose memory pool is fixed and fully assigned, a plug-in that receives tensors from a host framework
 * but has no allocator of its own, a latency-critical thread that must stay clear of cudaMalloc (which serialises the
 * device).  Same inputs, outputs and results as tg_cache_lookup; the scan's scratch is a fixed array inside the library
 * image instead of `ws`.
 *   Limit.    U <= TG_CACHE_STATIC_MAX_IDS (2^22 unique ids per call); a larger U returns TG_ERR_WORKSPACE with a message
 *             and launches nothing -- use tg_cache_lookup there.  The array is about 17 KB and stays resident on every GPU
 *             that uses this library, from first use until the process exits.
 *   Allocation. The call performs no cudaMalloc / cudaFree and calls no allocating library routine.
 *   First call. The first call on each device (with that device current) asks the runtime for the array's device address
 *             and caches it; make that first call outside any stream capture.  Later calls on the device only launch.
 *   Sharing.  Every call on a device uses the same array, whatever the stream or thread.  Nothing in it has to be cleared
 *             between calls (each call overwrites what it later reads), but two calls whose kernels may run at the same
 *             time on one GPU race on it: keep calls on one device ordered (one stream, or events between streams).  The
 *             call itself ends with a stream synchronisation, like tg_cache_lookup, so back-to-back calls from one
 *             thread are already ordered.
 * Errors: as tg_cache_lookup, plus TG_ERR_WORKSPACE (U beyond the limit) and TG_ERR_UNSUPPORTED (device ordinal >= 64). */
#define TG_CACHE_STATIC_MAX_IDS (1 << 22)
TG_API tg_status_t tg_cache_lookup_static(int64_t U, const int64_t* uniq_ids, const int32_t* slot_of_id, int32_t* map,
                                          int64_t* fresh_ids, int64_t* n_fresh_host /*HOST*/, tg_stream_t stream);

#ifdef __cplusplus
}
#endif
#endif /* FASTTG_H_ */
