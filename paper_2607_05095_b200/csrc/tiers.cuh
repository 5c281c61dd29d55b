// tiers.cuh -- the degree-tiered driver shared by every row-gather operator.
//
// A CSR side with >= TG_FORK_MIN_EDGES edges is covered by these launches (largest work first):
//   tg_warp_kernel      warp tier : one warp per chunk (<= tg_side::chunk edges) of a large row; its G groups stride over
//                                   the chunk's edges, states are merged by shuffles; a hub (row with several chunks)
//                                   writes an fp32 partial per chunk.  1-warp CTAs, items sorted longest first.
//   tg_hub_warp_kernel  one warp per hub with <= TG_HUB_DIRECT chunks folds its partials
//   tg_hub_kernel       two-level fold of the few big hubs (TG_HUB_SPLIT CTAs per hub, then one)
//   tg_group_kernel x2  group tier: one group per row, degree classes 9..TG_GROUP_MAX (pipelined edge loop) and classes
//                                   <= 8 (plain edge loop, small register budget: these rows are pure latency chains);
//                                   both run on auxiliary streams beside the warp tier (fork / join by events)
// A smaller side is launch-latency bound and runs the warp tier and both group tiers in ONE launch (tg_small_side_kernel).
// Rows of one class are contiguous in the schedule, so the groups of a warp run the same number of trips.
//
// An operator Op supplies: Tr (RowTraits), NS (fp32 state words per lane), Params, and
//   idx_ptr()                     the per-edge row index array of this side (kv_row or t_dst)
//   Buf, load(buf, r, pos)        the gathered operands of one edge (row index r, edge position pos)
//   compute<U, MASK>(st, buf[U], pos0, stride, end)   fold U edges pos0 + u*stride into st; MASK: edges
//                                                      at positions >= end are ignored
//   init_row(row), init_state(st), merge(a, b),
//   write_final(row, st, first), write_partial(slot, st, first), load_partial(slot, st)
// Every warp-wide call (compute, merge) is reached by all 32 lanes with warp-uniform trip counts.
#pragma once
#include <string.h>

#include <type_traits>

#include "rowops.cuh"

template <class Op>
__device__ __forceinline__ void tg_warp_merge(Op& op, float (&st)[Op::NS1]) {
    using Tr = typename Op::Tr;
    if constexpr (Op::NS > 0) {
#pragma unroll
        for (int o = Tr::LPR; o < 32; o <<= 1) {
            float other[Op::NS];
#pragma unroll
            for (int i = 0; i < Op::NS; ++i) other[i] = __shfl_xor_sync(0xffffffffu, st[i], o);
            op.merge(st, other);
        }
    }
}

// CTA-wide merge through shared memory; the result lands in warp 0, lanes < LPR.  All threads call.
template <class Op>
__device__ __forceinline__ void tg_cta_merge(Op& op, float (&st)[Op::NS1], float* sm, int warp, int lane) {
    using Tr = typename Op::Tr;
    if constexpr (Op::NS > 0) {
        if (lane < Tr::LPR) {
#pragma unroll
            for (int i = 0; i < Op::NS; ++i) sm[(warp * Op::NS + i) * Tr::LPR + lane] = st[i];
        }
        __syncthreads();
        if (warp == 0 && lane < Tr::LPR) {
            for (int w = 1; w < TG_CTA_WARPS; ++w) {
                float other[Op::NS];
#pragma unroll
                for (int i = 0; i < Op::NS; ++i) other[i] = sm[(w * Op::NS + i) * Tr::LPR + lane];
                op.merge(st, other);
            }
        }
    }
}

// Where an edge loop takes its row indices from: global memory, positions clamped to the row's last edge.  (A chunk staged
// in shared memory was measured in round 2 and brought nothing on config 4: profiles/r01_other_configs_and_probes.md.)
struct tg_idx_global {
    const int32_t* __restrict__ p;
    int last;
    __device__ __forceinline__ int operator()(int pos) const { return tg_ldg_i32(p + min(pos, last)); }
};

// Plain edge loop of one group: edges pos = i0 + n*stride < end, U per trip, all loads of a trip issued
// before its arithmetic.  Latency is hidden by the other warps (small register budget).
template <int U, class Op>
__device__ __forceinline__ void tg_run_edges_plain(Op& op, float (&st)[Op::NS1], int i0, int end, int stride, int trips) {
    if (trips <= 0) return;
    const int last = max(end - 1, 0);
    const tg_idx_global idx{op.idx_ptr(), last};
    int pos = i0;
    for (int t = 0; t < trips; ++t) {
        typename Op::Buf A[U];
        int r[U];
#pragma unroll
        for (int u = 0; u < U; ++u) r[u] = idx(pos + u * stride);
#pragma unroll
        for (int u = 0; u < U; ++u) op.load(A[u], r[u], min(pos + u * stride, last));
        op.template compute<U, true>(st, A, pos, stride, end);
        pos += U * stride;
    }
}

// Software-pipelined edge loop with two register buffers: while trip t is computed the rows of trip t+1
// are in flight, so a warp exposes the gather latency once per loop, not once per trip.  The row indices
// are requested a whole iteration (two trips) before the row loads that use them: the per-edge index
// stream enters a new 32-byte sector every few trips, each first touch is an L2/DRAM round trip, and a
// single trip of lead does not cover it (measured: 25 % of the warp tier's stall samples sat on the
// index -> address dependency).  Positions past `end` are clamped for the loads (a valid row is fetched
// again) and masked in compute().  `full_until`: trips whose first position is below it need no mask
// (warp-uniform; pass i0 to mask everything).
template <int U, class Op, class Idx>
__device__ __forceinline__ void tg_run_edges_pipe_from(Op& op, float (&st)[Op::NS1], const Idx& idx, int i0, int end, int stride, int trips,
                                                       int full_until) {
    if (trips <= 0) return;
    const int last = max(end - 1, 0);
    typename Op::Buf A[U], B[U];
    int ia[U], ib[U], na[U], nb[U];   // indices of trips t+2, t+1 (used this iteration) and t+4, t+3 (next one)
    const int step = U * stride;
    int pos = i0;  // first position of the trip being computed
#pragma unroll
    for (int u = 0; u < U; ++u) na[u] = idx(pos + u * stride);
#pragma unroll
    for (int u = 0; u < U; ++u) ib[u] = idx(pos + step + u * stride);
#pragma unroll
    for (int u = 0; u < U; ++u) ia[u] = idx(pos + 2 * step + u * stride);
#pragma unroll
    for (int u = 0; u < U; ++u) op.load(A[u], na[u], min(pos + u * stride, last));
    for (int t = 0; t < trips; t += 2) {
#pragma unroll
        for (int u = 0; u < U; ++u) nb[u] = idx(pos + 3 * step + u * stride);
#pragma unroll
        for (int u = 0; u < U; ++u) na[u] = idx(pos + 4 * step + u * stride);
        if (t + 1 < trips) {
#pragma unroll
            for (int u = 0; u < U; ++u) op.load(B[u], ib[u], min(pos + step + u * stride, last));
        }
        if (pos < full_until) op.template compute<U, false>(st, A, pos, stride, end);
        else op.template compute<U, true>(st, A, pos, stride, end);
        if (t + 1 < trips) {
            if (t + 2 < trips) {
#pragma unroll
                for (int u = 0; u < U; ++u) op.load(A[u], ia[u], min(pos + 2 * step + u * stride, last));
            }
            if (pos + step < full_until) op.template compute<U, false>(st, B, pos + step, stride, end);
            else op.template compute<U, true>(st, B, pos + step, stride, end);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) { ia[u] = na[u]; ib[u] = nb[u]; }
        pos += 2 * step;
    }
}

template <int U, class Op>
__device__ __forceinline__ void tg_run_edges_pipe(Op& op, float (&st)[Op::NS1], int i0, int end, int stride, int trips, int full_until) {
    tg_run_edges_pipe_from<U>(op, st, tg_idx_global{op.idx_ptr(), max(end - 1, 0)}, i0, end, stride, trips, full_until);
}

// Warp tier: one warp per item {row, begin, end, slot}.  The warps of a CTA are independent; a CTA holds
// TG_WARP_CTA_WARPS of them (its registers are released only when its slowest warp ends, so smaller is better
// for the tail) and MIN_WARPS / TG_WARP_CTA_WARPS such CTAs are resident per SM.
#ifndef TG_WARP_CTA_WARPS
#define TG_WARP_CTA_WARPS 1
#endif
template <class Op, int U, bool PIPE>
__device__ __forceinline__ void tg_warp_body(const typename Op::Params& p, const int4* __restrict__ items,
                                             const int32_t* __restrict__ indptr, int n_items, int idx) {
    using Tr = typename Op::Tr;
    const int lane = threadIdx.x & 31;
    const int g = lane / Tr::LPR;
    if (idx >= n_items) return;
    const int4 it = items[idx];
    Op op(p, lane % Tr::LPR);
    float st[Op::NS1];
    op.init_row(it.x);
    op.init_state(st);
    const int n = it.z - it.y;
    const int trips = (n + Tr::G * U - 1) / (Tr::G * U);
    // a trip is full for every group when its last position (group G-1, edge U-1) is inside the chunk
    const int full_until = it.y + g + ((n / (Tr::G * U)) * (Tr::G * U));
    if constexpr (PIPE) tg_run_edges_pipe<U>(op, st, it.y + g, it.z, Tr::G, trips, full_until);
    else tg_run_edges_plain<U>(op, st, it.y + g, it.z, Tr::G, trips);
    tg_warp_merge(op, st);
    if (lane < Tr::LPR) {
        if (it.w < 0) op.write_final(it.x, st, true);
        else op.write_partial(it.w, st, it.y == indptr[it.x]);
    }
}
template <class Op, int U, int MIN_WARPS, bool PIPE>
__global__ void __launch_bounds__(TG_WARP_CTA_WARPS * 32, MIN_WARPS / TG_WARP_CTA_WARPS) tg_warp_kernel(typename Op::Params p, const int4* __restrict__ items,
                                                                           const int32_t* __restrict__ indptr, int n_items) {
    tg_warp_body<Op, U, PIPE>(p, items, indptr, n_items, blockIdx.x * TG_WARP_CTA_WARPS + (threadIdx.x >> 5));
}

// Group tier: one group per record {row, begin, end, 0}; TG_GROUP_CTA_WARPS independent warps per CTA.
#ifndef TG_GROUP_CTA_WARPS
#define TG_GROUP_CTA_WARPS 2
#endif
template <class Op, int U, bool PIPE>
__device__ __forceinline__ void tg_group_body(const typename Op::Params& p, const int4* __restrict__ rows, int n_rows, int warp_idx) {
    using Tr = typename Op::Tr;
    const int lane = threadIdx.x & 31;
    const int g = lane / Tr::LPR;
    const int idx = warp_idx * Tr::G + g;
    if (idx - g >= n_rows) return;  // the whole warp is idle
    const bool active = idx < n_rows;
    int4 it = make_int4(0, 0, 0, 0);  // an idle group re-reads row 0 and writes nothing
    if (active) it = rows[idx];
    Op op(p, lane % Tr::LPR);
    float st[Op::NS1];
    op.init_row(it.x);
    op.init_state(st);
    const int trips = __reduce_max_sync(0xffffffffu, (it.z - it.y + U - 1) / U);
    if constexpr (PIPE) tg_run_edges_pipe<U>(op, st, it.y, it.z, 1, trips, it.y);
    else tg_run_edges_plain<U>(op, st, it.y, it.z, 1, trips);
    if (active) op.write_final(it.x, st, true);
}
template <class Op, int U, int MIN_CTAS, bool PIPE>
__global__ void __launch_bounds__(TG_GROUP_CTA_WARPS * 32, MIN_CTAS * 8 / TG_GROUP_CTA_WARPS) tg_group_kernel(typename Op::Params p, const int4* __restrict__ rows,
                                                                            int n_rows) {
    tg_group_body<Op, U, PIPE>(p, rows, n_rows, blockIdx.x * TG_GROUP_CTA_WARPS + (threadIdx.x >> 5));
}

// Small sides (< TG_FORK_MIN_EDGES edges: the K <= 10-20 blocks of configs 1-3) are launch-latency bound: one launch
// covers the warp tier and both group tiers, 2 independent warps per CTA, blockIdx selects the tier (largest work first).
template <class Op, class OpW, int UW, int UB, int US, bool WARP_PIPE>
__global__ void __launch_bounds__(64, 8) tg_small_side_kernel(typename Op::Params p, typename OpW::Params pw, const int4* __restrict__ items, const int32_t* __restrict__ indptr,
                                                              int n_items, const int4* __restrict__ rows, int n_big, int n_small, int nb_items, int nb_big) {
    const int warp = threadIdx.x >> 5;
    int b = blockIdx.x;
    if (b < nb_items) { tg_warp_body<OpW, UW, WARP_PIPE>(pw, items, indptr, n_items, b * 2 + warp); return; }
    b -= nb_items;
    if (b < nb_big) { tg_group_body<Op, UB, WARP_PIPE>(p, rows, n_big, b * 2 + warp); return; }
    b -= nb_big;
    tg_group_body<Op, US, false>(p, rows + n_big, n_small, b * 2 + warp);
}

// Folds the partial slots first + c, c = c0, c0 + step, ... < n into st.  Four partials are requested before the first
// merge: a hub with hundreds of chunks is otherwise one round trip to L2 / HBM per partial (config 3's hottest source
// row: 18 us for a 0.6 M-instruction launch).
template <class Op>
__device__ __forceinline__ void tg_fold_partials(Op& op, float (&st)[Op::NS], int first, int c0, int n, int step) {
    constexpr int UNR = 4;
    for (int c = c0; c < n; c += UNR * step) {
        float other[UNR][Op::NS];
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            if (c + u * step < n) op.load_partial(first + c + u * step, other[u]);
            else op.init_state(other[u]);       // the identity of merge()
        }
#pragma unroll
        for (int u = 0; u < UNR; ++u) op.merge(st, other[u]);
    }
}

// Hub merge.  A hub with <= TG_HUB_DIRECT chunks is folded by one warp (tg_hub_warp_kernel).  Larger hubs (a hot
// source row can have thousands of chunks) are folded in two levels by tg_hub_kernel: TG_HUB_SPLIT CTAs per hub
// write second-level partials (slots n_slots + hub*TG_HUB_SPLIT + j; level 1, blockIdx.y = j), then one CTA per hub
// folds those (level 2); they run over the schedule's separate list of big hubs.  On a small (launch-bound) side one
// CTA per hub folds everything in a single launch (level 0).

// Small hubs (<= TG_HUB_DIRECT chunks -- nearly all of them: a destination of config 4 has at most 8): one WARP per
// hub, its G groups stride over the partial slots, shuffle merge, no shared memory and no barrier.
constexpr int TG_HUBW_WARPS = 4;
template <class Op>
__global__ void __launch_bounds__(TG_HUBW_WARPS * 32) tg_hub_warp_kernel(typename Op::Params p, const int4* __restrict__ hubs, int n_hubs) {
    using Tr = typename Op::Tr;
    static_assert(Op::NS > 0, "an operator without state has no partials");
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane / Tr::LPR;
    const int idx = blockIdx.x * TG_HUBW_WARPS + warp;
    if (idx >= n_hubs) return;
    const int4 hub = hubs[idx];  // row, first_slot, n_chunks
    if (hub.z > TG_HUB_DIRECT) return;   // folded by the two-level tg_hub_kernel
    Op op(p, lane % Tr::LPR);
    float st[Op::NS];
    op.init_state(st);
    tg_fold_partials<Op>(op, st, hub.y, g, hub.z, Tr::G);
    tg_warp_merge(op, st);
    if (lane < Tr::LPR) op.write_final(hub.x, st, false);
}

template <class Op>
__global__ void __launch_bounds__(TG_CTA_THREADS) tg_hub_kernel(typename Op::Params p, const int4* __restrict__ hubs, int n_slots,
                                                                int level) {
    using Tr = typename Op::Tr;
    static_assert(Op::NS > 0, "an operator without state has no partials");
    __shared__ float sm[TG_CTA_WARPS * Tr::LPR * Op::NS];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane / Tr::LPR;
    const int4 hub = hubs[blockIdx.x];  // row, first_slot, n_chunks (levels 1, 2: the list of big hubs)
    int first = hub.y, n = hub.z, start = 0, stride = 1, out_slot = -1;   // level 0: one CTA folds the whole hub
    if (level == 1) {
        start = blockIdx.y; stride = TG_HUB_SPLIT; out_slot = n_slots + blockIdx.x * TG_HUB_SPLIT + blockIdx.y;
    } else if (level == 2) {
        first = n_slots + blockIdx.x * TG_HUB_SPLIT; n = TG_HUB_SPLIT;
    }
    Op op(p, lane % Tr::LPR);
    float st[Op::NS];
    op.init_state(st);
    tg_fold_partials<Op>(op, st, first, start + (warp * Tr::G + g) * stride, n, TG_CTA_WARPS * Tr::G * stride);
    tg_warp_merge(op, st);
    tg_cta_merge(op, st, sm, warp, lane);
    if (warp == 0 && lane < Tr::LPR) {
        if (out_slot < 0) op.write_final(hub.x, st, false);
        else op.write_partial(out_slot, st, false);
    }
}

// generic partial store / load: [slot][NS][LPR] fp32, lane-minor
template <class Tr, int NS>
__device__ __forceinline__ void tg_partial_store(float* part, int slot, int lig, const float (&st)[NS]) {
    float* p = part + (size_t)slot * NS * Tr::LPR + lig;
#pragma unroll
    for (int i = 0; i < NS; ++i) p[i * Tr::LPR] = st[i];
}
template <class Tr, int NS>
__device__ __forceinline__ void tg_partial_load(const float* part, int slot, int lig, float (&st)[NS]) {
    const float* p = part + (size_t)slot * NS * Tr::LPR + lig;
#pragma unroll
    for (int i = 0; i < NS; ++i) st[i] = p[i * Tr::LPR];
}

// Launch policy of one operator: edges per trip (U) and minimum resident CTAs per SM for the pipelined
// (warp tier, big group classes) and the plain (small group classes) variants.
template <int U_PIPE_, int CTAS_PIPE_, int U_PLAIN_, int CTAS_PLAIN_, int U_WARP_ = U_PIPE_, int WARPS_WARP_ = 8 * CTAS_PIPE_, bool WARP_PIPE_ = true>
struct TierPolicy {
    static constexpr int U_PIPE = U_PIPE_, CTAS_PIPE = CTAS_PIPE_, U_PLAIN = U_PLAIN_, CTAS_PLAIN = CTAS_PLAIN_;
    static constexpr int U_WARP = U_WARP_, WARPS_WARP = WARPS_WARP_;   // warp tier: edges per trip, resident warps per SM, pipelined or plain loop
    static constexpr bool WARP_PIPE = WARP_PIPE_;
};

template <class Op>
static tg_status_t tg_launch_hub_merge(const typename Op::Params& p, const tg_side& s, cudaStream_t stream, const char* name) {
    if (s.n_hubs <= 0) return TG_OK;
    if (s.n_edges < TG_FORK_MIN_EDGES) {   // launch-bound small side: one CTA per hub, whatever its size, in a single launch
        tg_hub_kernel<Op><<<(unsigned)s.n_hubs, TG_CTA_THREADS, 0, stream>>>(p, s.hubs, s.n_slots, 0);
        TG_LAUNCH_CHECK(name);
        return TG_OK;
    }
    tg_hub_warp_kernel<Op><<<(unsigned)((s.n_hubs + TG_HUBW_WARPS - 1) / TG_HUBW_WARPS), TG_HUBW_WARPS * 32, 0, stream>>>(p, s.hubs, s.n_hubs);
    TG_LAUNCH_CHECK(name);
    if (s.n_bighubs > 0) {
        tg_hub_kernel<Op><<<dim3((unsigned)s.n_bighubs, TG_HUB_SPLIT), TG_CTA_THREADS, 0, stream>>>(p, s.bighubs, s.n_slots, 1);
        TG_LAUNCH_CHECK(name);
        tg_hub_kernel<Op><<<(unsigned)s.n_bighubs, TG_CTA_THREADS, 0, stream>>>(p, s.bighubs, s.n_slots, 2);
        TG_LAUNCH_CHECK(name);
    }
    return TG_OK;
}

// Launch helper: all tiers of one side.  The group tiers touch other rows than the warp tier: on a large side
// they run on two auxiliary streams forked from and joined back into the caller's stream, so that each launch's
// tail is filled by the others (the fork / join is a plain event pattern and can be captured into a CUDA graph).
// OpW: the operator of the warp tier (same Params, same state layout outside the edge loop; e.g. the HMMA variants of ops_mma.cuh).
template <class Op, class Pol, class OpW = Op>
static tg_status_t tg_launch_tiers(const typename Op::Params& p, const tg_side& s, cudaStream_t stream, const char* name) {
    // The warp tier (and the hub merges, which read its partials) may run the operator in another lane layout than the group
    // tiers: Params hold only pointers and scalars, field for field the same whatever the layout.
    static_assert(sizeof(typename Op::Params) == sizeof(typename OpW::Params) && std::is_trivially_copyable<typename Op::Params>::value &&
                      std::is_trivially_copyable<typename OpW::Params>::value, "warp-tier operator must share the Params fields");
    typename OpW::Params pw;
    memcpy(&pw, &p, sizeof(pw));
    using Tr = typename Op::Tr;
    if (s.n_rows == 0) return TG_OK;
    constexpr int rows_per_cta = TG_GROUP_CTA_WARPS * Tr::G;
    const int n_big = s.n_group_big(), n_small = s.n_group_small();
    if (s.n_edges < TG_FORK_MIN_EDGES) {
        const int nb_items = (s.n_items + 1) / 2, nb_big = (n_big + 2 * Tr::G - 1) / (2 * Tr::G), nb_small = (n_small + 2 * Tr::G - 1) / (2 * Tr::G);
        if (nb_items + nb_big + nb_small > 0) {
            tg_small_side_kernel<Op, OpW, Pol::U_WARP, Pol::U_PIPE, Pol::U_PLAIN, Pol::WARP_PIPE><<<(unsigned)(nb_items + nb_big + nb_small), 64, 0, stream>>>(
                p, pw, s.items, s.indptr, s.n_items, s.rows, n_big, n_small, nb_items, nb_big);
            TG_LAUNCH_CHECK(name);
        }
        if constexpr (Op::NS > 0) TG_TRY((tg_launch_hub_merge<OpW>(pw, s, stream, name)));
        return TG_OK;
    }
    const bool fork = s.n_items > 0 && (n_big > 0 || n_small > 0);
    tg_aux_streams* aux = nullptr;
    if (fork) {
        aux = tg_get_aux_streams();
        if (!aux) return TG_ERR_CUDA;
        TG_CUDA(cudaEventRecord(aux->fork, stream));
    }
    // After the fork every path joins the auxiliary streams back, error or not (an unjoined fork would invalidate a stream
    // capture and break "the call behaves like one kernel on `stream`"): the first error is kept and returned at the end.
    tg_status_t st = TG_OK;
    bool forked[2] = {false, false};
    auto launch_all = [&]() -> tg_status_t {
        if (s.n_items > 0) {
            const unsigned grid = (unsigned)((s.n_items + TG_WARP_CTA_WARPS - 1) / TG_WARP_CTA_WARPS);
            tg_warp_kernel<OpW, Pol::U_WARP, Pol::WARPS_WARP, Pol::WARP_PIPE><<<grid, TG_WARP_CTA_WARPS * 32, 0, stream>>>(pw, s.items, s.indptr, s.n_items);
            TG_LAUNCH_CHECK(name);
        }
        if (n_big > 0) {
            cudaStream_t sx = fork ? aux->s[0] : stream;
            if (fork) { TG_CUDA(cudaStreamWaitEvent(sx, aux->fork, 0)); forked[0] = true; }
            const unsigned grid = (unsigned)((n_big + rows_per_cta - 1) / rows_per_cta);
            tg_group_kernel<Op, Pol::U_PIPE, Pol::CTAS_PIPE, Pol::WARP_PIPE><<<grid, TG_GROUP_CTA_WARPS * 32, 0, sx>>>(p, s.rows, n_big);
            TG_LAUNCH_CHECK(name);
        }
        if (n_small > 0) {
            cudaStream_t sx = fork ? aux->s[1] : stream;
            if (fork) { TG_CUDA(cudaStreamWaitEvent(sx, aux->fork, 0)); forked[1] = true; }
            const unsigned grid = (unsigned)((n_small + rows_per_cta - 1) / rows_per_cta);
            tg_group_kernel<Op, Pol::U_PLAIN, Pol::CTAS_PLAIN, false><<<grid, TG_GROUP_CTA_WARPS * 32, 0, sx>>>(p, s.rows + n_big, n_small);
            TG_LAUNCH_CHECK(name);
        }
        if constexpr (Op::NS > 0) TG_TRY((tg_launch_hub_merge<OpW>(pw, s, stream, name)));
        return TG_OK;
    };
    st = launch_all();
    for (int i = 0; i < 2; ++i) {
        if (!forked[i]) continue;
        if (cudaEventRecord(aux->join[i], aux->s[i]) != cudaSuccess || cudaStreamWaitEvent(stream, aux->join[i], 0) != cudaSuccess) {
            if (st == TG_OK) { tg_set_error("%s: joining the auxiliary stream failed: %s", name, cudaGetErrorString(cudaGetLastError())); st = TG_ERR_CUDA; }
        }
    }
    return st;
}
