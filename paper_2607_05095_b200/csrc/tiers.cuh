// tiers.cuh -- the degree-tiered driver shared by every row-gather operator.
//
// One launch covers a whole CSR side.  blockIdx selects the tier, largest work first:
//   [0, n_items)              cta tier  : one CTA per chunk (<= TG_CTA_CHUNK edges) of a large row; the 8
//                                         warps take contiguous sub-ranges, groups stride inside them,
//                                         states are merged by shuffles, then through shared memory;
//                                         a hub (row with several chunks) writes an fp32 partial
//   [.., + ceil(n_warp/8))    warp tier : one warp per row, its G groups stride over the row's edges
//   [.., + ceil(n_small/8G))  small tier: one group per row (deg <= TG_SMALL_MAX, the K<=10 common case)
// A second launch (tg_hub_kernel) merges the partials of each hub.
//
// An operator Op supplies: Tr (RowTraits), NS (fp32 state words per lane), Params, and
//   init_row(row), init_state(st), edges(st, i0, end, stride, trips), merge(a, b),
//   write_final(row, st, first), write_partial(slot, st, first), load_partial(slot, st)
// `trips` is warp-uniform so that the shuffles inside edges() are executed by all 32 lanes.
#pragma once
#include "rowops.cuh"

struct SideDev {
    const int32_t* indptr;
    const int32_t* order;
    const int4* items;
    const int4* hubs;
    int n_small, n_warp, n_items, n_hubs;
};

static inline SideDev tg_side_dev(const tg_side& s) {
    SideDev d;
    d.indptr = s.indptr; d.order = s.order; d.items = s.items; d.hubs = s.hubs;
    d.n_small = s.n_small; d.n_warp = s.n_warp; d.n_items = s.n_items; d.n_hubs = s.n_hubs;
    return d;
}

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

template <class Op>
__global__ void __launch_bounds__(TG_CTA_THREADS) tg_tier_kernel(typename Op::Params p, SideDev sd, int nb_warp) {
    using Tr = typename Op::Tr;
    __shared__ float sm[Op::NS > 0 ? TG_CTA_WARPS * Tr::LPR * Op::NS : 1];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane / Tr::LPR;
    Op op(p, lane % Tr::LPR);
    float st[Op::NS1];
    int bid = blockIdx.x;
    if (bid < sd.n_items) {
        const int4 it = sd.items[bid];
        const int n = it.z - it.y;
        const int per = (n + TG_CTA_WARPS - 1) / TG_CTA_WARPS;
        const int wb = min(it.y + warp * per, it.z), we = min(wb + per, it.z);
        op.init_row(it.x);
        op.init_state(st);
        const int trips = (we - wb + Tr::G * Op::UNR - 1) / (Tr::G * Op::UNR);
        op.edges(st, wb + g, we, Tr::G, trips);
        tg_warp_merge(op, st);
        tg_cta_merge(op, st, sm, warp, lane);
        if (warp == 0 && lane < Tr::LPR) {
            const bool first = (it.y == sd.indptr[it.x]);
            if (it.w < 0) op.write_final(it.x, st, first);
            else op.write_partial(it.w, st, first);
        }
    } else if ((bid -= sd.n_items) < nb_warp) {
        const int idx = bid * TG_CTA_WARPS + warp;
        if (idx >= sd.n_warp) return;
        const int row = sd.order[sd.n_small + idx];
        const int b = sd.indptr[row], e = sd.indptr[row + 1];
        op.init_row(row);
        op.init_state(st);
        const int trips = (e - b + Tr::G * Op::UNR - 1) / (Tr::G * Op::UNR);
        op.edges(st, b + g, e, Tr::G, trips);
        tg_warp_merge(op, st);
        if (lane < Tr::LPR) op.write_final(row, st, true);
    } else {
        bid -= nb_warp;
        const int idx = (bid * TG_CTA_WARPS + warp) * Tr::G + g;
        const bool active = idx < sd.n_small;
        const int row = active ? sd.order[idx] : 0;
        int b = 0, e = 0;
        if (active) { b = sd.indptr[row]; e = sd.indptr[row + 1]; }
        op.init_row(row);  // all lanes: init_row may shuffle (an idle group re-reads row 0)
        op.init_state(st);
        const int trips = __reduce_max_sync(0xffffffffu, (e - b + Op::UNR - 1) / Op::UNR);
        op.edges(st, b, e, 1, trips);
        if (active) op.write_final(row, st, true);
    }
}

// One CTA per hub: every (warp, group) folds a strided subset of the hub's partial slots.
template <class Op>
__global__ void __launch_bounds__(TG_CTA_THREADS) tg_hub_kernel(typename Op::Params p, SideDev sd) {
    using Tr = typename Op::Tr;
    static_assert(Op::NS > 0, "an operator without state has no partials");
    __shared__ float sm[TG_CTA_WARPS * Tr::LPR * Op::NS];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane / Tr::LPR;
    Op op(p, lane % Tr::LPR);
    const int4 hub = sd.hubs[blockIdx.x];  // row, first_slot, n_chunks
    float st[Op::NS];
    op.init_state(st);
    for (int c = warp * Tr::G + g; c < hub.z; c += TG_CTA_WARPS * Tr::G) {
        float other[Op::NS];
        op.load_partial(hub.y + c, other);
        op.merge(st, other);
    }
    tg_warp_merge(op, st);
    tg_cta_merge(op, st, sm, warp, lane);
    if (warp == 0 && lane < Tr::LPR) op.write_final(hub.x, st, false);
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

// Launch helper: tier kernel + (if the side has hubs) the hub merge.
template <class Op>
static tg_status_t tg_launch_tiers(const typename Op::Params& p, const tg_side& s, cudaStream_t stream, const char* name) {
    using Tr = typename Op::Tr;
    if (s.n_rows == 0) return TG_OK;
    SideDev sd = tg_side_dev(s);
    const int nb_warp = (s.n_warp + TG_CTA_WARPS - 1) / TG_CTA_WARPS;
    const int nb_small = (s.n_small + TG_CTA_WARPS * Tr::G - 1) / (TG_CTA_WARPS * Tr::G);
    const long long grid = (long long)s.n_items + nb_warp + nb_small;
    if (grid > 0x7fffffffLL) TG_FAIL(TG_ERR_INTERNAL, "%s: grid too large", name);
    if (grid > 0) {
        tg_tier_kernel<Op><<<(unsigned)grid, TG_CTA_THREADS, 0, stream>>>(p, sd, nb_warp);
        TG_LAUNCH_CHECK(name);
    }
    if constexpr (Op::NS > 0) {
        if (s.n_hubs > 0) {
            tg_hub_kernel<Op><<<(unsigned)s.n_hubs, TG_CTA_THREADS, 0, stream>>>(p, sd);
            TG_LAUNCH_CHECK(name);
        }
    }
    return TG_OK;
}
