// fused_edge.cu -- tg_attn_edge_fused_fwd / tg_attn_edge_fused_bwd: NEXT-1 of SURVEY.md §8(f), the full TGAT edge term
// (per-edge additive key / value rows + LeakyReLU on the logits).
//   forward : one pass, FwdEOp (online softmax fused with the aggregation, four gathered rows per edge)
//   backward: (1) Bwd1EOp, destination-major: delta, dQ, {lse2, delta} table
//             (2) BwdEdgeOp, destination-major, stateless: dKe[e], dVe[e] rows (bf16 only; fp32 writes them in pass 1)
//             (3) Bwd2EOp, source-major over the transposed CSR: dK, dV accumulated in fp32 from recomputed terms
#include "dispatch.cuh"
#include "ops_edge.cuh"

// single-buffer loops: four gathered rows per edge leave no registers for a second buffer
using EdgePolicy = TierPolicy<1, 2, 1, 2, 1, 16, false>;
#ifndef TG_EDGE_FWD_WARPS
#define TG_EDGE_FWD_WARPS 24
#endif
using EdgeFwdPolicy = TierPolicy<1, 2, 1, 2, 1, TG_EDGE_FWD_WARPS, false>;

struct EdgeArgs {
    const tg_block* b;
    const void *Q, *K, *V, *Ke, *Ve, *O, *dO;
    const float* lse_in;
    float scale, slope;
    void *Oout, *dQ, *dK, *dV, *dKe, *dVe;
    float* lse_out;
    void* ws;
    size_t ws_bytes;
    int H;
    cudaStream_t stream;
};

template <class Tr>
struct EdgeFwdFn {
    static tg_status_t run(const EdgeArgs& a) {
        using Op = FwdEOp<Tr>;
        using T = typename Tr::T;
        typename Op::Params p;
        p.Q = static_cast<const T*>(a.Q); p.K = static_cast<const T*>(a.K); p.V = static_cast<const T*>(a.V);
        p.Ke = static_cast<const T*>(a.Ke); p.Ve = static_cast<const T*>(a.Ve);
        p.kv = a.b->kv_row;
        p.O = static_cast<T*>(a.Oout); p.lse = a.lse_out; p.part = static_cast<float*>(a.ws);
        p.scale2 = a.scale * TG_LOG2E; p.slope = a.slope;
        return tg_launch_tiers<Op, EdgeFwdPolicy>(p, a.b->dst, a.stream, "tg_attn_edge_fused_fwd");
    }
};

template <class Tr>
struct EdgeBwdFn {
    static tg_status_t run(const EdgeArgs& a) {
        using T = typename Tr::T;
        tg_geom g{Tr::NE, Tr::LPR, Tr::NHL};
        const tg_attn_ws_sizes sz = tg_attn_ws(a.b, a.H, g);
        tg_carver c(a.ws, a.ws_bytes);
        float2* ld = static_cast<float2*>(c.take(sz.ld));
        float* dq_part = static_cast<float*>(c.take(sz.dq_part));
        float* agg_part = static_cast<float*>(c.take(sz.dkv_part));
        if (!c.ok()) TG_FAIL(TG_ERR_WORKSPACE, "edge-term bwd needs %zu workspace bytes", c.off);
        {
            using Op = Bwd1EOp<Tr>;
            typename Op::Params p;
            p.Q = static_cast<const T*>(a.Q); p.K = static_cast<const T*>(a.K); p.V = static_cast<const T*>(a.V);
            p.Ke = static_cast<const T*>(a.Ke); p.Ve = static_cast<const T*>(a.Ve);
            p.O = static_cast<const T*>(a.O); p.dO = static_cast<const T*>(a.dO);
            p.kv = a.b->kv_row; p.lse = a.lse_in;
            p.dQ = static_cast<T*>(a.dQ); p.ld = ld; p.part = dq_part;
            p.dKe = static_cast<T*>(a.dKe); p.dVe = static_cast<T*>(a.dVe);
            p.scale = a.scale; p.scale2 = a.scale * TG_LOG2E; p.slope = a.slope;
            TG_TRY((tg_launch_tiers<Op, EdgePolicy>(p, a.b->dst, a.stream, "tg_attn_edge_fused_bwd/dst")));
        }
        if constexpr (Tr::BF16) {   // bf16: delta comes from the edges and is final only now -> separate per-edge pass
            if (a.b->E > 0) {
            using Op = BwdEdgeOp<Tr>;
            typename Op::Params p;
            p.Q = static_cast<const T*>(a.Q); p.K = static_cast<const T*>(a.K); p.V = static_cast<const T*>(a.V);
            p.Ke = static_cast<const T*>(a.Ke); p.Ve = static_cast<const T*>(a.Ve); p.dO = static_cast<const T*>(a.dO);
            p.kv = a.b->kv_row; p.ld = ld;
            p.dKe = static_cast<T*>(a.dKe); p.dVe = static_cast<T*>(a.dVe);
            p.scale = a.scale; p.scale2 = a.scale * TG_LOG2E; p.slope = a.slope;
            TG_TRY((tg_launch_tiers<Op, EdgePolicy>(p, a.b->dst, a.stream, "tg_attn_edge_fused_bwd/edge")));
            }
        }
        if (a.b->E > 0) {
            using Op2 = Bwd2EOp<Tr>;
            typename Op2::Params q;
            q.Q = static_cast<const T*>(a.Q); q.K = static_cast<const T*>(a.K); q.V = static_cast<const T*>(a.V);
            q.Ke = static_cast<const T*>(a.Ke); q.Ve = static_cast<const T*>(a.Ve); q.dO = static_cast<const T*>(a.dO);
            q.t_dst = a.b->t_dst; q.t_edge = a.b->t_edge; q.ld = ld;
            q.dK = static_cast<T*>(a.dK); q.dV = static_cast<T*>(a.dV); q.part = agg_part;
            q.scale = a.scale; q.scale2 = a.scale * TG_LOG2E; q.slope = a.slope;
            TG_TRY((tg_launch_tiers<Op2, EdgePolicy>(q, a.b->src, a.stream, "tg_attn_edge_fused_bwd/src")));
        }
        return TG_OK;
    }
};

static tg_status_t edge_check(const tg_block_t* b, int H, int D, tg_dtype_t dtype) {
    TG_CHECK_PTR(b);
    if (!tg_shape_supported(H, D, dtype)) TG_FAIL(TG_ERR_UNSUPPORTED, "unsupported (H=%d, D=%d, dtype=%d)", H, D, (int)dtype);
    return TG_OK;
}

extern "C" tg_status_t tg_attn_edge_fused_fwd(const tg_block_t* b, int H, int D, tg_dtype_t dtype, const void* Q, const void* K,
                                              const void* V, const void* Ke, const void* Ve, float scale, float slope, void* O,
                                              float* lse, void* ws, size_t ws_bytes, tg_stream_t stream) {
    TG_TRY(edge_check(b, H, D, dtype));
    if (b->R == 0) return TG_OK;
    TG_CHECK_ROWS(Q); TG_CHECK_ROWS(O); TG_CHECK_PTR(lse);
    if (b->E > 0) { TG_CHECK_ROWS(K); TG_CHECK_ROWS(V); TG_CHECK_ROWS(Ke); TG_CHECK_ROWS(Ve); }
    tg_geom g;
    TG_TRY(tg_get_geom(H, D, dtype, &g));
    const tg_attn_ws_sizes s = tg_attn_ws(b, H, g);
    if (s.fwd_part > 0 && (!ws || ws_bytes < s.fwd_part)) TG_FAIL(TG_ERR_WORKSPACE, "edge-term fwd needs %zu workspace bytes", s.fwd_part);
    EdgeArgs a{};
    a.b = b; a.Q = Q; a.K = K; a.V = V; a.Ke = Ke; a.Ve = Ve; a.scale = scale; a.slope = slope;
    a.Oout = O; a.lse_out = lse; a.ws = ws; a.ws_bytes = ws_bytes; a.H = H; a.stream = static_cast<cudaStream_t>(stream);
    return tg_dispatch<EdgeFwdFn>(H, D, dtype, a);
}

extern "C" tg_status_t tg_attn_edge_fused_bwd(const tg_block_t* b, int H, int D, tg_dtype_t dtype, const void* Q, const void* K,
                                              const void* V, const void* Ke, const void* Ve, const void* O, const float* lse,
                                              const void* dO, float scale, float slope, void* dQ, void* dK, void* dV, void* dKe,
                                              void* dVe, void* ws, size_t ws_bytes, tg_stream_t stream) {
    TG_TRY(edge_check(b, H, D, dtype));
    if (b->R == 0) return TG_OK;
    TG_CHECK_ROWS(Q); TG_CHECK_ROWS(O); TG_CHECK_ROWS(dO); TG_CHECK_ROWS(dQ); TG_CHECK_PTR(lse);
    if (b->E > 0) {
        TG_CHECK_ROWS(K); TG_CHECK_ROWS(V); TG_CHECK_ROWS(Ke); TG_CHECK_ROWS(Ve);
        TG_CHECK_ROWS(dK); TG_CHECK_ROWS(dV); TG_CHECK_ROWS(dKe); TG_CHECK_ROWS(dVe);
    }
    if (!ws) TG_FAIL(TG_ERR_WORKSPACE, "edge-term bwd needs a workspace (tg_attn_workspace_bytes)");
    EdgeArgs a{};
    a.b = b; a.Q = Q; a.K = K; a.V = V; a.Ke = Ke; a.Ve = Ve; a.O = O; a.dO = dO; a.lse_in = lse; a.scale = scale; a.slope = slope;
    a.dQ = dQ; a.dK = dK; a.dV = dV; a.dKe = dKe; a.dVe = dVe; a.ws = ws; a.ws_bytes = ws_bytes; a.H = H;
    a.stream = static_cast<cudaStream_t>(stream);
    return tg_dispatch<EdgeBwdFn>(H, D, dtype, a);
}
