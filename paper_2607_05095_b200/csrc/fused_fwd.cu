// fused_fwd.cu -- tg_attn_fused_fwd: SDDMM -> edge softmax -> alpha-weighted aggregation in one pass
// (DESIGN.md §2, §5.3).  s and alpha never reach HBM.
#include "dispatch.cuh"
#include "ops.cuh"

// Launch policy TierPolicy<U pipelined, min CTAs/SM pipelined, U plain, min CTAs/SM plain, U warp tier, resident warps/SM of the
// warp tier, warp tier pipelined>: two edges per trip everywhere; the values are the round-2 sweep's winners on config 4
// (profiles/r01_other_configs_and_probes.md lists the variants: U = 1, other occupancy caps, the HMMA logits of
// profiles/r02_hmma_probe.md -- all measured slower and no longer in the tree).
using FwdPolicy = TierPolicy<2, 2, 2, 3, 2, 16, true>;
using FwdPolicyNarrow = TierPolicy<2, 2, 2, 3, 2, 24, true>;   // one vector per lane (92 registers): 24 resident warps per SM
// Words of a gathered row per lane in the warp tier: bf16 rows of 256 bytes at 4 (LPR 16, one 16-byte vector per lane: half the
// buffer / accumulator registers of LPR 8), fp32 rows of 512 bytes at 4 (LPR 32; config 5: forward 5.98 -> 5.36 ms vs LPR 16).
// The group tiers use the warp tier's layout too (config 3: 53.4 -> 51.3 us per step; config 4 indifferent).
constexpr int TG_FWD_MAXW_BF16_256 = 4, TG_FWD_MAXW_F32_512 = 4;

struct FwdArgs {
    const tg_block* b;
    const void *Q, *K, *V;
    float scale;
    void* O;
    float* lse;
    void* ws;
    cudaStream_t stream;
    float* O32;
};

template <class Tr0>
struct FwdFn {
    static tg_status_t run(const FwdArgs& a) {
        using TrW = typename tg_relayout<Tr0, (Tr0::BF16 && Tr0::F * Tr0::EB == 256) ? TG_FWD_MAXW_BF16_256 : (!Tr0::BF16 && Tr0::F * Tr0::EB == 512) ? TG_FWD_MAXW_F32_512 : 8>::type;
        using Op = FwdOp<TrW>;
        using T = typename Tr0::T;
        typename Op::Params p;
        p.Q = static_cast<const T*>(a.Q); p.K = static_cast<const T*>(a.K); p.V = static_cast<const T*>(a.V);
        p.kv = a.b->kv_row;
        p.O = static_cast<T*>(a.O);
        p.lse = a.lse;
        p.part = static_cast<float*>(a.ws);
        p.scale2 = a.scale * TG_LOG2E;
        p.O32 = a.O32;
        if constexpr ((TrW::LPR == 16 && TrW::BF16) || (TrW::LPR == 32 && !TrW::BF16 && TrW::NW == 4))
            return tg_launch_tiers<Op, FwdPolicyNarrow>(p, a.b->dst, a.stream, "tg_attn_fused_fwd");
        else
            return tg_launch_tiers<Op, FwdPolicy>(p, a.b->dst, a.stream, "tg_attn_fused_fwd");
    }
};

extern "C" tg_status_t tg_attn_workspace_bytes(const tg_block_t* b, int H, int D, tg_dtype_t dtype, size_t* fwd_bytes,
                                               size_t* bwd_bytes) {
    TG_CHECK_PTR(b);
    tg_geom g;
    TG_TRY(tg_get_geom(H, D, dtype, &g));
    const tg_attn_ws_sizes s = tg_attn_ws(b, H, g);
    // the unfused aggregate calls reuse these workspaces: fwd needs NE*LPR per dst slot, bwd NE*LPR per src slot
    if (fwd_bytes) *fwd_bytes = tg_align_up(s.fwd_part) + 256;
    if (bwd_bytes) *bwd_bytes = tg_align_up(s.ld) + tg_align_up(s.dq_part) + tg_align_up(s.dkv_part) + 256;
    return TG_OK;
}

extern "C" tg_status_t tg_attn_fused_fwd(const tg_block_t* b, int H, int D, tg_dtype_t dtype, const void* Q, const void* K,
                                         const void* V, float scale, void* O, float* lse, float* o_f32, void* ws, size_t ws_bytes,
                                         tg_stream_t stream) {
    TG_CHECK_PTR(b);
    if (!tg_shape_supported(H, D, dtype)) TG_FAIL(TG_ERR_UNSUPPORTED, "unsupported (H=%d, D=%d, dtype=%d)", H, D, (int)dtype);
    if (b->R == 0) return TG_OK;
    TG_CHECK_ROWS(Q); TG_CHECK_ROWS(O); TG_CHECK_PTR(lse);
    if (b->E > 0) { TG_CHECK_ROWS(K); TG_CHECK_ROWS(V); }
    tg_geom g;
    TG_TRY(tg_get_geom(H, D, dtype, &g));
    const tg_attn_ws_sizes s = tg_attn_ws(b, H, g);
    if (s.fwd_part > 0 && (!ws || ws_bytes < s.fwd_part)) TG_FAIL(TG_ERR_WORKSPACE, "fused fwd needs %zu workspace bytes", s.fwd_part);
    if (o_f32 && (reinterpret_cast<uintptr_t>(o_f32) & 15u)) TG_FAIL(TG_ERR_ALIGNMENT, "o_f32 is not 16-byte aligned");
    FwdArgs a{b, Q, K, V, scale, O, lse, ws, static_cast<cudaStream_t>(stream), o_f32};
    return tg_dispatch<FwdFn>(H, D, dtype, a);
}
