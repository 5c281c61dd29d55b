// fused_fwd.cu -- tg_attn_fused_fwd: SDDMM -> edge softmax -> alpha-weighted aggregation in one pass
// (DESIGN.md §2, §5.3).  s and alpha never reach HBM.
#include "dispatch.cuh"
#include "ops_mma.cuh"

// launch policy {edges per trip, min CTAs per SM} for the pipelined and the plain kernel variants
#ifndef TG_FWD_U
#define TG_FWD_U 2
#endif
#ifndef TG_FWD_CTAS
#define TG_FWD_CTAS 2
#endif
#ifndef TG_FWD_UP
#define TG_FWD_UP 2
#endif
#ifndef TG_FWD_CTASP
#define TG_FWD_CTASP 3
#endif
#ifndef TG_FWD_UW
#define TG_FWD_UW TG_FWD_U
#endif
#ifndef TG_FWD_WARPSW
#define TG_FWD_WARPSW (8 * TG_FWD_CTAS)
#endif
#ifndef TG_FWD_WPIPE
#define TG_FWD_WPIPE true
#endif
// 1: bf16 rows of 256 bytes with D in {16, 32}: the warp tier takes its logits from HMMA (ops_mma.cuh); 0 (default): FHFMA.
// Measured on config 4 (profiles/r02_hmma_probe.md): parity green, 6 % fewer instructions, but 0.365 -> 0.396 ms: the
// dependent HMMA chain (23 cycles each) and the block-diagonal padding cost more issue time than the FHFMA they replace.
#ifndef TG_FWD_MMA
#define TG_FWD_MMA 0
#endif
#define TG_FWD_POLICY TG_FWD_U, TG_FWD_CTAS, TG_FWD_UP, TG_FWD_CTASP, TG_FWD_UW, TG_FWD_WARPSW, TG_FWD_WPIPE

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

#ifndef TG_FWD_GROUP_RELAYOUT
#define TG_FWD_GROUP_RELAYOUT 1   // 1: the group tiers use the warp tier's layout too (config 3: 53.4 -> 51.3 us; config 4 indifferent)
#endif
#ifndef TG_FWD_MAXW
#define TG_FWD_MAXW 4   // words of a gathered 256-byte bf16 row per lane (8: LPR 8, 4: LPR 16), see fused_bwd.cu
#endif
#ifndef TG_FWD_MAXW_F32
#define TG_FWD_MAXW_F32 4   // the same knob for fp32 rows of 512 bytes: 4 = LPR 32 (config 5: forward 5.98 -> 5.36 ms), 8 = LPR 16
#endif
#ifndef TG_FWD_WARPSW16
#define TG_FWD_WARPSW16 24   // resident warps per SM of the warp tier in the LPR-16 layout (92 registers)
#endif
template <class Tr0>
struct FwdFn {
    static tg_status_t run(const FwdArgs& a) {
        // group tiers: default layout (LPR 8: four rows per warp instruction); warp tier + hub merges: bf16 rows of 256 bytes in the
        // LPR-16 layout (one vector per lane, half the buffer / accumulator registers, 24 resident warps)
        using TrW = typename tg_relayout<Tr0, (Tr0::BF16 && Tr0::F * Tr0::EB == 256) ? TG_FWD_MAXW : (!Tr0::BF16 && Tr0::F * Tr0::EB == 512) ? TG_FWD_MAXW_F32 : 8>::type;
        using TrG = typename std::conditional<TG_FWD_GROUP_RELAYOUT != 0, TrW, Tr0>::type;
        using Op = FwdOp<TrG>;
        using OpW = typename tg_warp_op<FwdOp<TrW>, (TG_FWD_MMA != 0) && MmaDotOk<TrW>::value>::type;
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
            return tg_launch_tiers<Op, TierPolicy<TG_FWD_U, TG_FWD_CTAS, TG_FWD_UP, TG_FWD_CTASP, TG_FWD_UW, TG_FWD_WARPSW16, TG_FWD_WPIPE>, OpW>(p, a.b->dst, a.stream, "tg_attn_fused_fwd");
        else
            return tg_launch_tiers<Op, TierPolicy<TG_FWD_POLICY>, OpW>(p, a.b->dst, a.stream, "tg_attn_fused_fwd");
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
