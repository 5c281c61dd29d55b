// fused_bwd.cu -- tg_attn_fused_bwd ("forward and backward"; formulas DESIGN.md §2).
// Pass 1, destination-major: delta, dQ (and the {lse2, delta} table).  Pass 2, source-major over the
// transposed CSR: dK, dV by gather -- no float atomics, run-to-run bitwise reproducible.
#include "dispatch.cuh"
#include "ops.cuh"

// Launch policies (TierPolicy<U pipelined, min CTAs/SM pipelined, U plain, min CTAs/SM plain, U warp tier, resident warps/SM of
// the warp tier, warp tier pipelined>): one edge per trip in both passes.  The values are the round-2 sweep's winners on
// configs 4 / 5; the alternatives (U = 2, other occupancy caps, source-major loop variants, HMMA dot products) are recorded
// in profiles/r01_other_configs_and_probes.md and profiles/r02_hmma_probe.md and are no longer in the tree.
using BwdPolicy = TierPolicy<1, 2, 1, 3, 1, 16, true>;
using BwdPolicyNarrow = TierPolicy<1, 2, 1, 3, 1, 24, true>;    // one vector per lane: 24 resident warps per SM
using BwdPolicyWide = TierPolicy<1, 2, 1, 2, 1, 16, false>;     // fp32 rows at 16 words per lane: single-buffered loops
// Words of a gathered row per lane.  bf16 rows of 256 bytes: 8 = LPR 8 (two vectors per lane), 4 = LPR 16 (one vector per lane:
// half the buffer / accumulator registers, the same instructions per edge, 24 instead of 16 resident warps).  Measured on
// config 4: destination-major 0.475 -> 0.450 ms at LPR 16, source-major 0.539 -> 0.592 ms -- so pass 1 uses LPR 16 (group
// tiers included) and pass 2 stays at LPR 8 with its group tiers in the default layout.  fp32 rows of 512 bytes: 16 = the wide
// single-buffered layout (LPR 8), 8 = LPR 16, 4 = LPR 32.  Measured on config 5: destination-major 6.92 / 7.69 / 6.43 ms,
// source-major 6.20 / 8.06 / 7.90 ms.
constexpr int TG_BWD1_MAXW_BF16_256 = 4, TG_BWD2_MAXW_BF16_256 = 8;
constexpr int TG_BWD1_MAXW_F32_512 = 4, TG_BWD2_MAXW_F32_512 = 16;
constexpr bool TG_BWD1_GROUP_RELAYOUT = true, TG_BWD2_GROUP_RELAYOUT = false;

struct BwdArgs {
    const tg_block* b;
    const void *Q, *K, *V, *O, *dO;
    const float* lse;
    float scale;
    void *dQ, *dK, *dV;
    void* ws;
    size_t ws_bytes;
    int H;
    cudaStream_t stream;
    const float* O32;
};

template <class Tr>
struct BwdFn {
    // which: 1 = destination-major pass only, 2 = source-major pass only, 3 = both
    static tg_status_t run(const BwdArgs& a, int which) {
        using T = typename Tr::T;
        tg_geom g{Tr::NE, Tr::LPR, Tr::NHL};
        const tg_attn_ws_sizes sz = tg_attn_ws(a.b, a.H, g);
        tg_carver c(a.ws, a.ws_bytes);
        float2* ld = static_cast<float2*>(c.take(sz.ld));
        float* dq_part = static_cast<float*>(c.take(sz.dq_part));
        float* dkv_part = static_cast<float*>(c.take(sz.dkv_part));
        if (!c.ok()) TG_FAIL(TG_ERR_WORKSPACE, "fused bwd needs %zu workspace bytes", c.off);
        // Lane layouts (rowops.cuh): wide fp32 rows run at 16 words per lane, single-buffered; bf16 rows of 256 bytes run their WARP
        // tier (and the hub merges that read its partials) at 4 words per lane (LPR 16) where that was measured faster, their group
        // tiers in the default layout (LPR 8: four rows per warp instruction).  The layout is private to a launch.
        constexpr bool F512 = !Tr::BF16 && Tr::F * Tr::EB == 512;
        constexpr bool B256 = Tr::BF16 && Tr::F * Tr::EB == 256;
        if (which & 1) {
            constexpr bool WIDE = !Tr::BF16 && Tr::F * Tr::EB >= 512 && !(F512 && TG_BWD1_MAXW_F32_512 != 16);
            using TrW = typename std::conditional<WIDE, RowTraits<T, Tr::H, Tr::D, 16>, typename tg_relayout<Tr, B256 ? TG_BWD1_MAXW_BF16_256 : F512 ? TG_BWD1_MAXW_F32_512 : 8>::type>::type;
            using TrG = typename std::conditional<WIDE || TG_BWD1_GROUP_RELAYOUT, TrW, Tr>::type;
            static_assert(TrW::NE * TrW::LPR <= Tr::NE * Tr::LPR, "the partial workspace is sized with the default layout");
            auto launch = [&](auto tag) -> tg_status_t {
                constexpr bool ED = decltype(tag)::value;      // delta from the edges (bf16 without the fp32 copy of O)
                using Op = Bwd1Op<TrG, ED>;
                using OpW = Bwd1Op<TrW, ED>;      // the warp tier and the hub merges may use another lane layout
                typename Op::Params p;
                p.Q = static_cast<const T*>(a.Q); p.K = static_cast<const T*>(a.K); p.V = static_cast<const T*>(a.V);
                p.O = static_cast<const T*>(a.O); p.dO = static_cast<const T*>(a.dO);
                p.kv = a.b->kv_row; p.lse = a.lse;
                p.dQ = static_cast<T*>(a.dQ); p.ld = ld; p.part = dq_part;
                p.scale = a.scale; p.scale2 = a.scale * TG_LOG2E;
                p.O32 = a.O32;
                if constexpr (WIDE)
                    return tg_launch_tiers<Op, BwdPolicyWide, OpW>(p, a.b->dst, a.stream, "tg_attn_fused_bwd/dst");
                else if constexpr ((TrW::LPR == 16 && TrW::BF16) || (TrW::LPR == 32 && !TrW::BF16 && TrW::NW == 4))
                    return tg_launch_tiers<Op, BwdPolicyNarrow, OpW>(p, a.b->dst, a.stream, "tg_attn_fused_bwd/dst");
                else
                    return tg_launch_tiers<Op, BwdPolicy, OpW>(p, a.b->dst, a.stream, "tg_attn_fused_bwd/dst");
            };
            // bf16 storage: with the forward's fp32 copy of O delta = <dO, O> is taken up front (one accumulator and 16 registers
            // fewer per lane); without it delta is accumulated from the edges
            if (Tr::BF16 && !a.O32) TG_TRY(launch(std::true_type{}));
            else TG_TRY(launch(std::false_type{}));
        }
        if (which & 2) {
            constexpr bool WIDE = !Tr::BF16 && Tr::F * Tr::EB >= 512 && !(F512 && TG_BWD2_MAXW_F32_512 != 16);
            using TrW = typename std::conditional<WIDE, RowTraits<T, Tr::H, Tr::D, 16>, typename tg_relayout<Tr, B256 ? TG_BWD2_MAXW_BF16_256 : F512 ? TG_BWD2_MAXW_F32_512 : 8>::type>::type;
            using TrG = typename std::conditional<WIDE || TG_BWD2_GROUP_RELAYOUT, TrW, Tr>::type;
            static_assert(TrW::NE * TrW::LPR <= Tr::NE * Tr::LPR, "the partial workspace is sized with the default layout");
            using Op = Bwd2Op<TrG>;
            using OpW = Bwd2Op<TrW>;
            typename Op::Params p;
            p.Q = static_cast<const T*>(a.Q); p.K = static_cast<const T*>(a.K); p.V = static_cast<const T*>(a.V);
            p.dO = static_cast<const T*>(a.dO);
            p.t_dst = a.b->t_dst; p.ld = ld;
            p.dK = static_cast<T*>(a.dK); p.dV = static_cast<T*>(a.dV); p.part = dkv_part;
            p.scale = a.scale; p.scale2 = a.scale * TG_LOG2E;
            if constexpr (WIDE)
                TG_TRY((tg_launch_tiers<Op, BwdPolicyWide, OpW>(p, a.b->src, a.stream, "tg_attn_fused_bwd/src")));
            else if constexpr ((TrW::LPR == 16 && TrW::BF16) || (TrW::LPR == 32 && !TrW::BF16 && TrW::NW == 4))
                TG_TRY((tg_launch_tiers<Op, BwdPolicyNarrow, OpW>(p, a.b->src, a.stream, "tg_attn_fused_bwd/src")));
            else
                TG_TRY((tg_launch_tiers<Op, BwdPolicy, OpW>(p, a.b->src, a.stream, "tg_attn_fused_bwd/src")));
        }
        return TG_OK;
    }
};

static tg_status_t bwd_common(const tg_block_t* b, int H, int D, tg_dtype_t dtype, const void* Q, const void* K, const void* V,
                              const void* O, const float* o_f32, const float* lse, const void* dO, float scale, void* dQ, void* dK, void* dV,
                              void* ws, size_t ws_bytes, tg_stream_t stream, int which) {
    TG_CHECK_PTR(b);
    if (!tg_shape_supported(H, D, dtype)) TG_FAIL(TG_ERR_UNSUPPORTED, "unsupported (H=%d, D=%d, dtype=%d)", H, D, (int)dtype);
    if (b->R == 0) return TG_OK;
    TG_CHECK_ROWS(Q); TG_CHECK_ROWS(dO);
    if (which & 1) { TG_CHECK_ROWS(O); TG_CHECK_ROWS(dQ); TG_CHECK_PTR(lse); }
    if (b->E > 0) {
        TG_CHECK_ROWS(K); TG_CHECK_ROWS(V);
        if (which & 2) { TG_CHECK_ROWS(dK); TG_CHECK_ROWS(dV); }
    }
    if (!ws) TG_FAIL(TG_ERR_WORKSPACE, "fused bwd needs a workspace (tg_attn_workspace_bytes)");
    if (o_f32 && (reinterpret_cast<uintptr_t>(o_f32) & 15u)) TG_FAIL(TG_ERR_ALIGNMENT, "o_f32 is not 16-byte aligned");
    BwdArgs a{b, Q, K, V, O, dO, lse, scale, dQ, dK, dV, ws, ws_bytes, H, static_cast<cudaStream_t>(stream), o_f32};
    return tg_dispatch<BwdFn>(H, D, dtype, a, which);
}

extern "C" tg_status_t tg_attn_fused_bwd(const tg_block_t* b, int H, int D, tg_dtype_t dtype, const void* Q, const void* K,
                                         const void* V, const void* O, const float* o_f32, const float* lse, const void* dO, float scale,
                                         void* dQ, void* dK, void* dV, void* ws, size_t ws_bytes, tg_stream_t stream) {
    return bwd_common(b, H, D, dtype, Q, K, V, O, o_f32, lse, dO, scale, dQ, dK, dV, ws, ws_bytes, stream, 3);
}

extern "C" tg_status_t tg_attn_fused_bwd_dst(const tg_block_t* b, int H, int D, tg_dtype_t dtype, const void* Q, const void* K,
                                             const void* V, const void* O, const float* o_f32, const float* lse, const void* dO, float scale,
                                             void* dQ, void* ws, size_t ws_bytes, tg_stream_t stream) {
    return bwd_common(b, H, D, dtype, Q, K, V, O, o_f32, lse, dO, scale, dQ, nullptr, nullptr, ws, ws_bytes, stream, 1);
}

extern "C" tg_status_t tg_attn_fused_bwd_src(const tg_block_t* b, int H, int D, tg_dtype_t dtype, const void* Q, const void* K,
                                             const void* V, const void* dO, float scale, void* dK, void* dV, void* ws,
                                             size_t ws_bytes, tg_stream_t stream) {
    return bwd_common(b, H, D, dtype, Q, K, V, nullptr, nullptr, nullptr, dO, scale, nullptr, dK, dV, ws, ws_bytes, stream, 2);
}
