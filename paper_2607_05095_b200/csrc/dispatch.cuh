// dispatch.cuh -- the compiled (H, D, dtype) set and argument checks shared by the operator entry points.
#pragma once
#include "ops.cuh"

// The supported (H, D) pairs; each is compiled for fp32 and bf16 storage.
#define TG_SHAPES(X) X(2, 50) X(4, 32) X(8, 16) X(2, 64) X(1, 128) X(2, 32) X(4, 16) X(2, 128)

// tg_dispatch<Fn>(H, D, dtype, args...) calls Fn<RowTraits<T,H,D>>::run(args...) for the matching compiled shape.
template <template <class> class Fn, class... Args>
static tg_status_t tg_dispatch(int H, int D, tg_dtype_t dtype, Args&&... args) {
#define X(h, d)                                                                              \
    if (H == h && D == d) {                                                                  \
        if (dtype == TG_F32) return Fn<RowTraits<float, h, d>>::run(args...);                \
        if (dtype == TG_BF16) return Fn<RowTraits<__nv_bfloat16, h, d>>::run(args...);       \
    }
    TG_SHAPES(X)
#undef X
    TG_FAIL(TG_ERR_UNSUPPORTED, "unsupported (H=%d, D=%d, dtype=%d); see tg_supported()", H, D, (int)dtype);
}

static inline bool tg_shape_supported(int H, int D, tg_dtype_t dtype) {
    if (dtype != TG_F32 && dtype != TG_BF16) return false;
#define X(h, d) if (H == h && D == d) return true;
    TG_SHAPES(X)
#undef X
    return false;
}

// Layout override for one kernel: RowTraits with MAXW words per lane if that keeps every partial-state size of the default
// layout (the workspaces are sized with the default layout), else the default layout.
template <class Tr0, int MAXW>
struct tg_relayout {
    using Alt = RowTraits<typename Tr0::T, Tr0::H, Tr0::D, MAXW>;
    static constexpr bool same = Alt::NE * Alt::LPR == Tr0::NE * Tr0::LPR && Alt::NHL * Alt::LPR == Tr0::NHL * Tr0::LPR;
    using type = typename std::conditional<same, Alt, Tr0>::type;
};

// per-lane geometry for workspace sizing
struct tg_geom { int NE, LPR, NHL; };
template <class Tr> struct GeomFn {
    static tg_status_t run(tg_geom* g) { g->NE = Tr::NE; g->LPR = Tr::LPR; g->NHL = Tr::NHL; return TG_OK; }
};
static inline tg_status_t tg_get_geom(int H, int D, tg_dtype_t dtype, tg_geom* g) {
    return tg_dispatch<GeomFn>(H, D, dtype, g);
}

static inline tg_status_t tg_check_rows(const void* p, const char* name) {
    if (!p) TG_FAIL(TG_ERR_INVALID_ARG, "%s is null", name);
    if ((reinterpret_cast<uintptr_t>(p) & 15u) != 0) TG_FAIL(TG_ERR_ALIGNMENT, "%s is not 16-byte aligned", name);
    return TG_OK;
}
#define TG_CHECK_ROWS(p)                              \
    do {                                              \
        tg_status_t _s = tg_check_rows((p), #p);      \
        if (_s != TG_OK) return _s;                   \
    } while (0)
#define TG_CHECK_PTR(p)                                                  \
    do {                                                                 \
        if (!(p)) TG_FAIL(TG_ERR_INVALID_ARG, "%s is null", #p);         \
    } while (0)

// workspace carving
struct tg_carver {
    char* base;
    size_t off = 0, cap;
    tg_carver(void* b, size_t c) : base(static_cast<char*>(b)), cap(c) {}
    void* take(size_t bytes) {
        void* p = base ? base + off : nullptr;
        off += tg_align_up(bytes);
        return p;
    }
    bool ok() const { return off <= cap && (base != nullptr || off == 0); }
};

// partial slots of one side: one per hub chunk plus the second-level slots of the split hub merge (tiers.cuh)
static inline size_t tg_part_slots(const tg_side& s) { return (size_t)s.n_slots + (size_t)s.n_bighubs * TG_HUB_SPLIT; }

struct tg_attn_ws_sizes { size_t fwd_part, ld, dq_part, dkv_part; };
static inline tg_attn_ws_sizes tg_attn_ws(const tg_block* b, int H, const tg_geom& g) {
    tg_attn_ws_sizes s;
    s.fwd_part = tg_part_slots(b->dst) * (g.NE + 2 * g.NHL) * g.LPR * sizeof(float);
    s.ld = (size_t)b->R * H * sizeof(float2);
    s.dq_part = tg_part_slots(b->dst) * (2 * g.NE + g.NHL) * g.LPR * sizeof(float);  // bf16: {A1, A2, d}; fp32 uses NE of it
    s.dkv_part = tg_part_slots(b->src) * 2 * g.NE * g.LPR * sizeof(float);
    return s;
}
