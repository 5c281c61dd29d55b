// rowops.cuh -- lane layout of one [H, D] row inside a sub-warp group, and the per-lane row
// arithmetic (vector loads, per-head dot products, axpy) for fp32 and bf16 storage.  sm_100a only.
//
// Layout.  A row of F = H*D elements is NV vectors of VB bytes (VB = 16, 8 or 4: the
// widest that divides one head's D*sizeof(T) bytes, so a vector never straddles two heads).  The row is
// owned by a GROUP of LPR lanes; lane i owns the vectors  i + LPR*k,  k = 0..NK-1  ("slot" k).  For a
// fixed k the LPR lanes of a group therefore read LPR*VB CONTIGUOUS bytes -- with 16-byte vectors and
// LPR = 8 one 128-byte line per group and instruction, which is what the L1 wavefront count wants
// (B300_MICROARCH.md "L1tex wavefront queue": one wavefront per 128-byte line touched).
// A warp holds G = 32/LPR groups, i.e. works on G gathered rows per instruction.
//
// Heads.  A lane's slots belong to different heads, so per-edge scalars (logit, probability, lse, delta)
// are small per-lane arrays over "head slots" j = 0..NHL-1:
//   MODE_A (VPH = vectors per head divides LPR, no tail): slot k of lane i lies in head i/VPH + (LPR/VPH)*k;
//           NHL = NK, head slot j = slot j, and the S = VPH neighbouring lanes share it.
//   general (VPH > LPR or ragged, e.g. D = 50): every lane tracks all heads, NHL = H, S = LPR; slot k lies
//           in head (i + LPR*k)/VPH, which is the same for all lanes of the group ("pure" slot) or one of
//           two neighbouring heads picked per lane ("mixed" slot, a bit in LanePos::mix).
// A dot product is reduced over the S lanes that share a head slot with xor-shuffles; every one of them
// ends with the total.
#pragma once
#include "common.cuh"

// MAXW_: 32-bit words of one gathered row a lane may hold.  8 everywhere (two gather buffers + state fit 128 registers),
// except the two backward passes on fp32 rows of >= 512 bytes, which run single-buffered at 16 (LPR 8 instead of 16:
// half the per-edge overhead instructions; config 5: bwd_src 8.2 -> 6.3 ms, bwd_dst 7.8 -> 7.0 ms; no gain in the forward).
template <typename T_, int H_, int D_, int MAXW_ = 8>
struct RowTraits {
    using T = T_;
    static constexpr int H = H_, D = D_, F = H_ * D_;
    static constexpr int EB = sizeof(T_);
    static constexpr bool BF16 = (EB == 2);
    static constexpr int VB = ((D_ * EB) % 16 == 0) ? 16 : (((D_ * EB) % 8 == 0) ? 8 : 4);
    static constexpr int VEC = VB / EB;         // elements per vector
    static constexpr int WV = VB / 4;           // 32-bit words per vector
    static constexpr int VPH = D_ / VEC;        // vectors per head
    static constexpr int NV = H_ * VPH;         // vectors per row
    static constexpr int pick_lpr() {
        int lpr = 8;
        while (lpr > NV) lpr /= 2;
        while (((NV + lpr - 1) / lpr) * WV > MAXW_ && lpr < 32) lpr *= 2;
        return lpr;
    }
    static constexpr int LPR = pick_lpr();      // lanes per row
    static constexpr int G = 32 / LPR;          // rows per warp instruction
    static constexpr int NK = (NV + LPR - 1) / LPR;
    static constexpr int NW = NK * WV;          // 32-bit words per lane
    static constexpr int NE = NK * VEC;         // elements per lane
    static constexpr bool TAIL = (NV % LPR) != 0;
    static constexpr bool MODE_A = (VPH <= LPR) && (LPR % VPH == 0) && !TAIL;
    static constexpr int NHL = MODE_A ? NK : H_;   // head slots per lane
    static constexpr int S = MODE_A ? VPH : LPR;   // lanes sharing a head slot
    // general mode: heads of the first / last lane's vector in slot k
    __host__ __device__ static constexpr int slot_lo(int k) { return (LPR * k) / VPH; }
    __host__ __device__ static constexpr int slot_hi(int k) {
        int last = LPR * k + LPR - 1;
        if (last > NV - 1) last = NV - 1;
        return last / VPH;
    }
    static_assert((D_ * EB) % 4 == 0, "row head slice must be a multiple of 4 bytes");
    static_assert(LPR <= 32 && (32 % LPR) == 0, "group must tile a warp");
    static_assert(NE <= 32 && NK <= 16, "too many elements per lane");
    static_assert((S & (S - 1)) == 0, "head-sharing lanes must be a power of two");
};

// Per-lane position inside its group.
template <class Tr>
struct LanePos {
    int lig;        // lane in group
    int off;        // element offset of this lane's vector in slot 0
    unsigned mix;   // general mode: bit k set = this lane's slot-k vector lies in head slot_hi(k)
    __device__ __forceinline__ explicit LanePos(int lig_) : lig(lig_), off(lig_ * Tr::VEC), mix(0u) {
        if constexpr (!Tr::MODE_A) {
#pragma unroll
            for (int k = 0; k < Tr::NK; ++k)
                if (Tr::slot_lo(k) != Tr::slot_hi(k) && (lig_ + Tr::LPR * k) >= Tr::slot_hi(k) * Tr::VPH) mix |= 1u << k;
        }
    }
    // head index of head slot j (for per-head scalars in global memory)
    __device__ __forceinline__ int head(int j) const {
        if constexpr (Tr::MODE_A) return lig / Tr::VPH + (Tr::LPR / Tr::VPH) * j;
        else return j;
    }
    // exactly one lane per (group, head) writes per-head scalars
    __device__ __forceinline__ bool head_writer() const { return (lig % Tr::S) == 0; }
    __device__ __forceinline__ bool slot_valid(int k) const { return !Tr::TAIL || (lig + Tr::LPR * k < Tr::NV); }
};

// raw 32-bit words of this lane's share of a row
template <class Tr>
struct RowReg {
    uint32_t w[Tr::NW];
};

// load this lane's vectors of a row; `p` = pointer to the row's element 0 PLUS lp.off (the operators keep
// lane-offset base pointers so that a gather address is one IMAD.WIDE)
template <class Tr>
__device__ __forceinline__ void row_load(RowReg<Tr>& r, const typename Tr::T* p, const LanePos<Tr>& lp) {
#pragma unroll
    for (int k = 0; k < Tr::NK; ++k) {
        const void* a = p + k * Tr::LPR * Tr::VEC;
        if (lp.slot_valid(k)) {
            if constexpr (Tr::WV == 4) {
                uint4 x = tg_ldg128(a);
                r.w[4 * k] = x.x; r.w[4 * k + 1] = x.y; r.w[4 * k + 2] = x.z; r.w[4 * k + 3] = x.w;
            } else if constexpr (Tr::WV == 2) {
                uint2 x = tg_ldg64(a);
                r.w[2 * k] = x.x; r.w[2 * k + 1] = x.y;
            } else {
                r.w[k] = (uint32_t)tg_ldg_i32(reinterpret_cast<const int32_t*>(a));
            }
        } else {
#pragma unroll
            for (int i = 0; i < Tr::WV; ++i) r.w[Tr::WV * k + i] = 0u;
        }
    }
}

// widen this lane's share of a row to fp32 (element order = ownership order)
template <class Tr>
__device__ __forceinline__ void row_to_float(const RowReg<Tr>& r, float (&x)[Tr::NE]) {
    if constexpr (Tr::BF16) {
#pragma unroll
        for (int i = 0; i < Tr::NW; ++i) { x[2 * i] = tg_bf16lo(r.w[i]); x[2 * i + 1] = tg_bf16hi(r.w[i]); }
    } else {
#pragma unroll
        for (int i = 0; i < Tr::NW; ++i) x[i] = __uint_as_float(r.w[i]);
    }
}

// head slot of element slot k for this lane (general mode; MODE_A: k itself)
template <class Tr, int k>
__device__ __forceinline__ float slot_pick(const float (&x)[Tr::NHL], const LanePos<Tr>& lp) {
    if constexpr (Tr::MODE_A) return x[k];
    else if constexpr (Tr::slot_lo(k) == Tr::slot_hi(k)) return x[Tr::slot_lo(k)];
    else return ((lp.mix >> k) & 1u) ? x[Tr::slot_hi(k)] : x[Tr::slot_lo(k)];
}

// lane-local dot product of the words of slot k.  bf16: products of two bf16 are exact in fp32; the
// mixed-precision FMA (PTX fma.rn.f32.bf16 -> SASS FHFMA.BF16) takes the packed halves directly.
// fp32: packed FFMA2 on element pairs.
template <class Tr, int k>
__device__ __forceinline__ float slot_dot(const RowReg<Tr>& a, const RowReg<Tr>& b) {
    if constexpr (Tr::BF16) {
        float acc0 = 0.f, acc1 = 0.f;   // two chains: the FHFMA result latency is not exposed back to back
#pragma unroll
        for (int i = Tr::WV * k; i < Tr::WV * (k + 1); ++i) {
            asm("{\n\t.reg .b16 al, ah, bl, bh;\n\t"
                "mov.b32 {al, ah}, %2;\n\tmov.b32 {bl, bh}, %3;\n\t"
                "fma.rn.f32.bf16 %0, al, bl, %0;\n\tfma.rn.f32.bf16 %1, ah, bh, %1;\n\t}"
                : "+f"(acc0), "+f"(acc1) : "r"(a.w[i]), "r"(b.w[i]));
        }
        return acc0 + acc1;
    } else {
        static_assert(Tr::BF16 || Tr::WV % 2 == 0, "fp32 vectors hold an even number of elements");
        float acc0 = 0.f, acc1 = 0.f;
#pragma unroll
        for (int i = Tr::WV * k; i < Tr::WV * (k + 1); i += 2)
            tg_ffma2(acc0, acc1, __uint_as_float(a.w[i]), __uint_as_float(a.w[i + 1]), __uint_as_float(b.w[i]), __uint_as_float(b.w[i + 1]));
        return acc0 + acc1;
    }
}

template <class Tr, int k>
__device__ __forceinline__ void dot_slots(const RowReg<Tr>& a, const RowReg<Tr>& b, const LanePos<Tr>& lp, float (&s)[Tr::NHL]) {
    if constexpr (k < Tr::NK) {
        const float part = slot_dot<Tr, k>(a, b);
        if constexpr (Tr::MODE_A) {
            s[k] = part;
        } else if constexpr (Tr::slot_lo(k) == Tr::slot_hi(k)) {
            s[Tr::slot_lo(k)] += part;
        } else {
            static_assert(Tr::slot_hi(k) == Tr::slot_lo(k) + 1 || Tr::MODE_A, "a slot spans at most two heads");
            const bool hi = (lp.mix >> k) & 1u;
            s[Tr::slot_lo(k)] += hi ? 0.f : part;
            s[Tr::slot_hi(k)] += hi ? part : 0.f;
        }
        dot_slots<Tr, k + 1>(a, b, lp, s);
    }
}

// s[j] = <a, b> restricted to head slot j, summed over the S lanes that share it (all of them get the total)
template <class Tr>
__device__ __forceinline__ void row_dot_heads(const RowReg<Tr>& a, const RowReg<Tr>& b, const LanePos<Tr>& lp, float (&s)[Tr::NHL]) {
    if constexpr (!Tr::MODE_A) {
#pragma unroll
        for (int j = 0; j < Tr::NHL; ++j) s[j] = 0.f;
    }
    dot_slots<Tr, 0>(a, b, lp, s);
#pragma unroll
    for (int o = 1; o < Tr::S; o <<= 1) {
#pragma unroll
        for (int j = 0; j < Tr::NHL; ++j) s[j] += __shfl_xor_sync(0xffffffffu, s[j], o);
    }
}

template <class Tr, int k>
__device__ __forceinline__ void axpy_slots(float* acc, const float (&p)[Tr::NHL], const RowReg<Tr>& r, const LanePos<Tr>& lp) {
    if constexpr (k < Tr::NK) {
        const float pk = slot_pick<Tr, k>(p, lp);
        if constexpr (Tr::BF16) {
#pragma unroll
            for (int i = Tr::WV * k; i < Tr::WV * (k + 1); ++i)
                tg_ffma2(acc[2 * i], acc[2 * i + 1], pk, pk, tg_bf16lo(r.w[i]), tg_bf16hi(r.w[i]));
        } else {
#pragma unroll
            for (int i = Tr::WV * k; i < Tr::WV * (k + 1); i += 2)
                tg_ffma2(acc[i], acc[i + 1], pk, pk, __uint_as_float(r.w[i]), __uint_as_float(r.w[i + 1]));
        }
        axpy_slots<Tr, k + 1>(acc, p, r, lp);
    }
}
// acc[e] += p[head slot of e] * row[e]
template <class Tr>
__device__ __forceinline__ void row_axpy_heads(float* acc, const float (&p)[Tr::NHL], const RowReg<Tr>& r, const LanePos<Tr>& lp) {
    axpy_slots<Tr, 0>(acc, p, r, lp);
}

template <class Tr, int k>
__device__ __forceinline__ void axpy2_slots(float* acc1, float* acc2, const float (&p1)[Tr::NHL], const float (&p2)[Tr::NHL],
                                            const RowReg<Tr>& r, const LanePos<Tr>& lp) {
    if constexpr (k < Tr::NK) {
        const float a = slot_pick<Tr, k>(p1, lp), b = slot_pick<Tr, k>(p2, lp);
        if constexpr (Tr::BF16) {
#pragma unroll
            for (int i = Tr::WV * k; i < Tr::WV * (k + 1); ++i) {
                const float lo = tg_bf16lo(r.w[i]), hi = tg_bf16hi(r.w[i]);
                tg_ffma2(acc1[2 * i], acc1[2 * i + 1], a, a, lo, hi);
                tg_ffma2(acc2[2 * i], acc2[2 * i + 1], b, b, lo, hi);
            }
        } else {
#pragma unroll
            for (int i = Tr::WV * k; i < Tr::WV * (k + 1); i += 2) {
                const float x = __uint_as_float(r.w[i]), y = __uint_as_float(r.w[i + 1]);
                tg_ffma2(acc1[i], acc1[i + 1], a, a, x, y);
                tg_ffma2(acc2[i], acc2[i + 1], b, b, x, y);
            }
        }
        axpy2_slots<Tr, k + 1>(acc1, acc2, p1, p2, r, lp);
    }
}
// acc1 += p1 * row; acc2 += p2 * row  (one widening of the row for both)
template <class Tr>
__device__ __forceinline__ void row_axpy2_heads(float* acc1, float* acc2, const float (&p1)[Tr::NHL], const float (&p2)[Tr::NHL],
                                                const RowReg<Tr>& r, const LanePos<Tr>& lp) {
    axpy2_slots<Tr, 0>(acc1, acc2, p1, p2, r, lp);
}

template <class Tr, int k>
__device__ __forceinline__ void scale_slots(float* acc, const float (&c)[Tr::NHL], const LanePos<Tr>& lp) {
    if constexpr (k < Tr::NK) {
        const float ck = slot_pick<Tr, k>(c, lp);
#pragma unroll
        for (int e = Tr::VEC * k; e < Tr::VEC * (k + 1); ++e) acc[e] *= ck;
        scale_slots<Tr, k + 1>(acc, c, lp);
    }
}
// acc[e] *= c[head slot of e]
template <class Tr>
__device__ __forceinline__ void row_scale_heads(float* acc, const float (&c)[Tr::NHL], const LanePos<Tr>& lp) {
    scale_slots<Tr, 0>(acc, c, lp);
}

template <class Tr, int k>
__device__ __forceinline__ void fnma_slots(float* a, const float (&d)[Tr::NHL], const float* b, const LanePos<Tr>& lp) {
    if constexpr (k < Tr::NK) {
        const float dk = slot_pick<Tr, k>(d, lp);
#pragma unroll
        for (int e = Tr::VEC * k; e < Tr::VEC * (k + 1); ++e) a[e] = fmaf(-dk, b[e], a[e]);
        fnma_slots<Tr, k + 1>(a, d, b, lp);
    }
}
// a[e] -= d[head slot of e] * b[e]
template <class Tr>
__device__ __forceinline__ void row_fnma_heads(float* a, const float (&d)[Tr::NHL], const float* b, const LanePos<Tr>& lp) {
    fnma_slots<Tr, 0>(a, d, b, lp);
}

// store fp32 lane values (scaled by `mul`) as storage dtype into the row starting at `row`
template <class Tr>
__device__ __forceinline__ void row_store(typename Tr::T* row, const LanePos<Tr>& lp, const float* x, float mul) {
    typename Tr::T* p = row + lp.off;
#pragma unroll
    for (int k = 0; k < Tr::NK; ++k) {
        if (!lp.slot_valid(k)) continue;
        void* a = p + k * Tr::LPR * Tr::VEC;
        uint32_t w[Tr::WV];
        if constexpr (Tr::BF16) {
#pragma unroll
            for (int i = 0; i < Tr::WV; ++i)
                w[i] = tg_pack_bf16(x[k * Tr::VEC + 2 * i] * mul, x[k * Tr::VEC + 2 * i + 1] * mul);
        } else {
#pragma unroll
            for (int i = 0; i < Tr::WV; ++i) w[i] = __float_as_uint(x[k * Tr::VEC + i] * mul);
        }
        if constexpr (Tr::WV == 4) *reinterpret_cast<uint4*>(a) = make_uint4(w[0], w[1], w[2], w[3]);
        else if constexpr (Tr::WV == 2) *reinterpret_cast<uint2*>(a) = make_uint2(w[0], w[1]);
        else *reinterpret_cast<uint32_t*>(a) = w[0];
    }
}

// fp32 view of a row in the lane layout (a side copy kept in float whatever the storage dtype): lane's slot k covers the
// VEC consecutive floats of vector lig + LPR*k.
template <class Tr>
__device__ __forceinline__ void row_store_f32(float* row, const LanePos<Tr>& lp, const float* x) {
#pragma unroll
    for (int k = 0; k < Tr::NK; ++k) {
        if (!lp.slot_valid(k)) continue;
        float* a = row + (lp.lig + Tr::LPR * k) * Tr::VEC;
#pragma unroll
        for (int e = 0; e < Tr::VEC; ++e) a[e] = x[k * Tr::VEC + e];
    }
}
template <class Tr>
__device__ __forceinline__ void row_load_f32(float (&x)[Tr::NE], const float* row, const LanePos<Tr>& lp) {
#pragma unroll
    for (int k = 0; k < Tr::NK; ++k) {
        const float* a = row + (lp.lig + Tr::LPR * k) * Tr::VEC;
#pragma unroll
        for (int e = 0; e < Tr::VEC; ++e) x[k * Tr::VEC + e] = lp.slot_valid(k) ? a[e] : 0.f;
    }
}
// s[j] = <a, b> restricted to head slot j for two rows already widened to float (same reduction as row_dot_heads)
template <class Tr, int k>
__device__ __forceinline__ void dotf_slots(const float* a, const float* b, const LanePos<Tr>& lp, float (&s)[Tr::NHL]) {
    if constexpr (k < Tr::NK) {
        float part = 0.f;
#pragma unroll
        for (int e = Tr::VEC * k; e < Tr::VEC * (k + 1); ++e) part = fmaf(a[e], b[e], part);
        if constexpr (Tr::MODE_A) {
            s[k] = part;
        } else if constexpr (Tr::slot_lo(k) == Tr::slot_hi(k)) {
            s[Tr::slot_lo(k)] += part;
        } else {
            const bool hi = (lp.mix >> k) & 1u;
            s[Tr::slot_lo(k)] += hi ? 0.f : part;
            s[Tr::slot_hi(k)] += hi ? part : 0.f;
        }
        dotf_slots<Tr, k + 1>(a, b, lp, s);
    }
}
template <class Tr>
__device__ __forceinline__ void row_dotf_heads(const float* a, const float* b, const LanePos<Tr>& lp, float (&s)[Tr::NHL]) {
    if constexpr (!Tr::MODE_A) {
#pragma unroll
        for (int j = 0; j < Tr::NHL; ++j) s[j] = 0.f;
    }
    dotf_slots<Tr, 0>(a, b, lp, s);
#pragma unroll
    for (int o = 1; o < Tr::S; o <<= 1) {
#pragma unroll
        for (int j = 0; j < Tr::NHL; ++j) s[j] += __shfl_xor_sync(0xffffffffu, s[j], o);
    }
}
