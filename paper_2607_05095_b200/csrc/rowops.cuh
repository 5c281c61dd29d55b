// rowops.cuh -- lane layout of one [H, D] row inside a sub-warp group, and the per-lane row
// arithmetic (vector loads, dot products, axpy) for fp32 and bf16 storage.  sm_100a only.
//
// Layout.  A row of F = H*D elements is owned by a GROUP of LPR = H*LPH lanes;
// LPH lanes share a head.  Lane (h, j) holds the vectors vi = j + LPH*k, k = 0..NK-1, of head h,
// each VEC elements (VB = 16, 8 or 4 bytes; the widest that divides D*sizeof(T)), so that for a
// fixed k the LPH lanes of a head read LPH*VB contiguous bytes.  A warp holds G = 32/LPR groups.
// D = 50 fp32 (VB = 8, NV = 25 vectors, LPH = 8) leaves a tail: only j = 0 owns a 4th vector.
#pragma once
#include "common.cuh"

template <typename T_, int H_, int D_>
struct RowTraits {
    using T = T_;
    static constexpr int H = H_, D = D_, F = H_ * D_;
    static constexpr int EB = sizeof(T_);
    static constexpr bool BF16 = (EB == 2);
    static constexpr int VB = ((D_ * EB) % 16 == 0) ? 16 : (((D_ * EB) % 8 == 0) ? 8 : 4);
    static constexpr int VEC = VB / EB;
    static constexpr int NV = D_ / VEC;
    static constexpr int pick_lph() {
        int lph = (8 / H_) > 1 ? (8 / H_) : 1;
        while ((NV + lph - 1) / lph > 4 && H_ * lph * 2 <= 32) lph *= 2;
        while (lph > NV && lph > 1) lph /= 2;
        return lph;
    }
    static constexpr int LPH = pick_lph();
    static constexpr int LPR = H_ * LPH;
    static constexpr int G = 32 / LPR;
    static constexpr int NK = (NV + LPH - 1) / LPH;
    static constexpr int NE = NK * VEC;        // elements per lane
    static constexpr int WV = VB / 4;          // 32-bit words per vector
    static constexpr int NW = NK * WV;         // 32-bit words per lane
    static constexpr bool TAIL = (NV % LPH) != 0;
    static_assert((D_ * EB) % 4 == 0, "row head slice must be a multiple of 4 bytes");
    static_assert(D_ % VEC == 0, "vector width must divide D");
    static_assert(LPR <= 32 && (32 % LPR) == 0, "group must tile a warp");
    static_assert(NE <= 32, "too many elements per lane");
};

// Per-lane position inside its group.
template <class Tr>
struct LanePos {
    int lig, h, j, off;  // lane in group, head, lane in head, element offset of vector k = 0
    __device__ __forceinline__ explicit LanePos(int lig_) : lig(lig_) {
        h = lig_ / Tr::LPH;
        j = lig_ % Tr::LPH;
        off = h * Tr::D + j * Tr::VEC;
    }
};

// raw 32-bit words of this lane's share of a row
template <class Tr>
struct RowReg {
    uint32_t w[Tr::NW];
};

template <class Tr>
__device__ __forceinline__ void row_zero(RowReg<Tr>& r) {
#pragma unroll
    for (int i = 0; i < Tr::NW; ++i) r.w[i] = 0u;
}

// load this lane's vectors of the row that starts at `row` (pointer to element 0 of the row)
template <class Tr>
__device__ __forceinline__ void row_load(RowReg<Tr>& r, const typename Tr::T* row, const LanePos<Tr>& lp) {
    const typename Tr::T* p = row + lp.off;
#pragma unroll
    for (int k = 0; k < Tr::NK; ++k) {
        const bool in = !Tr::TAIL || (lp.j + Tr::LPH * k < Tr::NV);
        const void* a = p + k * Tr::LPH * Tr::VEC;
        if (in) {
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

// widen to fp32 (element order = ownership order)
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

// store fp32 lane values (scaled) as storage dtype into the row starting at `row`
template <class Tr>
__device__ __forceinline__ void row_store(typename Tr::T* row, const LanePos<Tr>& lp, const float* x, float mul) {
    typename Tr::T* p = row + lp.off;
#pragma unroll
    for (int k = 0; k < Tr::NK; ++k) {
        const bool in = !Tr::TAIL || (lp.j + Tr::LPH * k < Tr::NV);
        if (!in) continue;
        void* a = p + k * Tr::LPH * Tr::VEC;
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

// lane-local partial dot product of two rows.  bf16: products of two bf16 are exact in fp32; the
// mixed-precision FMA (PTX fma.rn.f32.bf16 -> SASS FHFMA.BF16) takes the packed halves directly, so
// no widening instructions are spent.  Two accumulators shorten the dependency chain.
template <class Tr>
__device__ __forceinline__ float row_dot(const RowReg<Tr>& a, const RowReg<Tr>& b) {
    float acc0 = 0.f, acc1 = 0.f;
    if constexpr (Tr::BF16) {
#pragma unroll
        for (int i = 0; i < Tr::NW; ++i) {
            asm("{\n\t.reg .b16 al, ah, bl, bh;\n\t"
                "mov.b32 {al, ah}, %2;\n\tmov.b32 {bl, bh}, %3;\n\t"
                "fma.rn.f32.bf16 %0, al, bl, %0;\n\tfma.rn.f32.bf16 %1, ah, bh, %1;\n\t}"
                : "+f"(acc0), "+f"(acc1) : "r"(a.w[i]), "r"(b.w[i]));
        }
    } else {
#pragma unroll
        for (int i = 0; i < Tr::NW; i += 2) {
            acc0 = fmaf(__uint_as_float(a.w[i]), __uint_as_float(b.w[i]), acc0);
            if (i + 1 < Tr::NW) acc1 = fmaf(__uint_as_float(a.w[i + 1]), __uint_as_float(b.w[i + 1]), acc1);
        }
    }
    return acc0 + acc1;
}

// sum over the LPH lanes that share a head (xor butterfly; every lane ends with the total)
template <class Tr>
__device__ __forceinline__ float head_sum(float x) {
#pragma unroll
    for (int o = 1; o < Tr::LPH; o <<= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// acc += p * row
template <class Tr>
__device__ __forceinline__ void row_axpy(float* acc, float p, const RowReg<Tr>& r) {
    if constexpr (Tr::BF16) {
#pragma unroll
        for (int i = 0; i < Tr::NW; ++i) {
            acc[2 * i] = fmaf(p, tg_bf16lo(r.w[i]), acc[2 * i]);
            acc[2 * i + 1] = fmaf(p, tg_bf16hi(r.w[i]), acc[2 * i + 1]);
        }
    } else {
#pragma unroll
        for (int i = 0; i < Tr::NW; ++i) acc[i] = fmaf(p, __uint_as_float(r.w[i]), acc[i]);
    }
}

// acc1 += p1 * row; acc2 += p2 * row  (one widening of the row for both)
template <class Tr>
__device__ __forceinline__ void row_axpy2(float* acc1, float* acc2, float p1, float p2, const RowReg<Tr>& r) {
    if constexpr (Tr::BF16) {
#pragma unroll
        for (int i = 0; i < Tr::NW; ++i) {
            const float lo = tg_bf16lo(r.w[i]), hi = tg_bf16hi(r.w[i]);
            acc1[2 * i] = fmaf(p1, lo, acc1[2 * i]);
            acc1[2 * i + 1] = fmaf(p1, hi, acc1[2 * i + 1]);
            acc2[2 * i] = fmaf(p2, lo, acc2[2 * i]);
            acc2[2 * i + 1] = fmaf(p2, hi, acc2[2 * i + 1]);
        }
    } else {
#pragma unroll
        for (int i = 0; i < Tr::NW; ++i) {
            const float x = __uint_as_float(r.w[i]);
            acc1[i] = fmaf(p1, x, acc1[i]);
            acc2[i] = fmaf(p2, x, acc2[i]);
        }
    }
}
