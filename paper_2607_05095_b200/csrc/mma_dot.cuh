// mma_dot.cuh -- per-head dot products of gathered bf16 rows on the tensor cores (mma.sync.m16n8k16, SASS HMMA), for
// the WARP tier (all four groups of the warp work on the same fixed row).
//
// The row-gather kernels spend 30-40 % of their issue slots on the per-head dot products <Q[v,h], K[r(e),h]> (one FHFMA
// per bf16 pair and lane, plus the shuffle reduction).  One query row per (destination, head) makes this a matrix-VECTOR
// product, so a tensor-core tile is mostly padding -- but the tile is free and the issue slots are not.
//
//   B (16 x 8, col)  = the gathered rows, straight from the registers the LDG.128 filled (rowops.cuh layout, LPR = 8):
//                      column n = quad n of the warp = the 64-byte half `par = n & 1` of the row of group `n >> 1`;
//                      the pair (w0, w1) resp. (w2, w3) of a lane's 16-byte vector is the (b0, b1) of one HMMA, so the
//                      contraction index k is a private permutation of the row's elements, fixed by the loads.
//   A (16 x 16, row) = the fixed row (Q in the destination-major passes, K / V of the source row in the source-major
//                      pass), block-diagonal: A[m][k] = fixed[element of k] if that element lies in head m, else 0
//                      (rows 8..15 are zero).  "element of k" depends on the parity of the column; the two candidates
//                      lie in different heads, i.e. different rows m, so both can be stored.
//   C (16 x 8)       = C[m][n] = <fixed row, gathered half-row n> restricted to head m.  Head m lies entirely in the
//                      half-rows of one parity: lane (m, t) finds the logit of (head m, edge of group t) in c0 or c1.
// NK * 2 HMMA per edge set (one edge per group) replace NK * 8 FHFMA + 3 * NHL reduction instructions, and every lane
// ends up with ONE per-head scalar (head = lane >> 2, group = lane & 3): the softmax scalar work halves as well.  The
// probabilities reach the lanes that own the matching V vectors ("slot layout" of rowops.cuh) by one shuffle per slot.
//
// Supported layouts: bf16, 16-byte vectors, LPR = 8, NK = 2 (256-byte rows), D in {16, 32}: (H, D) = (8, 16), (4, 32).
#pragma once
#include "rowops.cuh"

template <class Tr>
struct MmaDotOk {
    static constexpr bool value = Tr::BF16 && Tr::VB == 16 && Tr::LPR == 8 && Tr::NK == 2 && Tr::MODE_A && (Tr::VPH == 2 || Tr::VPH == 4) && Tr::H <= 8;
};

__device__ __forceinline__ void tg_hmma16816(float (&c)[4], const uint4& a, uint32_t b0, uint32_t b1) {
    asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a.x), "r"(a.y), "r"(a.z), "r"(a.w), "r"(b0), "r"(b1));
}

// Geometry of one lane.  Gather side: lane = 8*grp + i (i = lane in group).  Scalar side ("head layout"): the lane owns
// the per-head scalars of head hd = lane >> 2 for the edge of group gt = lane & 3.
template <class Tr>
struct MmaLane {
    int hd, gt, grp;
    bool odd;             // the logit of head hd comes out in c1 (columns of parity 1) instead of c0
    bool live;            // hd < H
    int src[Tr::NK];      // lane that owns the scalars of (head of this lane's slot-k vector, this lane's group)
    __device__ __forceinline__ explicit MmaLane(int lane) {
        const int i = lane & 7;
        hd = lane >> 2; gt = lane & 3; grp = lane >> 3;
        odd = (((hd * Tr::VPH) & 7) >> 2) != 0;      // the head's vectors hd*VPH .. sit at lanes (hd*VPH) % 8 .. of a group
        live = hd < Tr::H;
#pragma unroll
        for (int k = 0; k < Tr::NK; ++k) src[k] = 4 * ((i + Tr::LPR * k) / Tr::VPH) + grp;
    }
    // head layout -> slot layout: the scalar of (head of slot k, own group)
    __device__ __forceinline__ float to_slot(float x, int k) const { return __shfl_sync(0xffffffffu, x, src[k]); }
};

// Block-diagonal A fragments of a fixed row (`row` = pointer to its element 0): [slot][half of the 16-byte vector].
template <class Tr>
struct MmaFixed {
    uint4 a[Tr::NK][2];
    __device__ __forceinline__ void load(const typename Tr::T* row, int lane) {
        const int m = lane >> 2, t = lane & 3;    // A row (head) and k-pair of this lane
#pragma unroll
        for (int k = 0; k < Tr::NK; ++k) {
            uint4 x = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
            for (int pp = 0; pp < 2; ++pp) {
                const int vi = 4 * pp + t + Tr::LPR * k;          // the vector a column of parity pp feeds into k-pair t
                if (vi / Tr::VPH == m && m < Tr::H) x = tg_ldg128(row + vi * Tr::VEC);
            }
            a[k][0] = make_uint4(x.x, 0u, x.y, 0u);
            a[k][1] = make_uint4(x.z, 0u, x.w, 0u);
        }
    }
    // logit of (head lane >> 2, edge of group lane & 3): c0 (parity-0 columns) or c1
    __device__ __forceinline__ float dot(const RowReg<Tr>& r, bool odd) const {
        // one accumulator chain per slot: a dependent HMMA costs ~23 cycles (measured), two chains of two halve the wait
        float c[Tr::NK][4];
#pragma unroll
        for (int k = 0; k < Tr::NK; ++k) {
            c[k][0] = c[k][1] = c[k][2] = c[k][3] = 0.f;
            tg_hmma16816(c[k], a[k][0], r.w[4 * k], r.w[4 * k + 1]);
            tg_hmma16816(c[k], a[k][1], r.w[4 * k + 2], r.w[4 * k + 3]);
        }
        float v = odd ? c[0][1] : c[0][0];
#pragma unroll
        for (int k = 1; k < Tr::NK; ++k) v += odd ? c[k][1] : c[k][0];
        return v;
    }
};
