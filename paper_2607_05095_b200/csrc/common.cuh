// common.cuh -- internal declarations shared by the libfasttg translation units (sm_100a only).
// Nothing here is shared with oracle/ (the CPU oracle is an independent program).
#pragma once

#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <stdio.h>

#include "fasttg.h"

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "libfasttg is written for sm_100a (B200) only"
#endif

// ---------------------------------------------------------------------------------------------
// Errors
// ---------------------------------------------------------------------------------------------
void tg_set_error(const char* fmt, ...);

#define TG_FAIL(code, ...)            \
    do {                              \
        tg_set_error(__VA_ARGS__);    \
        return (code);                \
    } while (0)

#define TG_CUDA(expr)                                                                              \
    do {                                                                                           \
        cudaError_t _e = (expr);                                                                   \
        if (_e != cudaSuccess) {                                                                   \
            tg_set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
            return TG_ERR_CUDA;                                                                    \
        }                                                                                          \
    } while (0)

#define TG_TRY(expr)                      \
    do {                                  \
        tg_status_t _s = (expr);          \
        if (_s != TG_OK) return _s;       \
    } while (0)

// process-wide count of kernels launched by the library (tg_launch_count)
void tg_count_launch();

#define TG_LAUNCH_CHECK(name)                                                                     \
    do {                                                                                          \
        tg_count_launch();                                                                        \
        cudaError_t _e = cudaGetLastError();                                                      \
        if (_e != cudaSuccess) {                                                                  \
            tg_set_error("launch of %s failed: %s", name, cudaGetErrorString(_e));                \
            return TG_ERR_CUDA;                                                                   \
        }                                                                                         \
    } while (0)

// ---------------------------------------------------------------------------------------------
// Schedules.  A "side" is a CSR (rows, indptr): the destination side (rows = destinations, edges
// in CSR order) or the source side (rows = unique source rows, edges in transposed order).
// Rows are split into two tiers by degree:
//   group tier: deg <= TG_GROUP_MAX    one sub-warp group per row (the K <= 10-20 common case); rows are
//                                      bucketed into TG_NCLS power-of-two degree classes so that the
//                                      groups of a warp run the same number of trips
//   warp tier : larger                 one warp per chunk of <= `chunk` edges (TG_CHUNK_MIN..TG_CHUNK_MAX, picked per
//                                      side so that a small block still spreads over the SMs: a lone warp walks
//                                      its chunk as one latency chain); a row with more than one
//                                      chunk ("hub") writes fp32 partials, merged by a second launch
// Every schedule record carries {row, begin, end}: one load instead of the order -> indptr chain.
// ---------------------------------------------------------------------------------------------
#ifndef TG_NCLS_N
#define TG_NCLS_N 6
#endif
#ifndef TG_NCLS_SMALL_N
#define TG_NCLS_SMALL_N 3
#endif
constexpr int TG_NCLS = TG_NCLS_N;              // degree classes <=2, 3-4, 5-8, 9-16, 17-32, 33-64 (, 65-128)
constexpr int TG_NCLS_SMALL = TG_NCLS_SMALL_N;  // classes 0..2 (deg <= 8) run in the high-occupancy kernel variant
constexpr int TG_GROUP_MAX = 2 << (TG_NCLS - 1);
#ifndef TG_GROUP_MAX_SMALL_N
#define TG_GROUP_MAX_SMALL_N 32
#endif
constexpr int TG_GROUP_MAX_SMALL = TG_GROUP_MAX_SMALL_N;   // group-tier limit of a launch-bound side (< TG_FORK_MIN_EDGES edges)
#ifndef TG_CHUNK_MAX_EDGES
#define TG_CHUNK_MAX_EDGES 1024
#endif
constexpr int TG_CHUNK_MIN = 64, TG_CHUNK_MAX = TG_CHUNK_MAX_EDGES;
constexpr int TG_CTA_THREADS = 256;
constexpr int TG_HUB_DIRECT = 32;   // a hub with more chunks is merged in two levels
constexpr int TG_HUB_SPLIT = 16;    // CTAs per big hub in the first level
constexpr int TG_CTA_WARPS = TG_CTA_THREADS / 32;

__host__ __device__ constexpr int tg_degree_class(int deg) {
    return deg <= 2 ? 0 : deg <= 4 ? 1 : deg <= 8 ? 2 : deg <= 16 ? 3 : deg <= 32 ? 4 : deg <= 64 ? 5 : deg <= 128 ? 6 : 7;
}

struct tg_side {
    int64_t n_rows = 0, n_edges = 0;
    const int32_t* indptr = nullptr;
    int4* rows = nullptr;      // group tier {row, begin, end, 0}: class TG_NCLS-1 first ... class 0 last
    int4* items = nullptr;     // warp tier {row, begin, end, slot}; slot < 0: the row's only chunk
    int4* hubs = nullptr;      // {row, first_slot, n_chunks, 0}
    int4* bighubs = nullptr;   // the hubs with more than TG_HUB_DIRECT chunks again (two-level merge)
    int32_t n_cls[TG_NCLS] = {};
    int32_t n_group = 0, n_items = 0, n_hubs = 0, n_bighubs = 0, n_slots = 0;
    int32_t max_deg = 0;
    int32_t chunk = TG_CHUNK_MAX;   // edges per warp item of this side
    int32_t group_max = TG_GROUP_MAX;   // rows up to this degree are group-tier rows
    // group-tier rows of the classes >= TG_NCLS_SMALL come first in `rows`
    int32_t n_group_big() const { int n = 0; for (int c = TG_NCLS_SMALL; c < TG_NCLS; ++c) n += n_cls[c]; return n; }
    int32_t n_group_small() const { return n_group - n_group_big(); }
};

// Largest R / E: positions are int32 and the edge loops look a few trips (<= 4 * 32 positions) past a row's end before clamping.
constexpr int64_t TG_MAX_INDEX = (1LL << 31) - 4096;

struct tg_block {
    int64_t R = 0, E = 0, U = 0;
    const int32_t* indptr = nullptr;
    const int32_t* kv_row = nullptr;
    const int32_t* t_indptr = nullptr;
    const int32_t* t_edge = nullptr;
    const int32_t* t_dst = nullptr;
    tg_side dst, src;
};

size_t tg_side_bytes(int64_t n_rows_bound, int64_t n_edges);
// Builds one side's schedule in `ws` (must hold tg_side_bytes).  Synchronises the stream.
tg_status_t tg_side_build(tg_side* s, int64_t n_rows, int64_t n_edges, const int32_t* indptr, void* ws,
                          size_t ws_bytes, cudaStream_t stream);

// Auxiliary streams of the calling thread (created on first use, never destroyed) for the fork / join in tiers.cuh.
struct tg_aux_streams {
    cudaStream_t s[2];
    cudaEvent_t fork, join[2];
};
tg_aux_streams* tg_get_aux_streams();   // nullptr + tg_last_error() on failure
constexpr int64_t TG_FORK_MIN_EDGES = 1 << 20;

static inline size_t tg_align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// ---------------------------------------------------------------------------------------------
// Device helpers
// ---------------------------------------------------------------------------------------------
#ifdef __CUDACC__

constexpr float TG_LOG2E = 1.4426950408889634f;
constexpr float TG_LN2 = 0.6931471805599453f;

__device__ __forceinline__ float tg_exp2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// 16-byte read-only load (LDG.E.128.CONSTANT)
__device__ __forceinline__ uint4 tg_ldg128(const void* p) {
    uint4 r;
    asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ uint2 tg_ldg64(const void* p) {
    uint2 r;
    asm volatile("ld.global.nc.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "l"(p));
    return r;
}
__device__ __forceinline__ int tg_ldg_i32(const int32_t* p) {
    int r;
    asm volatile("ld.global.nc.s32 %0, [%1];" : "=r"(r) : "l"(p));
    return r;
}
// load whose value is never used: brings the sector into L1 ahead of time (a CCTL prefetch serialises here)
__device__ __forceinline__ void tg_touch_i32(const int32_t* p) {
    int r;
    asm volatile("ld.global.nc.s32 %0, [%1];" : "=r"(r) : "l"(p));
}
__device__ __forceinline__ float tg_ldg_f32(const float* p) {
    float r;
    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(r) : "l"(p));
    return r;
}

__device__ __forceinline__ float tg_bf16lo(uint32_t x) { return __uint_as_float(x << 16); }
__device__ __forceinline__ float tg_bf16hi(uint32_t x) { return __uint_as_float(x & 0xffff0000u); }
// packed fp32 FMA (SASS FFMA2): (d0, d1) += (a0, a1) * (b0, b1); one issue slot for two FMAs.
__device__ __forceinline__ void tg_ffma2(float& d0, float& d1, float a0, float a1, float b0, float b1) {
    uint64_t a, b, c;
    asm("mov.b64 %0, {%1, %2};" : "=l"(a) : "f"(a0), "f"(a1));
    asm("mov.b64 %0, {%1, %2};" : "=l"(b) : "f"(b0), "f"(b1));
    asm("mov.b64 %0, {%1, %2};" : "=l"(c) : "f"(d0), "f"(d1));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(c) : "l"(a), "l"(b));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d0), "=f"(d1) : "l"(c));
}
// round-to-nearest-even pack of two floats into bf16x2 (lo = a, hi = b)
__device__ __forceinline__ uint32_t tg_pack_bf16(float a, float b) {
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(b), "f"(a));
    return r;
}

#endif  // __CUDACC__
