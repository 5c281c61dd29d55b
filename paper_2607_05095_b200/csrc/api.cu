// api.cu -- status strings, thread-local error text, version and capability queries.
#include <stdarg.h>

#include <atomic>

#include "dispatch.cuh"
#include "fasttg_diag.h"

static thread_local char g_err[512] = "";

void tg_set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

extern "C" const char* tg_last_error(void) { return g_err; }

static std::atomic<unsigned long long> g_launches{0};
void tg_count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }
extern "C" unsigned long long tg_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

// One set of auxiliary streams per (thread, device), created on first use and kept for the life of the thread.
tg_aux_streams* tg_get_aux_streams() {
    constexpr int MAX_DEV = 64;
    struct Slot { tg_aux_streams aux; bool ready = false; };
    static thread_local Slot table[MAX_DEV];
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur < 0 || cur >= MAX_DEV) { tg_set_error("cudaGetDevice failed or device index %d >= %d", cur, MAX_DEV); return nullptr; }
    Slot& sl = table[cur];
    if (!sl.ready) {
        bool ok = true;
        for (int i = 0; i < 2; ++i) {
            ok = ok && cudaStreamCreateWithFlags(&sl.aux.s[i], cudaStreamNonBlocking) == cudaSuccess;
            ok = ok && cudaEventCreateWithFlags(&sl.aux.join[i], cudaEventDisableTiming) == cudaSuccess;
        }
        ok = ok && cudaEventCreateWithFlags(&sl.aux.fork, cudaEventDisableTiming) == cudaSuccess;
        if (!ok) { tg_set_error("creating the auxiliary streams failed: %s", cudaGetErrorString(cudaGetLastError())); return nullptr; }
        sl.ready = true;
    }
    return &sl.aux;
}

extern "C" const char* tg_status_string(tg_status_t s) {
    switch (s) {
        case TG_OK: return "TG_OK";
        case TG_ERR_INVALID_ARG: return "TG_ERR_INVALID_ARG";
        case TG_ERR_UNSUPPORTED: return "TG_ERR_UNSUPPORTED";
        case TG_ERR_ALIGNMENT: return "TG_ERR_ALIGNMENT";
        case TG_ERR_WORKSPACE: return "TG_ERR_WORKSPACE";
        case TG_ERR_CUDA: return "TG_ERR_CUDA";
        case TG_ERR_INTERNAL: return "TG_ERR_INTERNAL";
    }
    return "TG_ERR_UNKNOWN";
}

extern "C" int tg_version(void) { return 100; }

extern "C" int tg_supported(int H, int D, tg_dtype_t dtype) { return tg_shape_supported(H, D, dtype) ? 1 : 0; }

// ---------------------------------------------------------------------------------------------
// tg_probe_gather: measures the L1 gather roof that the row-gather kernels sit against.  Every group of
// 8 lanes reads one 256-byte row (two LDG.128 per lane, one 128-byte line per group and instruction -- the
// access shape of rowops.cuh) at a pseudo-random index of a table of `table_rows` rows and xors it into a
// register; table_rows small => every access hits L1.  Returns the time of `iters` launches.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_probe_gather(const uint4* __restrict__ table, int table_rows, int gathers_per_group,
                                                       uint32_t* sink) {
    const int lane = threadIdx.x & 31, lig = lane & 7;
    uint32_t h = (blockIdx.x * blockDim.x + threadIdx.x) >> 3;   // group id
    uint4 acc = make_uint4(0, 0, 0, 0);
#pragma unroll 4
    for (int i = 0; i < gathers_per_group; ++i) {
        h = h * 1664525u + 1013904223u;
        const uint4* row = table + (size_t)((h >> 8) % (uint32_t)table_rows) * 16;   // 16 x 16 bytes per row
        const uint4 a = tg_ldg128(row + lig), b = tg_ldg128(row + lig + 8);
        acc.x ^= a.x ^ b.x; acc.y ^= a.y ^ b.y; acc.z ^= a.z ^ b.z; acc.w ^= a.w ^ b.w;
    }
    if ((acc.x ^ acc.y ^ acc.z ^ acc.w) == 0x12345678u) sink[0] = acc.x;   // keeps the loads alive
}

extern "C" tg_status_t tg_probe_gather(const void* table, int table_rows, int gathers_per_group, int iters, void* sink,
                                       tg_stream_t stream_, float* ms, double* bytes) {
    if (!table || !sink || !ms || !bytes || table_rows < 1 || gathers_per_group < 1 || iters < 1)
        TG_FAIL(TG_ERR_INVALID_ARG, "tg_probe_gather: bad argument");
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const int grid = 148 * 8;   // 8 CTAs of 256 threads per SM
    cudaEvent_t e0, e1;
    TG_CUDA(cudaEventCreate(&e0));
    TG_CUDA(cudaEventCreate(&e1));
    k_probe_gather<<<grid, 256, 0, stream>>>(static_cast<const uint4*>(table), table_rows, gathers_per_group, static_cast<uint32_t*>(sink));
    TG_LAUNCH_CHECK("k_probe_gather");
    TG_CUDA(cudaEventRecord(e0, stream));
    for (int i = 0; i < iters; ++i) {
        k_probe_gather<<<grid, 256, 0, stream>>>(static_cast<const uint4*>(table), table_rows, gathers_per_group, static_cast<uint32_t*>(sink));
        TG_LAUNCH_CHECK("k_probe_gather");
    }
    TG_CUDA(cudaEventRecord(e1, stream));
    TG_CUDA(cudaEventSynchronize(e1));
    TG_CUDA(cudaEventElapsedTime(ms, e0, e1));
    TG_CUDA(cudaEventDestroy(e0));
    TG_CUDA(cudaEventDestroy(e1));
    *bytes = (double)iters * grid * 32.0 /*groups per CTA*/ * gathers_per_group * 256.0;
    return TG_OK;
}
