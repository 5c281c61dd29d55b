// api.cu -- status strings, thread-local error text, version and capability queries.
#include <stdarg.h>

#include <atomic>

#include "dispatch.cuh"

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
