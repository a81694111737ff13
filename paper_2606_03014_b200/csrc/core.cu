// core.cu -- status strings, version, launch counter, device query.
#include <atomic>

#include "common.cuh"

namespace mosaic {
thread_local int g_last_cuda_error = 0;
static std::atomic<int64_t> g_launches{0};
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

int num_sms() {
    thread_local int cached = 0;
    if (cached == 0) {
        int dev = 0, n = 0;
        if (cudaGetDevice(&dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0)
            cached = n;
        else
            return kNumSMsB200;
    }
    return cached;
}
}  // namespace mosaic

extern "C" const char* mosaic_status_string(mosaic_status_t status) {
    switch (status) {
        case MOSAIC_OK: return "MOSAIC_OK";
        case MOSAIC_ERR_INVALID_ARG: return "MOSAIC_ERR_INVALID_ARG";
        case MOSAIC_ERR_UNSUPPORTED: return "MOSAIC_ERR_UNSUPPORTED";
        case MOSAIC_ERR_WORKSPACE_TOO_SMALL: return "MOSAIC_ERR_WORKSPACE_TOO_SMALL";
        case MOSAIC_ERR_CUDA: return "MOSAIC_ERR_CUDA";
    }
    return "MOSAIC_ERR_UNKNOWN";
}

extern "C" int mosaic_version(void) { return 100; }
extern "C" int mosaic_last_cuda_error(void) { return mosaic::g_last_cuda_error; }
extern "C" int64_t mosaic_kernel_launch_count(void) {
    return mosaic::g_launches.load(std::memory_order_relaxed);
}
