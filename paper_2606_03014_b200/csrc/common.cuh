// common.cuh -- host-side helpers shared by the translation units of libmosaic.so.
// Product code: includes nothing from oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "mosaic.h"

namespace mosaic {

// Last failed CUDA call on this thread (mosaic_last_cuda_error()).
extern thread_local int g_last_cuda_error;
// Kernels enqueued since load (mosaic_kernel_launch_count()).
void count_launch(int n = 1);

inline mosaic_status_t cuda_fail(cudaError_t e) {
    g_last_cuda_error = static_cast<int>(e);
    return MOSAIC_ERR_CUDA;
}

#define MOSAIC_CUDA_TRY(expr)                                   \
    do {                                                        \
        cudaError_t e__ = (expr);                               \
        if (e__ != cudaSuccess) return ::mosaic::cuda_fail(e__); \
    } while (0)

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

constexpr int kNumSMsB200 = 148;

// Number of SMs of the current device (cached per thread; 148 on B200).
int num_sms();

}  // namespace mosaic
