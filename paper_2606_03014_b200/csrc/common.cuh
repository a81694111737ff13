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

// One sequence of an attention call as explicit views (attn.cu: attn_impl with `desc`): q rows
// [q_start, q_start + q_len) of the packed q / o / lse, keys [k_start, k_start + k_len) of k / v.
struct SeqDesc {
    int64_t q_start, k_start;
    int32_t q_len, k_len;
};
// The attention behind mosaic_agg_prefill_attn[_kv] (attn.cu), for the entry points built on it.
// k_prefix / v_prefix [prefix_len, Hkv, D]: a block of keys every sequence sees in front of its own
// (causal only; the shared-prefix cascade).
mosaic_status_t attn_impl(const void* q, const void* k, const void* v, const int64_t* cu_seqlens,
                          const int64_t* cu_seqlens_k, const SeqDesc* desc, int32_t n_seqs,
                          int64_t total_tokens, int64_t total_k_tokens, int32_t max_seqlen,
                          int32_t Hq, int32_t Hkv, int32_t D, float softmax_scale, int causal,
                          void* o, float* lse, void* workspace, size_t workspace_bytes,
                          void* cuda_stream, const void* k_prefix = nullptr,
                          const void* v_prefix = nullptr, int32_t prefix_len = 0);

// Number of SMs of the current device (cached per thread; 148 on B200).
int num_sms();

}  // namespace mosaic
