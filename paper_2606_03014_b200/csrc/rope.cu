// rope.cu -- SURVEY.md section 8(f) N1, second half: rotary position embedding applied in place to
// the packed Q / K of the survivors' contexts, by the position_ids mosaic_assemble_context wrote.
// The paper runs Qwen-family aggregators inside vLLM and says nothing about the embedding
// itself; reading N1-4 fixes the convention those models use: pairs (i, i + D/2),
// w_i = theta^(-2 i / D), angle = position * w_i,
//     out[i]       = x[i] cos - x[i + D/2] sin,      out[i + D/2] = x[i + D/2] cos + x[i] sin.
//
// HBM-bound: every element of Q and K is read and written once (2 bytes each way).  A thread owns
// 8 frequencies of one token: angle and sin / cos in binary64 (8 per thread, amortised over all
// Hq + Hkv heads; positions reach 45 k, where an fp32 angle is already off by a bf16 ulp), then per
// head two 16-byte loads, 16 fp32 FMAs and two 16-byte stores.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "common.cuh"

namespace mosaic {
namespace {

constexpr int kRopeThreads = 256;

template <int D>
__global__ void __launch_bounds__(kRopeThreads) rope_kernel(__nv_bfloat16* __restrict__ q,
                                                            __nv_bfloat16* __restrict__ k,
                                                            const int32_t* __restrict__ position_ids,
                                                            int64_t T, int Hq, int Hkv,
                                                            double log2_theta) {
    constexpr int kPer = D / 16;  // threads per token: 8 frequencies each
    const int64_t gid = (int64_t)blockIdx.x * kRopeThreads + threadIdx.x;
    const int64_t tok = gid / kPer;
    if (tok >= T) return;
    const int i0 = (int)(gid - tok * kPer) * 8;
    const double pos = (double)position_ids[tok];
    float c[8], s[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
        const double w = exp2(-(2.0 * (i0 + u) / D) * log2_theta);
        double sn, cs;
        sincos(pos * w, &sn, &cs);
        c[u] = (float)cs;
        s[u] = (float)sn;
    }
    auto rotate = [&](__nv_bfloat16* row) {
        uint4 lo = *reinterpret_cast<const uint4*>(row + i0);
        uint4 hi = *reinterpret_cast<const uint4*>(row + i0 + D / 2);
        __nv_bfloat162* a = reinterpret_cast<__nv_bfloat162*>(&lo);
        __nv_bfloat162* b = reinterpret_cast<__nv_bfloat162*>(&hi);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const float2 x = __bfloat1622float2(a[u]), y = __bfloat1622float2(b[u]);
            const float ox0 = fmaf(x.x, c[2 * u], -(y.x * s[2 * u]));
            const float ox1 = fmaf(x.y, c[2 * u + 1], -(y.y * s[2 * u + 1]));
            const float oy0 = fmaf(y.x, c[2 * u], x.x * s[2 * u]);
            const float oy1 = fmaf(y.y, c[2 * u + 1], x.y * s[2 * u + 1]);
            a[u] = __floats2bfloat162_rn(ox0, ox1);
            b[u] = __floats2bfloat162_rn(oy0, oy1);
        }
        *reinterpret_cast<uint4*>(row + i0) = lo;
        *reinterpret_cast<uint4*>(row + i0 + D / 2) = hi;
    };
    __nv_bfloat16* qrow = q + tok * Hq * (int64_t)D;
    for (int h = 0; h < Hq; ++h) rotate(qrow + h * D);
    __nv_bfloat16* krow = k + tok * Hkv * (int64_t)D;
    for (int h = 0; h < Hkv; ++h) rotate(krow + h * D);
}

}  // namespace
}  // namespace mosaic

using namespace mosaic;

extern "C" mosaic_status_t mosaic_rope_packed(void* q, void* k, const int32_t* position_ids,
                                              int64_t total_tokens, int32_t Hq, int32_t Hkv,
                                              int32_t D, float theta, void* cuda_stream) {
    if (total_tokens < 0 || Hq < 0 || Hkv < 0 || !(theta > 0.f) || !isfinite(theta))
        return MOSAIC_ERR_INVALID_ARG;
    if (D != 64 && D != 128) return MOSAIC_ERR_UNSUPPORTED;
    if (total_tokens == 0 || Hq + Hkv == 0) return MOSAIC_OK;
    if (!position_ids || (Hq > 0 && (!q || !aligned16(q))) || (Hkv > 0 && (!k || !aligned16(k))))
        return MOSAIC_ERR_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const int64_t threads = total_tokens * (D / 16);
    const int64_t blocks = (threads + kRopeThreads - 1) / kRopeThreads;
    if (blocks >= (1ll << 31)) return MOSAIC_ERR_UNSUPPORTED;
    const double l2t = log2((double)theta);
    __nv_bfloat16* qp = static_cast<__nv_bfloat16*>(q);
    __nv_bfloat16* kp = static_cast<__nv_bfloat16*>(k);
    if (D == 64)
        rope_kernel<64><<<(unsigned)blocks, kRopeThreads, 0, s>>>(qp, kp, position_ids, total_tokens,
                                                                 Hq, Hkv, l2t);
    else
        rope_kernel<128><<<(unsigned)blocks, kRopeThreads, 0, s>>>(qp, kp, position_ids,
                                                                  total_tokens, Hq, Hkv, l2t);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());
    return MOSAIC_OK;
}
