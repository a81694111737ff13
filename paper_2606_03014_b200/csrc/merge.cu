// merge.cu -- SURVEY.md section 8(f) N2: merging the partial attention results of two disjoint
// key sets for the same q rows (split-KV / chunked prefill of the aggregator's long contexts).
// With (O_a, LSE_a) over keys A and (O_b, LSE_b) over keys B, the result over A u B is
//     LSE = ln(e^LSE_a + e^LSE_b),   O = O_a e^(LSE_a - LSE) + O_b e^(LSE_b - LSE)
// (the softmax weights of a row over A u B are those over A scaled by e^(LSE_a - LSE), and likewise
// for B).  LSE = -inf marks an empty partial (weight 0).
//
// HBM-bound elementwise: a thread takes 8 consecutive elements of one (token, head) row: two
// 16-byte loads, fp32 math, one 16-byte store; the thread of a row's first chunk writes its LSE.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "common.cuh"

namespace mosaic {
namespace {

constexpr int kMergeThreads = 256;

__global__ void __launch_bounds__(kMergeThreads) lse_merge_kernel(
    const __nv_bfloat16* __restrict__ oa, const float* __restrict__ la,
    const __nv_bfloat16* __restrict__ ob, const float* __restrict__ lb, int64_t T, int Hq, int D,
    __nv_bfloat16* __restrict__ o, float* __restrict__ lse) {
    // two 8-element chunks of a row per thread when the row has an even number of them: the row's
    // LSE pair and weights are computed once for both, and four loads are in flight
    const int n_sub = (D % 16 == 0) ? 2 : 1;
    const int per_row = D / (8 * n_sub);
    const int64_t gid = (int64_t)blockIdx.x * kMergeThreads + threadIdx.x;
    const int64_t rowi = gid / per_row;  // (token, head) row
    if (rowi >= T * Hq) return;
    const int c = (int)(gid - rowi * per_row);
    const int64_t t = rowi / Hq;
    const int h = (int)(rowi - t * Hq);
    const float xa = la[(int64_t)h * T + t], xb = lb[(int64_t)h * T + t];
    uint4 va[2], vb[2];
#pragma unroll
    for (int u = 0; u < 2; ++u) {
        if (u < n_sub) {
            va[u] = *reinterpret_cast<const uint4*>(oa + rowi * D + (c + u * per_row) * 8);
            vb[u] = *reinterpret_cast<const uint4*>(ob + rowi * D + (c + u * per_row) * 8);
        }
    }
    const float m = fmaxf(xa, xb);
    float wa = 0.f, wb = 0.f, out_lse = -INFINITY;
    if (m > -INFINITY) {
        const float ea = expf(xa - m), eb = expf(xb - m);  // exp(-inf) = 0 for an empty partial
        const float z = ea + eb;
        wa = ea / z;
        wb = eb / z;
        out_lse = m + logf(z);
    }
#pragma unroll
    for (int u = 0; u < 2; ++u) {
        if (u < n_sub) {
            const __nv_bfloat162* pa = reinterpret_cast<const __nv_bfloat162*>(&va[u]);
            const __nv_bfloat162* pb = reinterpret_cast<const __nv_bfloat162*>(&vb[u]);
            uint4 vo;
            __nv_bfloat162* po = reinterpret_cast<__nv_bfloat162*>(&vo);
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const float2 a = __bfloat1622float2(pa[e]), b = __bfloat1622float2(pb[e]);
                // (a weight of exactly 0 must not turn an uninitialised partial into NaN)
                const float x = (wa != 0.f ? a.x * wa : 0.f) + (wb != 0.f ? b.x * wb : 0.f);
                const float y = (wa != 0.f ? a.y * wa : 0.f) + (wb != 0.f ? b.y * wb : 0.f);
                po[e] = __floats2bfloat162_rn(x, y);
            }
            *reinterpret_cast<uint4*>(o + rowi * D + (c + u * per_row) * 8) = vo;
        }
    }
    if (c == 0) lse[(int64_t)h * T + t] = out_lse;
}

}  // namespace
}  // namespace mosaic

using namespace mosaic;

extern "C" mosaic_status_t mosaic_lse_merge(const void* o_a, const float* lse_a, const void* o_b,
                                            const float* lse_b, int64_t total_tokens, int32_t Hq,
                                            int32_t D, void* o, float* lse, void* cuda_stream) {
    if (total_tokens < 0 || Hq < 1 || D < 8 || D % 8 != 0) return MOSAIC_ERR_INVALID_ARG;
    if (total_tokens == 0) return MOSAIC_OK;
    if (!o_a || !o_b || !lse_a || !lse_b || !o || !lse || !aligned16(o_a) || !aligned16(o_b) ||
        !aligned16(o))
        return MOSAIC_ERR_INVALID_ARG;
    const int64_t threads = total_tokens * Hq * (D % 16 == 0 ? D / 16 : D / 8);
    const int64_t blocks = (threads + kMergeThreads - 1) / kMergeThreads;
    if (blocks >= (1ll << 31)) return MOSAIC_ERR_UNSUPPORTED;
    lse_merge_kernel<<<(unsigned)blocks, kMergeThreads, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
        static_cast<const __nv_bfloat16*>(o_a), lse_a, static_cast<const __nv_bfloat16*>(o_b), lse_b,
        total_tokens, Hq, D, static_cast<__nv_bfloat16*>(o), lse);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());
    return MOSAIC_OK;
}

// ------------------------------------------------------------------------------------------
// mosaic_lse_merge_n: the same merge for n partial results at once (the chunks of a split-KV
// pass): LSE = ln sum_p e^LSE_p, O = sum_p O_p e^(LSE_p - LSE).  A thread takes 8 consecutive
// elements of one (token, head) row and walks the n parts twice (the row's n logsumexps for the
// maximum, then the weighted sum in fp32): every O_p element is read once.
namespace mosaic {
namespace {
__global__ void __launch_bounds__(kMergeThreads) lse_merge_n_kernel(
    const __nv_bfloat16* __restrict__ o_parts, const float* __restrict__ lse_parts, int n_parts,
    int64_t T, int Hq, int D, __nv_bfloat16* __restrict__ o, float* __restrict__ lse) {
    const int per_row = D / 8;
    const int64_t gid = (int64_t)blockIdx.x * kMergeThreads + threadIdx.x;
    const int64_t rowi = gid / per_row;  // (token, head) row
    if (rowi >= T * Hq) return;
    const int c = (int)(gid - rowi * per_row);
    const int64_t t = rowi / Hq;
    const int h = (int)(rowi - t * Hq);
    const int64_t o_stride = T * (int64_t)Hq * D, l_stride = (int64_t)Hq * T;
    const float* lrow = lse_parts + (int64_t)h * T + t;
    const __nv_bfloat16* orow = o_parts + rowi * D + c * 8;
    // One pass, four parts in flight: running maximum m, weights relative to it, the accumulator
    // rescaled when the maximum moves (an empty partial -- LSE = -inf -- has weight 0 and its O,
    // which may be uninitialised, is multiplied by nothing).
    float m = -INFINITY, z = 0.f;
    float acc[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) acc[u] = 0.f;
    for (int p0 = 0; p0 < n_parts; p0 += 4) {
        float l[4];
        uint4 v[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const bool in = p0 + j < n_parts;
            l[j] = in ? __ldg(lrow + (int64_t)(p0 + j) * l_stride) : -INFINITY;
            v[j] = in ? __ldcs(reinterpret_cast<const uint4*>(orow + (int64_t)(p0 + j) * o_stride))
                      : make_uint4(0u, 0u, 0u, 0u);
        }
        const float m_new = fmaxf(fmaxf(m, fmaxf(l[0], l[1])), fmaxf(l[2], l[3]));
        if (m_new == -INFINITY) continue;
        const float r = m == -INFINITY ? 0.f : expf(m - m_new);
        z *= r;
#pragma unroll
        for (int u = 0; u < 8; ++u) acc[u] *= r;
        m = m_new;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if (l[j] == -INFINITY) continue;
            const float w = expf(l[j] - m);
            z += w;
            const __nv_bfloat162* pv = reinterpret_cast<const __nv_bfloat162*>(&v[j]);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float2 f = __bfloat1622float2(pv[u]);
                acc[2 * u] = fmaf(f.x, w, acc[2 * u]);
                acc[2 * u + 1] = fmaf(f.y, w, acc[2 * u + 1]);
            }
        }
    }
    const float inv = z > 0.f ? 1.f / z : 0.f;
    uint4 out;
    __nv_bfloat162* po = reinterpret_cast<__nv_bfloat162*>(&out);
#pragma unroll
    for (int u = 0; u < 4; ++u) po[u] = __floats2bfloat162_rn(acc[2 * u] * inv, acc[2 * u + 1] * inv);
    *reinterpret_cast<uint4*>(o + rowi * D + c * 8) = out;
    if (c == 0) lse[(int64_t)h * T + t] = z > 0.f ? m + logf(z) : -INFINITY;
}
}  // namespace
}  // namespace mosaic

extern "C" mosaic_status_t mosaic_lse_merge_n(const void* o_parts, const float* lse_parts,
                                              int32_t n_parts, int64_t total_tokens, int32_t Hq,
                                              int32_t D, void* o, float* lse, void* cuda_stream) {
    if (n_parts < 1 || total_tokens < 0 || Hq < 1 || D < 8 || D % 8 != 0)
        return MOSAIC_ERR_INVALID_ARG;
    if (total_tokens == 0) return MOSAIC_OK;
    if (!o_parts || !lse_parts || !o || !lse || !aligned16(o_parts) || !aligned16(o))
        return MOSAIC_ERR_INVALID_ARG;
    const int64_t threads = total_tokens * Hq * (D / 8);
    const int64_t blocks = (threads + kMergeThreads - 1) / kMergeThreads;
    if (blocks >= (1ll << 31)) return MOSAIC_ERR_UNSUPPORTED;
    lse_merge_n_kernel<<<(unsigned)blocks, kMergeThreads, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
        static_cast<const __nv_bfloat16*>(o_parts), lse_parts, n_parts, total_tokens, Hq, D,
        static_cast<__nv_bfloat16*>(o), lse);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());
    return MOSAIC_OK;
}
