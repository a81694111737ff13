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
// elements of one (token, head) row and walks the n parts once, two at a time, with a running
// maximum (an online softmax over the parts): every O_p element is read once.
namespace mosaic {
namespace {
__device__ __forceinline__ float ex2_approx(float x) {  // 2^x, 2 ulp; 2^-inf = 0
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// What bounds this kernel is the bytes in flight per SM, i.e. occupancy: at 61 registers (four parts
// in flight per thread, 4 blocks of 256 threads per SM) it ran at 5.0 TB/s; at 32 registers -- two
// parts in flight, 16 blocks of 128 threads, all 2048 thread slots of an SM -- at 5.85 TB/s.
// idx_t: 32-bit chunk / row indices whenever the call's chunk count fits (32-bit divisions).
constexpr int kMergeNThreads = 128;
constexpr int kMergeNBlocksPerSM = 16;
constexpr int kMergeNInFlight = 2;  // parts in flight per thread
template <typename idx_t>
__global__ void __launch_bounds__(kMergeNThreads, kMergeNBlocksPerSM) lse_merge_n_kernel(
    const __nv_bfloat16* __restrict__ o_parts, const float* __restrict__ lse_parts, int n_parts,
    int64_t T, int Hq, int D, __nv_bfloat16* __restrict__ o, float* __restrict__ lse) {
    const idx_t per_row = (idx_t)(D / 8);
    const idx_t gid = (idx_t)blockIdx.x * kMergeNThreads + threadIdx.x;  // 16-byte chunk of O
    const idx_t rowi = gid / per_row;                                   // (token, head) row
    if (rowi >= (idx_t)T * (idx_t)Hq) return;
    const idx_t t = rowi / (idx_t)Hq;
    const idx_t h = rowi - t * (idx_t)Hq;
    const int64_t o_stride = T * (int64_t)Hq * D, l_stride = (int64_t)Hq * T;
    const float* lrow = lse_parts + (int64_t)h * T + (int64_t)t;
    const __nv_bfloat16* orow = o_parts + (int64_t)gid * 8;
    // One pass, PF parts in flight: running maximum m, weights relative to it, the accumulator
    // rescaled when the maximum moves (an empty partial -- LSE = -inf -- has weight 0 and its O,
    // which may be uninitialised, is multiplied by nothing).
    constexpr float kLog2e = 1.4426950408889634f;
    float m = -INFINITY, z = 0.f;
    float acc[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) acc[u] = 0.f;
    constexpr int PF = kMergeNInFlight;
    for (int p0 = 0; p0 < n_parts; p0 += PF) {
        float l[PF];
        uint4 v[PF];
#pragma unroll
        for (int j = 0; j < PF; ++j) {
            const bool in = p0 + j < n_parts;
            l[j] = in ? __ldg(lrow + (int64_t)(p0 + j) * l_stride) : -INFINITY;
            v[j] = in ? __ldcs(reinterpret_cast<const uint4*>(orow + (int64_t)(p0 + j) * o_stride))
                      : make_uint4(0u, 0u, 0u, 0u);
        }
        float m_new = m;
#pragma unroll
        for (int j = 0; j < PF; ++j) m_new = fmaxf(m_new, l[j]);
        if (m_new == -INFINITY) continue;
        const float r = ex2_approx((m - m_new) * kLog2e);  // m = -inf (nothing yet): 0
        z *= r;
#pragma unroll
        for (int u = 0; u < 8; ++u) acc[u] *= r;
        m = m_new;
#pragma unroll
        for (int j = 0; j < PF; ++j) {
            const float w = ex2_approx((l[j] - m) * kLog2e);
            if (w == 0.f) continue;
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
    *reinterpret_cast<uint4*>(o + (int64_t)gid * 8) = out;
    if (gid == rowi * per_row) lse[(int64_t)h * T + (int64_t)t] = z > 0.f ? m + logf(z) : -INFINITY;
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
    const int64_t blocks = (threads + kMergeNThreads - 1) / kMergeNThreads;
    if (blocks >= (1ll << 31)) return MOSAIC_ERR_UNSUPPORTED;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    if (blocks * kMergeNThreads < (1ll << 32))
        lse_merge_n_kernel<uint32_t><<<(unsigned)blocks, kMergeNThreads, 0, s>>>(
            static_cast<const __nv_bfloat16*>(o_parts), lse_parts, n_parts, total_tokens, Hq, D,
            static_cast<__nv_bfloat16*>(o), lse);
    else
        lse_merge_n_kernel<int64_t><<<(unsigned)blocks, kMergeNThreads, 0, s>>>(
            static_cast<const __nv_bfloat16*>(o_parts), lse_parts, n_parts, total_tokens, Hq, D,
            static_cast<__nv_bfloat16*>(o), lse);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());
    return MOSAIC_OK;
}
