// decode.cu -- SURVEY.md section 8(f) N2: the aggregator's GQA decode attention (one new q token per
// sequence against all its Lk cached keys; decode follows prefill in the aggregator).
// It is HBM-bound -- K and V are read once, 4 Hkv D bytes per key -- as long as the G = Hq / Hkv
// q heads that share a KV head go through the tensor core TOGETHER.  That is what this file
// arranges, with the prefill kernel unchanged: the G heads of (sequence s, kv head g) are
// re-packed as the G q ROWS of a virtual sequence with a single q head per kv head,
//     Q'[s G + r, g, :] = Q[s, g G + r, :],
// mosaic_agg_prefill_attn_kv runs on (Q', K, V) with causal = 0 (every row sees all Lk keys), one
// 128-row tile per (s, g) holding the G rows, and O / LSE are unpacked the same way.  The two
// re-packing kernels move n_seqs Hq D elements: nothing next to the K / V stream.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "common.cuh"

namespace mosaic {
namespace {

struct DecodeWs {
    __nv_bfloat16 *q2, *o2;
    float* lse2;
    int64_t* cu_q;
    void* attn_ws;
    size_t attn_ws_bytes, total;
};

DecodeWs carve_decode(void* base, int32_t n_seqs, int32_t Hq, int32_t Hkv, int32_t D) {
    DecodeWs w{};
    char* p = static_cast<char*>(base);
    size_t off = 0;
    auto take = [&](size_t bytes) {
        char* r = p + off;
        off += (bytes + 255) & ~size_t(255);
        return r;
    };
    const size_t rows = (size_t)n_seqs * Hq;
    w.q2 = reinterpret_cast<__nv_bfloat16*>(take(rows * D * 2));
    w.o2 = reinterpret_cast<__nv_bfloat16*>(take(rows * D * 2));
    w.lse2 = reinterpret_cast<float*>(take(rows * 4));
    w.cu_q = reinterpret_cast<int64_t*>(take((size_t)(n_seqs + 1) * 8));
    const int G = Hkv > 0 ? Hq / Hkv : 1;
    w.attn_ws_bytes =
        mosaic_agg_prefill_attn_workspace_bytes(n_seqs, (int64_t)n_seqs * G, Hkv, Hkv, D);
    w.attn_ws = take(w.attn_ws_bytes);
    w.total = off;
    return w;
}

// 8 elements (16 bytes) per thread.  pack: Q -> Q' and cu_q[s] = s G; unpack: O' -> O, LSE' -> LSE.
__global__ void __launch_bounds__(256) decode_pack(const __nv_bfloat16* __restrict__ q,
                                                   __nv_bfloat16* __restrict__ q2,
                                                   int64_t* __restrict__ cu_q, int n_seqs, int Hkv,
                                                   int G, int D) {
    const int per = D / 8;
    const int64_t gid = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (gid <= n_seqs) cu_q[gid] = gid * G;
    const int64_t row = gid / per;  // row of Q: (s, g, r)
    if (row >= (int64_t)n_seqs * Hkv * G) return;
    const int c = (int)(gid - row * per);
    const int r = (int)(row % G);
    const int g = (int)((row / G) % Hkv);
    const int64_t s = row / ((int64_t)G * Hkv);
    const int64_t row2 = (s * G + r) * Hkv + g;
    reinterpret_cast<uint4*>(q2 + row2 * D)[c] = reinterpret_cast<const uint4*>(q + row * D)[c];
}

__global__ void __launch_bounds__(256) decode_unpack(const __nv_bfloat16* __restrict__ o2,
                                                     const float* __restrict__ lse2,
                                                     __nv_bfloat16* __restrict__ o,
                                                     float* __restrict__ lse, int n_seqs, int Hkv,
                                                     int G, int D) {
    const int per = D / 8;
    const int64_t gid = (int64_t)blockIdx.x * 256 + threadIdx.x;
    const int64_t row = gid / per;
    if (row >= (int64_t)n_seqs * Hkv * G) return;
    const int c = (int)(gid - row * per);
    const int r = (int)(row % G);
    const int g = (int)((row / G) % Hkv);
    const int64_t s = row / ((int64_t)G * Hkv);
    const int64_t row2 = (s * G + r) * Hkv + g;
    reinterpret_cast<uint4*>(o + row * D)[c] = reinterpret_cast<const uint4*>(o2 + row2 * D)[c];
    // LSE' is [Hkv, n_seqs G]; LSE is [Hq, n_seqs]
    if (c == 0) lse[(int64_t)(g * G + r) * n_seqs + s] = lse2[(int64_t)g * n_seqs * G + s * G + r];
}

}  // namespace
}  // namespace mosaic

using namespace mosaic;

extern "C" size_t mosaic_agg_decode_attn_workspace_bytes(int32_t n_seqs, int32_t Hq, int32_t Hkv,
                                                         int32_t D) {
    if (n_seqs < 0 || Hq < 1 || Hkv < 1 || D < 8 || Hq % Hkv != 0) return 0;
    return carve_decode(nullptr, n_seqs, Hq, Hkv, D).total;
}

extern "C" mosaic_status_t mosaic_agg_decode_attn(const void* q, const void* k, const void* v,
                                                  const int64_t* cu_seqlens_k, int32_t n_seqs,
                                                  int64_t total_k_tokens, int32_t Hq, int32_t Hkv,
                                                  int32_t D, float softmax_scale, void* o,
                                                  float* lse, void* workspace,
                                                  size_t workspace_bytes, void* cuda_stream) {
    if (n_seqs < 0 || total_k_tokens < 0 || Hq < 1 || Hkv < 1 || Hq % Hkv != 0 ||
        !isfinite(softmax_scale))
        return MOSAIC_ERR_INVALID_ARG;
    if (D != 64 && D != 128) return MOSAIC_ERR_UNSUPPORTED;
    const int G = Hq / Hkv;
    if (G > 128) return MOSAIC_ERR_UNSUPPORTED;  // the heads of a group share one 128-row tile
    if (n_seqs == 0) return MOSAIC_OK;
    if (!q || !k || !v || !o || !lse || !cu_seqlens_k || !workspace || !aligned16(q) ||
        !aligned16(o) || !aligned16(workspace))
        return MOSAIC_ERR_INVALID_ARG;
    DecodeWs w = carve_decode(workspace, n_seqs, Hq, Hkv, D);
    if (workspace_bytes < w.total) return MOSAIC_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const int64_t threads = (int64_t)n_seqs * Hq * (D / 8);
    const int64_t need = threads > n_seqs + 1 ? threads : n_seqs + 1;
    const unsigned blocks = (unsigned)((need + 255) / 256);
    decode_pack<<<blocks, 256, 0, s>>>(static_cast<const __nv_bfloat16*>(q), w.q2, w.cu_q, n_seqs,
                                       Hkv, G, D);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());
    mosaic_status_t st = mosaic_agg_prefill_attn_kv(
        w.q2, k, v, w.cu_q, cu_seqlens_k, n_seqs, (int64_t)n_seqs * G, total_k_tokens, G, Hkv, Hkv,
        D, softmax_scale, /*causal=*/0, w.o2, w.lse2, w.attn_ws, w.attn_ws_bytes, cuda_stream);
    if (st != MOSAIC_OK) return st;
    decode_unpack<<<(unsigned)((threads + 255) / 256), 256, 0, s>>>(
        w.o2, w.lse2, static_cast<__nv_bfloat16*>(o), lse, n_seqs, Hkv, G, D);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());
    return MOSAIC_OK;
}
