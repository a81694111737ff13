// decode.cu -- SURVEY.md section 8(f) N2: the aggregator's GQA decode attention (one new q token per
// sequence against all its Lk cached keys; decode follows prefill in the aggregator).
// It is HBM-bound -- K and V are read once, 4 Hkv D bytes per key -- as long as (1) the G = Hq / Hkv
// q heads that share a KV head go through the tensor core TOGETHER and (2) there are enough
// independent pieces of work for 148 SMs even when the batch is a few long sequences.  This file
// arranges both around the prefill kernel, which stays as it is:
//   * the keys of every sequence are cut into chunks of C keys (C chosen on the host so that there
//     are a few chunk x KV-head units per SM); chunk j of sequence s is a virtual sequence v;
//   * the G heads of (s, kv head g) become the G q ROWS of v with a single q head per kv head,
//         Q'[v G + r, g, :] = Q[s, g G + r, :],
//     and mosaic_agg_prefill_attn_kv runs on (Q', K, V) with causal = 0: one 128-row tile per
//     (v, g) holding the G rows, every row seeing the chunk's keys;
//   * the partial results of a sequence's chunks are merged by their LSEs (as mosaic_lse_merge
//     does for two) into O and LSE.
// The helper kernels move O(n_seqs Hq D) elements per chunk: nothing next to the K / V stream.
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
    int64_t *cu_q, *cu_k;
    int* first_v;  // [n_seqs + 1] first virtual sequence of every sequence
    void* attn_ws;
    size_t attn_ws_bytes, total;
};

// Upper bound on the number of virtual sequences: every sequence has at least one chunk.
inline int64_t max_virtual(int32_t n_seqs, int64_t total_k_tokens, int chunk) {
    return total_k_tokens / chunk + n_seqs;
}
// Chunk length (a multiple of 128 keys): about four (chunk, kv head) units per SM.
inline int choose_chunk(int64_t total_k_tokens, int32_t Hkv) {
    int64_t c = total_k_tokens * Hkv / (4 * (int64_t)num_sms());
    c = (c + 127) / 128 * 128;
    if (c < 512) c = 512;
    if (c > 8192) c = 8192;
    return (int)c;
}

DecodeWs carve_decode(void* base, int32_t n_seqs, int64_t v_max, int32_t Hq, int32_t Hkv,
                      int32_t D) {
    DecodeWs w{};
    char* p = static_cast<char*>(base);
    size_t off = 0;
    auto take = [&](size_t bytes) {
        char* r = p + off;
        off += (bytes + 255) & ~size_t(255);
        return r;
    };
    const size_t rows = (size_t)v_max * Hq;
    w.q2 = reinterpret_cast<__nv_bfloat16*>(take(rows * D * 2));
    w.o2 = reinterpret_cast<__nv_bfloat16*>(take(rows * D * 2));
    w.lse2 = reinterpret_cast<float*>(take(rows * 4));
    w.cu_q = reinterpret_cast<int64_t*>(take((size_t)(v_max + 1) * 8));
    w.cu_k = reinterpret_cast<int64_t*>(take((size_t)(v_max + 1) * 8));
    w.first_v = reinterpret_cast<int*>(take((size_t)(n_seqs + 1) * 4));
    const int G = Hkv > 0 ? Hq / Hkv : 1;
    w.attn_ws_bytes =
        mosaic_agg_prefill_attn_workspace_bytes((int32_t)v_max, v_max * G, Hkv, Hkv, D);
    w.attn_ws = take(w.attn_ws_bytes);
    w.total = off;
    return w;
}

// One block: chunks per sequence, their exclusive scan, and the unused tail of the two cu arrays.
__global__ void __launch_bounds__(1024) decode_plan(const int64_t* __restrict__ cu_seqlens_k,
                                                    int n_seqs, int chunk, int G, int64_t v_max,
                                                    int64_t total_k, int* __restrict__ first_v,
                                                    int64_t* __restrict__ cu_q,
                                                    int64_t* __restrict__ cu_k) {
    __shared__ int warp_tot[32];
    __shared__ int carry;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) carry = 0;
    __syncthreads();
    for (int s0 = 0; s0 < n_seqs; s0 += 1024) {
        const int s = s0 + tid;
        int nc = 0;
        if (s < n_seqs) {
            const int64_t L = cu_seqlens_k[s + 1] - cu_seqlens_k[s];
            nc = L > 0 ? (int)((L + chunk - 1) / chunk) : 1;
        }
        int x = nc;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) warp_tot[warp] = x;
        __syncthreads();
        int before = carry;
        for (int w = 0; w < warp; ++w) before += warp_tot[w];
        if (s < n_seqs) first_v[s] = before + x - nc;
        __syncthreads();
        if (tid == 1023) carry = before + x;
        __syncthreads();
    }
    const int n_virt = carry;
    if (tid == 0) first_v[n_seqs] = n_virt;
    for (int64_t v = n_virt + tid; v <= v_max; v += 1024) {  // unused slots: empty sequences
        cu_q[v] = (int64_t)n_virt * G;
        cu_k[v] = total_k;
    }
}

// Block s: the cu entries of its chunks and their Q' rows (16 bytes per thread per element group).
__global__ void __launch_bounds__(256) decode_pack(const __nv_bfloat16* __restrict__ q,
                                                   const int64_t* __restrict__ cu_seqlens_k,
                                                   const int* __restrict__ first_v, int chunk,
                                                   int Hkv, int G, int D,
                                                   __nv_bfloat16* __restrict__ q2,
                                                   int64_t* __restrict__ cu_q,
                                                   int64_t* __restrict__ cu_k) {
    const int s = blockIdx.x;
    const int v0 = first_v[s], nc = first_v[s + 1] - v0;
    const int64_t k0 = cu_seqlens_k[s];
    for (int j = threadIdx.x; j < nc; j += 256) {
        cu_q[v0 + j] = (int64_t)(v0 + j) * G;
        cu_k[v0 + j] = k0 + (int64_t)j * chunk;
    }
    const int per = D / 8, Hq = Hkv * G;
    const int n = nc * Hq * per;
    for (int x = threadIdx.x; x < n; x += 256) {
        const int c = x % per;
        const int hq = (x / per) % Hq;  // q head = g G + r
        const int j = x / (per * Hq);
        const int g = hq / G, r = hq - g * G;
        const int64_t row2 = ((int64_t)(v0 + j) * G + r) * Hkv + g;
        reinterpret_cast<uint4*>(q2 + row2 * D)[c] =
            reinterpret_cast<const uint4*>(q + ((int64_t)s * Hq + hq) * D)[c];
    }
}

// Thread (s, h, 8 elements): merges the chunks' partial results by their LSEs.
__global__ void __launch_bounds__(256) decode_reduce(const __nv_bfloat16* __restrict__ o2,
                                                     const float* __restrict__ lse2,
                                                     const int64_t* __restrict__ cu_seqlens_k,
                                                     const int* __restrict__ first_v, int n_seqs,
                                                     int64_t lse2_stride, int Hkv, int G, int D,
                                                     __nv_bfloat16* __restrict__ o,
                                                     float* __restrict__ lse) {
    const int per = D / 8, Hq = Hkv * G;
    const int64_t gid = (int64_t)blockIdx.x * 256 + threadIdx.x;
    const int64_t row = gid / per;  // (s, hq)
    if (row >= (int64_t)n_seqs * Hq) return;
    const int c = (int)(gid - row * per);
    const int hq = (int)(row % Hq);
    const int s = (int)(row / Hq);
    const int g = hq / G, r = hq - g * G;
    const int v0 = first_v[s];
    // (a sequence without keys has one empty chunk whose partial result was never written)
    const int nc = cu_seqlens_k[s + 1] > cu_seqlens_k[s] ? first_v[s + 1] - v0 : 0;
    // LSE' is [Hkv, lse2_stride] with column v G + r
    float m = -INFINITY;
    for (int j = 0; j < nc; ++j)
        m = fmaxf(m, lse2[(int64_t)g * lse2_stride + (int64_t)(v0 + j) * G + r]);
    float acc[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) acc[u] = 0.f;
    float z = 0.f;
    for (int j = 0; j < nc; ++j) {
        const float l = lse2[(int64_t)g * lse2_stride + (int64_t)(v0 + j) * G + r];
        if (l == -INFINITY) continue;  // an empty chunk (a sequence without keys)
        const float w = expf(l - m);
        z += w;
        const int64_t row2 = ((int64_t)(v0 + j) * G + r) * Hkv + g;
        const uint4 v = reinterpret_cast<const uint4*>(o2 + row2 * D)[c];
        const __nv_bfloat162* pv = reinterpret_cast<const __nv_bfloat162*>(&v);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const float2 f = __bfloat1622float2(pv[u]);
            acc[2 * u] = fmaf(f.x, w, acc[2 * u]);
            acc[2 * u + 1] = fmaf(f.y, w, acc[2 * u + 1]);
        }
    }
    const float inv = z > 0.f ? 1.f / z : 0.f;
    uint4 out;
    __nv_bfloat162* po = reinterpret_cast<__nv_bfloat162*>(&out);
#pragma unroll
    for (int u = 0; u < 4; ++u) po[u] = __floats2bfloat162_rn(acc[2 * u] * inv, acc[2 * u + 1] * inv);
    reinterpret_cast<uint4*>(o + row * D)[c] = out;
    if (c == 0) lse[(int64_t)hq * n_seqs + s] = z > 0.f ? m + logf(z) : -INFINITY;
}

}  // namespace
}  // namespace mosaic

using namespace mosaic;

extern "C" size_t mosaic_agg_decode_attn_workspace_bytes(int32_t n_seqs, int64_t total_k_tokens,
                                                         int32_t Hq, int32_t Hkv, int32_t D) {
    if (n_seqs < 0 || total_k_tokens < 0 || Hq < 1 || Hkv < 1 || D < 8 || Hq % Hkv != 0) return 0;
    const int chunk = choose_chunk(total_k_tokens, Hkv);
    return carve_decode(nullptr, n_seqs, max_virtual(n_seqs, total_k_tokens, chunk), Hq, Hkv, D)
        .total;
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
    const int chunk = choose_chunk(total_k_tokens, Hkv);
    const int64_t v_max = max_virtual(n_seqs, total_k_tokens, chunk);
    if (v_max * G >= (1ll << 31)) return MOSAIC_ERR_UNSUPPORTED;
    DecodeWs w = carve_decode(workspace, n_seqs, v_max, Hq, Hkv, D);
    if (workspace_bytes < w.total) return MOSAIC_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    decode_plan<<<1, 1024, 0, s>>>(cu_seqlens_k, n_seqs, chunk, G, v_max, total_k_tokens, w.first_v,
                                   w.cu_q, w.cu_k);
    count_launch();
    decode_pack<<<(unsigned)n_seqs, 256, 0, s>>>(static_cast<const __nv_bfloat16*>(q), cu_seqlens_k,
                                                 w.first_v, chunk, Hkv, G, D, w.q2, w.cu_q, w.cu_k);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());
    mosaic_status_t st = mosaic_agg_prefill_attn_kv(
        w.q2, k, v, w.cu_q, w.cu_k, (int32_t)v_max, v_max * G, total_k_tokens, G, Hkv, Hkv, D,
        softmax_scale, /*causal=*/0, w.o2, w.lse2, w.attn_ws, w.attn_ws_bytes, cuda_stream);
    if (st != MOSAIC_OK) return st;
    const int64_t threads = (int64_t)n_seqs * Hq * (D / 8);
    decode_reduce<<<(unsigned)((threads + 255) / 256), 256, 0, s>>>(
        w.o2, w.lse2, cu_seqlens_k, w.first_v, n_seqs, v_max * G, Hkv, G, D,
        static_cast<__nv_bfloat16*>(o), lse);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());
    return MOSAIC_OK;
}
