// cascade.cu -- SURVEY.md section 8(f) N2, the LSE-merge variants built on the prefill kernel:
//   mosaic_agg_prefill_attn_chunked        chunked prefill of long contexts (32 k-class
//                                          windows; configs[2] allows 45 312 tokens) in ONE launch
//   mosaic_agg_prefill_attn_shared_prefix  shared-prefix cascade: every survivor's context starts
//                                          with the same block of keys (the aggregator's prompt
//                                          template, P:L225 / P:L377 `Aggregator(q, {a_i})`)
// Only plans and descriptors live here; the attention is attn.cu's kernel.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "common.cuh"

namespace mosaic {
namespace {

inline size_t align256(size_t x) { return (x + 255) & ~size_t(255); }

// ---- chunked prefill: chunk c of sequence s is a view of its own -- q rows [c C, min(L, (c+1) C))
// of the sequence against keys [0, that end): the bottom-right alignment of reading N2-1, so the
// rows see exactly the keys the plain prefill shows them.  One block: chunks per sequence, their
// exclusive scan, one descriptor per chunk, empty descriptors in the unused tail.
__global__ void __launch_bounds__(1024) chunk_plan_kernel(const int64_t* __restrict__ cu_seqlens,
                                                          int n_seqs, int q_chunk, int64_t v_max,
                                                          SeqDesc* __restrict__ desc) {
    __shared__ int warp_tot[32];
    __shared__ int carry;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) carry = 0;
    __syncthreads();
    for (int s0 = 0; s0 < n_seqs; s0 += 1024) {
        const int s = s0 + tid;
        int64_t t0 = 0, L = 0;
        if (s < n_seqs) {
            t0 = cu_seqlens[s];
            L = cu_seqlens[s + 1] - t0;
        }
        const int nc = (int)((L + q_chunk - 1) / q_chunk);
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
        const int first = before + x - nc;
        for (int c = 0; c < nc; ++c) {
            const int64_t r0 = (int64_t)c * q_chunk;
            const int64_t r1 = min(L, r0 + q_chunk);
            desc[first + c] = SeqDesc{t0 + r0, t0, (int32_t)(r1 - r0), (int32_t)r1};
        }
        __syncthreads();
        if (tid == 1023) carry = before + x;
        __syncthreads();
    }
    for (int64_t v = carry + tid; v < v_max; v += 1024) desc[v] = SeqDesc{0, 0, 0, 0};
}

struct ChunkWs {
    SeqDesc* desc;
    void* attn_ws;
    size_t attn_ws_bytes, total;
    int64_t v_max;
};
ChunkWs carve_chunked(void* base, int32_t n_seqs, int64_t total_tokens, int32_t q_chunk, int32_t Hq,
                      int32_t Hkv, int32_t D) {
    ChunkWs w{};
    w.v_max = total_tokens / q_chunk + n_seqs;
    char* p = static_cast<char*>(base);
    size_t off = 0;
    w.desc = reinterpret_cast<SeqDesc*>(p + off);
    off += align256((size_t)w.v_max * sizeof(SeqDesc));
    w.attn_ws_bytes = mosaic_agg_prefill_attn_workspace_bytes(
        (int32_t)(w.v_max < (1ll << 31) - 1 ? w.v_max : (1ll << 31) - 1), total_tokens, Hq, Hkv, D);
    w.attn_ws = p + off;
    off += align256(w.attn_ws_bytes);
    w.total = off;
    return w;
}

}  // namespace
}  // namespace mosaic

using namespace mosaic;

extern "C" size_t mosaic_agg_prefill_attn_chunked_workspace_bytes(int32_t n_seqs,
                                                                  int64_t total_tokens,
                                                                  int32_t q_chunk, int32_t Hq,
                                                                  int32_t Hkv, int32_t D) {
    if (n_seqs < 0 || total_tokens < 0 || q_chunk < 1) return 0;
    return carve_chunked(nullptr, n_seqs, total_tokens, q_chunk, Hq, Hkv, D).total;
}

extern "C" mosaic_status_t mosaic_agg_prefill_attn_chunked(
    const void* q, const void* k, const void* v, const int64_t* cu_seqlens, int32_t n_seqs,
    int64_t total_tokens, int32_t max_seqlen, int32_t Hq, int32_t Hkv, int32_t D,
    float softmax_scale, int32_t q_chunk, void* o, float* lse, void* workspace,
    size_t workspace_bytes, void* cuda_stream) {
    if (n_seqs < 0 || total_tokens < 0 || total_tokens >= (1ll << 31) || max_seqlen < 0 ||
        q_chunk < 1 || Hq < 1 || Hkv < 1 || Hq % Hkv != 0 || !isfinite(softmax_scale))
        return MOSAIC_ERR_INVALID_ARG;
    if (D != 64 && D != 128) return MOSAIC_ERR_UNSUPPORTED;
    if (n_seqs == 0 || total_tokens == 0) return MOSAIC_OK;
    if (!cu_seqlens || !workspace || !aligned16(workspace)) return MOSAIC_ERR_INVALID_ARG;
    ChunkWs w = carve_chunked(workspace, n_seqs, total_tokens, q_chunk, Hq, Hkv, D);
    if (workspace_bytes < w.total) return MOSAIC_ERR_WORKSPACE_TOO_SMALL;
    if (w.v_max >= (1ll << 31) - 1) return MOSAIC_ERR_UNSUPPORTED;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    chunk_plan_kernel<<<1, 1024, 0, s>>>(cu_seqlens, n_seqs, q_chunk, w.v_max, w.desc);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());
    return attn_impl(q, k, v, nullptr, nullptr, w.desc, (int32_t)w.v_max, total_tokens, total_tokens,
                     q_chunk < max_seqlen ? q_chunk : max_seqlen, Hq, Hkv, D, softmax_scale,
                     /*causal=*/1, o, lse, w.attn_ws, w.attn_ws_bytes, cuda_stream);
}

extern "C" size_t mosaic_agg_prefill_attn_shared_prefix_workspace_bytes(int32_t n_seqs,
                                                                        int64_t total_tokens,
                                                                        int32_t Hq, int32_t Hkv,
                                                                        int32_t D) {
    return mosaic_agg_prefill_attn_workspace_bytes(n_seqs, total_tokens, Hq, Hkv, D);
}

// One launch of the attention kernel: a work unit's KV tiles are the shared block's tiles (its own
// pair of tensor maps, the last tile padded to 128 keys and the padding masked) followed by the
// sequence's own; with the offset grown by the padded prefix length every role of the kernel sees
// an ordinary bottom-right causal problem.  The block's K / V (a few MB) stay in L2: they are
// read from HBM once for the whole batch.  (The first version ran the own keys and the shared block
// as two passes -- the second as ONE non-causal view of all packed q rows -- and merged them with
// mosaic_lse_merge: two more passes over O and Q read twice; 1 097 against 1 177 TFLOP/s on
// bench.py's shared_prefix leg.)
extern "C" mosaic_status_t mosaic_agg_prefill_attn_shared_prefix(
    const void* q, const void* k_prefix, const void* v_prefix, int32_t prefix_len, const void* k,
    const void* v, const int64_t* cu_seqlens, int32_t n_seqs, int64_t total_tokens,
    int32_t max_seqlen, int32_t Hq, int32_t Hkv, int32_t D, float softmax_scale, void* o,
    float* lse, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    if (prefix_len < 0) return MOSAIC_ERR_INVALID_ARG;
    if (prefix_len > 0 && n_seqs > 0 && total_tokens > 0 &&
        (!k_prefix || !v_prefix || !aligned16(k_prefix) || !aligned16(v_prefix)))
        return MOSAIC_ERR_INVALID_ARG;
    return attn_impl(q, k, v, cu_seqlens, cu_seqlens, nullptr, n_seqs, total_tokens, total_tokens,
                     max_seqlen, Hq, Hkv, D, softmax_scale, /*causal=*/1, o, lse, workspace,
                     workspace_bytes, cuda_stream, k_prefix, v_prefix, prefix_len);
}
