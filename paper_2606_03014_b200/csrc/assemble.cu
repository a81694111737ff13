// assemble.cu -- SURVEY.md section 8(f) N1, the step between G5 and A1: the survivors' aggregator
// contexts as one packed token batch.  The aggregator "process[es] the combined output or
// reasoning traces of its experts" (Alg. 1 `Aggregator(q, {a_i})`); the
// paper fixes neither template nor order, reading N1-1 does: the context of survivor j
// (question q = survivor_idx[j]) is prompt(q) ++ trace(q, 0) ++ ... ++ trace(q, E-1).
//
// HBM-bound ragged gather: 4 bytes read and 8 written per token (token id, position id).  Block
// (j, c) copies tokens [8192 c, 8192 c + 8192) of sequence j; a thread takes 4 consecutive tokens that
// are 16-byte aligned in the output, so every full group is one 128-bit store per output array.
#include <cuda_runtime.h>
#include <stdint.h>

#include "common.cuh"

namespace mosaic {
namespace {

constexpr int kAsmThreads = 256;
constexpr int kAsmChunk = 8192;  // tokens per block

struct AssembleArgs {
    const int32_t* survivor_idx;
    const int64_t* cu_seqlens;
    const int32_t* prompt_tokens;
    const int64_t* prompt_off;
    const int32_t* trace_tokens;
    const int64_t* trace_off;
    int32_t* input_ids;
    int32_t* position_ids;
    int32_t* n_mismatch;
    int E;
};

__global__ void __launch_bounds__(kAsmThreads) assemble_kernel(const AssembleArgs p) {
    // Segment 0 = prompt, 1 + e = trace e.  cum[g] = tokens of the segments before g; src[g] =
    // address of segment g's first token minus cum[g], so token i of the sequence is src[g][i].
    __shared__ int64_t cum[MOSAIC_MAX_EXPERTS + 2];
    __shared__ const int32_t* src[MOSAIC_MAX_EXPERTS + 1];
    const int j = blockIdx.x;
    const int64_t t0 = p.cu_seqlens[j];
    const int64_t L = p.cu_seqlens[j + 1] - t0;
    const int64_t i0 = (int64_t)blockIdx.y * kAsmChunk;
    if (i0 >= L) return;
    const int nseg = p.E + 1;  // <= MOSAIC_MAX_EXPERTS + 1 = 33
    if (threadIdx.x < 32) {
        // one lane per segment (lane 0 also takes segment 32 when E = 32): the offset loads are one
        // round trip, the prefix a full 32-lane warp scan
        const int g = threadIdx.x;
        const int64_t q = p.survivor_idx[j];
        auto bounds = [&](int seg, int64_t& first, int64_t& len) {
            const int64_t* off = seg == 0 ? p.prompt_off + q : p.trace_off + q * p.E + (seg - 1);
            first = off[0];
            len = off[1] - first;
        };
        int64_t first = 0, len = 0, first32 = 0, len32 = 0;
        if (g < nseg) bounds(g, first, len);
        if (g == 0 && nseg == 33) bounds(32, first32, len32);
        int64_t incl = len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int64_t y = __shfl_up_sync(0xffffffffu, incl, o);
            if (g >= o) incl += y;
        }
        if (g < nseg) {
            cum[g] = incl - len;
            src[g] = (g == 0 ? p.prompt_tokens : p.trace_tokens) + first - (incl - len);
        }
        const int64_t sum32 = __shfl_sync(0xffffffffu, incl, 31);  // segments 0..31 (absent ones are 0)
        if (g == 0) {
            int64_t total = sum32;
            if (nseg == 33) {
                cum[32] = sum32;
                src[32] = p.trace_tokens + first32 - sum32;
                total += len32;
            }
            cum[nseg] = total;
            if (blockIdx.y == 0 && total != L && p.n_mismatch) atomicAdd(p.n_mismatch, 1);
        }
    }
    __syncthreads();
    const int64_t i1 = min(L, i0 + kAsmChunk);
    const int64_t total = cum[nseg];
    auto token = [&](int64_t i) -> int32_t {
        if (i >= total) return -1;  // past the sources of a sequence whose length does not match them
        int g = 0;
        for (int k = 1; k < nseg; ++k) g += (i >= cum[k]) ? 1 : 0;  // (empty segments are skipped)
        return __ldg(src[g] + i);
    };
    // Groups of 4 tokens aligned to 16 bytes in the OUTPUT arrays (the sequence starts anywhere):
    // group k of this block covers output elements [base + 4 k, base + 4 k + 4); a full group is one
    // 16-byte store per array, the ragged first and last groups are written element by element.
    // (Staging the tokens through shared memory for fully coalesced loads was measured slower:
    //  153 against 132 us on the bench workload.)
    const int64_t base = (t0 + i0) & ~int64_t(3);
    const int64_t n_groups = (t0 + i1 - base + 3) >> 2;
#pragma unroll 2
    for (int64_t k = threadIdx.x; k < n_groups; k += kAsmThreads) {
        const int64_t o = base + 4 * k;  // output element of the group's first token
        const int64_t i = o - t0;        // its index in the sequence (may be < i0 in the first group)
        if (i >= i0 && i + 4 <= i1) {
            int4 tk, ps;
            int g = 0;
            for (int kk = 1; kk < nseg; ++kk) g += (i >= cum[kk]) ? 1 : 0;
            if (i + 4 <= cum[g + 1]) {  // the usual case: all four in one segment, one search
                const int32_t* from = src[g] + i;
                tk.x = __ldg(from);
                tk.y = __ldg(from + 1);
                tk.z = __ldg(from + 2);
                tk.w = __ldg(from + 3);
            } else {
                tk.x = token(i);
                tk.y = token(i + 1);
                tk.z = token(i + 2);
                tk.w = token(i + 3);
            }
            ps = make_int4((int)i, (int)i + 1, (int)i + 2, (int)i + 3);
            __stcs(reinterpret_cast<int4*>(p.input_ids + o), tk);
            __stcs(reinterpret_cast<int4*>(p.position_ids + o), ps);
        } else {
            for (int u = 0; u < 4; ++u) {
                const int64_t iu = i + u;
                if (iu >= i0 && iu < i1) {
                    __stcs(p.input_ids + o + u, token(iu));
                    __stcs(p.position_ids + o + u, (int32_t)iu);
                }
            }
        }
    }
}

}  // namespace
}  // namespace mosaic

using namespace mosaic;

extern "C" mosaic_status_t mosaic_assemble_context(
    const int32_t* survivor_idx, const int64_t* cu_seqlens, int32_t n_survivors,
    int32_t max_seqlen, const int32_t* prompt_tokens, const int64_t* prompt_off,
    const int32_t* trace_tokens, const int64_t* trace_off, int32_t E, int32_t* input_ids,
    int32_t* position_ids, int32_t* n_mismatch, void* cuda_stream) {
    if (n_survivors < 0 || max_seqlen < 0 || E < 1 || E > MOSAIC_MAX_EXPERTS)
        return MOSAIC_ERR_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    if (n_mismatch) MOSAIC_CUDA_TRY(cudaMemsetAsync(n_mismatch, 0, sizeof(int32_t), s));
    if (n_survivors == 0 || max_seqlen == 0) return MOSAIC_OK;
    if (!survivor_idx || !cu_seqlens || !prompt_tokens || !prompt_off || !trace_tokens ||
        !trace_off || !input_ids || !position_ids || !aligned16(input_ids) ||
        !aligned16(position_ids))
        return MOSAIC_ERR_INVALID_ARG;
    const int64_t chunks = ((int64_t)max_seqlen + kAsmChunk - 1) / kAsmChunk;
    if (chunks > 65535) return MOSAIC_ERR_UNSUPPORTED;  // sequences of more than 536 M tokens
    AssembleArgs a{survivor_idx, cu_seqlens, prompt_tokens, prompt_off, trace_tokens, trace_off,
                   input_ids,    position_ids, n_mismatch,  E};
    assemble_kernel<<<dim3((unsigned)n_survivors, (unsigned)chunks), kAsmThreads, 0, s>>>(a);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());
    return MOSAIC_OK;
}
