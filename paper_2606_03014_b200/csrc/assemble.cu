// assemble.cu -- SURVEY.md section 8(f) N1, the step between G5 and A1: the survivors' aggregator
// contexts as one packed token batch.  The aggregator "process[es] the combined output or
// reasoning traces of its experts" (Alg. 1 `Aggregator(q, {a_i})`); the
// paper fixes neither template nor order, reading N1-1 does: the context of survivor j
// (question q = survivor_idx[j]) is prompt(q) ++ trace(q, 0) ++ ... ++ trace(q, E-1).
//
// HBM-bound ragged gather: 4 bytes read and 8 written per token (token id, position id).  Block
// (j, c) copies tokens [2048 c, 2048 c + 2048) of sequence j; consecutive threads take consecutive
// tokens, so loads and stores are coalesced inside every segment.
#include <cuda_runtime.h>
#include <stdint.h>

#include "common.cuh"

namespace mosaic {
namespace {

constexpr int kAsmThreads = 256;
constexpr int kAsmChunk = 2048;  // tokens per block

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
    // cum[g] = tokens of the segments before g (segment 0 = prompt, 1 + e = trace e); src[g] = where
    // segment g starts in its token array
    __shared__ int64_t cum[MOSAIC_MAX_EXPERTS + 2];
    __shared__ int64_t src[MOSAIC_MAX_EXPERTS + 1];
    const int j = blockIdx.x;
    const int64_t t0 = p.cu_seqlens[j];
    const int64_t L = p.cu_seqlens[j + 1] - t0;
    const int64_t i0 = (int64_t)blockIdx.y * kAsmChunk;
    if (i0 >= L) return;
    const int nseg = p.E + 1;
    if (threadIdx.x == 0) {
        const int64_t q = p.survivor_idx[j];
        int64_t run = 0;
        for (int g = 0; g < nseg; ++g) {
            const int64_t* off = g == 0 ? p.prompt_off + q : p.trace_off + q * p.E + (g - 1);
            cum[g] = run;
            src[g] = off[0];
            run += off[1] - off[0];
        }
        cum[nseg] = run;
        if (blockIdx.y == 0 && run != L && p.n_mismatch) atomicAdd(p.n_mismatch, 1);
    }
    __syncthreads();
    const int64_t i1 = min(L, i0 + kAsmChunk);
    for (int64_t i = i0 + threadIdx.x; i < i1; i += kAsmThreads) {
        int32_t tok = -1;  // past the sources of a sequence whose length does not match them
        if (i < cum[nseg]) {
            int g = 0;
            while (i >= cum[g + 1]) ++g;  // <= E steps; empty segments are skipped
            const int64_t at = src[g] + (i - cum[g]);
            tok = g == 0 ? __ldg(p.prompt_tokens + at) : __ldg(p.trace_tokens + at);
        }
        __stcs(p.input_ids + t0 + i, tok);
        __stcs(p.position_ids + t0 + i, (int32_t)i);
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
        !trace_off || !input_ids || !position_ids)
        return MOSAIC_ERR_INVALID_ARG;
    const int64_t chunks = ((int64_t)max_seqlen + kAsmChunk - 1) / kAsmChunk;
    if (chunks > 65535) return MOSAIC_ERR_UNSUPPORTED;  // sequences of more than 134 M tokens
    AssembleArgs a{survivor_idx, cu_seqlens, prompt_tokens, prompt_off, trace_tokens, trace_off,
                   input_ids,    position_ids, n_mismatch,  E};
    assemble_kernel<<<dim3((unsigned)n_survivors, (unsigned)chunks), kAsmThreads, 0, s>>>(a);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());
    return MOSAIC_OK;
}
