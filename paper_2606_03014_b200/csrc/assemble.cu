// assemble.cu -- SURVEY.md section 8(f) N1, the step between G5 and A1: the survivors' aggregator
// contexts as one packed token batch.  The aggregator "process[es] the combined output or
// reasoning traces of its experts" (Alg. 1 `Aggregator(q, {a_i})`); the
// paper fixes neither template nor order, reading N1-1 does: the context of survivor j
// (question q = survivor_idx[j]) is prompt(q) ++ trace(q, 0) ++ ... ++ trace(q, E-1).
//
// HBM-bound ragged gather: 4 bytes read and 8 written per token (token id, position id).  Block
// (j, c) copies tokens [8192 c, 8192 c + 8192) of sequence j.  The sources are 4-byte aligned runs of
// any length, so they are fetched by bulk copies (TMA, `cp.async.bulk`) of the 16-byte-aligned
// window around each run into a shared-memory ring -- the bytes in flight are the ring's, 32 KB
// per block, where the first version (four 4-byte loads per thread and 16-byte stores: 4.7 TB/s)
// was bound by the latency of what its registers could hold -- and written out lane-contiguous
// from a 128-byte boundary of the output (whole-line stores, conflict-free shared-memory reads).
#include <cuda_runtime.h>
#include <stdint.h>

#include "common.cuh"
#include "ptx.cuh"

namespace mosaic {
namespace {

constexpr int kAsmThreads = 256;
constexpr int kAsmChunk = 8192;   // tokens per block
constexpr int kAsmPiece = 2048;   // tokens per bulk copy
constexpr int kAsmStages = 4;     // bulk copies in flight per block (2-6 x 1-4 k tokens measure alike)
constexpr int kAsmMaxPieces = kAsmChunk / kAsmPiece + MOSAIC_MAX_EXPERTS + 1;  // (a segment boundary ends a piece)

struct AssembleSmem {
    alignas(128) uint8_t stage[kAsmStages][kAsmPiece * 4 + 32];  // the aligned window of a piece
    alignas(8) uint64_t full[kAsmStages];
    int64_t piece_i[kAsmMaxPieces];           // first token (index in the sequence)
    const int32_t* piece_src[kAsmMaxPieces];  // its address
    int piece_n[kAsmMaxPieces];               // tokens
    int n_pieces;
};

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
    __shared__ AssembleSmem sm;
    auto fetch = [&](int q) {  // piece q -> its stage of the ring
        const uintptr_t a = reinterpret_cast<uintptr_t>(sm.piece_src[q]);
        const uintptr_t lo = a & ~uintptr_t(15), hi = (a + 4u * (uintptr_t)sm.piece_n[q] + 15u) & ~uintptr_t(15);
        const uint32_t bar = ptx::smem_u32(&sm.full[q % kAsmStages]);
        ptx::mbar_arrive_expect_tx(bar, (uint32_t)(hi - lo));
        ptx::bulk_load_1d(ptx::smem_u32(sm.stage[q % kAsmStages]), reinterpret_cast<const void*>(lo),
                          (uint32_t)(hi - lo), bar);
    };
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
    const int64_t have = min(i1, total);  // tokens of the chunk that have a source: [i0, have)
    // The chunk's tokens come from PIECES: runs of at most kAsmPiece tokens inside one segment.
    // Thread 0 lists them and fetches each with one bulk copy (the 16-byte-aligned window around
    // the run: sources are 4-byte aligned) into a ring of kAsmStages buffers; all threads then move
    // a piece from shared memory to the two outputs.  The bytes in flight are the ring's, not the
    // registers': kAsmStages x 8 KB per block.
    if (threadIdx.x == 0) {
        int np = 0, g = 0;
        for (int64_t pos = i0; pos < have;) {
            while (cum[g + 1] <= pos) ++g;  // (empty segments are skipped)
            const int64_t n = min(min(have, cum[g + 1]), pos + kAsmPiece) - pos;
            sm.piece_i[np] = pos;
            sm.piece_n[np] = (int)n;
            sm.piece_src[np] = src[g] + pos;
            ++np;
            pos += n;
        }
        sm.n_pieces = np;
        for (int s = 0; s < kAsmStages; ++s) ptx::mbar_init(ptx::smem_u32(&sm.full[s]), 1);
        ptx::fence_barrier_init();
        for (int q = 0; q < np && q < kAsmStages; ++q) fetch(q);
    }
    __syncthreads();
    const int np = sm.n_pieces;
    for (int q = 0; q < np; ++q) {
        const int s = q % kAsmStages;
        ptx::mbar_wait(ptx::smem_u32(&sm.full[s]), (uint32_t)(q / kAsmStages) & 1u);
        const int64_t pi = sm.piece_i[q];
        const int n = sm.piece_n[q];
        const int32_t* st = reinterpret_cast<const int32_t*>(sm.stage[s]) +
                            ((reinterpret_cast<uintptr_t>(sm.piece_src[q]) & 15u) >> 2);
        // lane-contiguous, starting at a 128-byte boundary of the OUTPUT: a warp's stores are whole
        // lines, its shared-memory reads conflict-free
        const int64_t o0 = t0 + pi;
        const int first = (int)((o0 & ~int64_t(31)) - o0) + (int)threadIdx.x;  // may be < 0
#pragma unroll 4
        for (int k = first; k < n; k += kAsmThreads) {
            if (k >= 0) {
                __stcs(p.input_ids + o0 + k, st[k]);
                __stcs(p.position_ids + o0 + k, (int32_t)(pi + k));
            }
        }
        __syncthreads();  // the stage is free
        if (threadIdx.x == 0 && q + kAsmStages < np) fetch(q + kAsmStages);
    }
    // past the sources of a sequence whose length does not match them
    for (int64_t i = max(i0, total) + threadIdx.x; i < i1; i += kAsmThreads) {
        __stcs(p.input_ids + t0 + i, -1);
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
