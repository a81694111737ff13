// compact_static.cu -- mosaic_compact_static: mosaic_compact (G4-G5, the stream compaction of the
// surviving questions into a ragged batch with cu_seqlens; Alg. 1, BASELINE.json
// north_star) for callers that cannot allocate device memory: code under CUDA graph capture, tight
// serving loops, harnesses that forbid cudaMalloc.  The kernel is the one mosaic_compact launches
// (compact_kernel.cuh, kSrcBypass); its scan state -- the tile ticket and one state per tile -- lives
// in a file-scope device array of this library instead of a caller workspace.
//
// The array: kStaticScratchBytes = 1 MiB, held by every GPU that loads the library until the process
// exits.  It bounds the call at MOSAIC_COMPACT_STATIC_MAX_Q questions.  Every call shares it, and it
// keeps the last call's contents: the zeroing kernel that precedes the scan kernel in every call
// (as in mosaic_compact, whose workspace is arbitrary on entry) clears what must start at zero.
// Two calls that overlap on the GPU (different streams, or two host threads) race on it.
//
// In host code the array's NAME is a host-side stand-in, not a device address: the address the
// kernels get is asked of the runtime once per device (cudaGetSymbolAddress, with that device
// current) and cached.  This file calls no cudaMalloc / cudaFree / allocating library routine.
#include <mutex>

#include "compact_kernel.cuh"

namespace mosaic {
namespace {

constexpr size_t kStaticScratchBytes = (size_t)1 << 20;
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

// Even with one state per smallest tile and no padding the maximum must fit (the launch uses
// 128-byte lines per state when they fit, which they do: at most Q / (4 kVoters) tiles beyond one wave).
static_assert(sizeof(ScanHeader) +
                      ((size_t)MOSAIC_COMPACT_STATIC_MAX_Q / kMinTileQuestions + 2) * sizeof(TileState) <=
                  kStaticScratchBytes,
              "static scratch holds the scan state of MOSAIC_COMPACT_STATIC_MAX_Q questions");

constexpr int kMaxDevices = 64;
constexpr int kLightBlocksStatic = kVoterWarps > 8 ? 2 : 3;  // as mosaic_compact

// Device address of g_static_scratch on the CURRENT device (asked once per device).
mosaic_status_t static_scratch(void** out) {
    static std::mutex mu;
    static void* addr[kMaxDevices] = {};
    int dev = -1;
    MOSAIC_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return MOSAIC_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        void* p = nullptr;
        MOSAIC_CUDA_TRY(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) return MOSAIC_ERR_CUDA;
        addr[dev] = p;
    }
    *out = addr[dev];
    return MOSAIC_OK;
}

}  // namespace
}  // namespace mosaic

using namespace mosaic;

extern "C" mosaic_status_t mosaic_compact_static(const uint8_t* bypass, const int32_t* ctx_len,
                                                 int64_t Q, int32_t* survivor_idx,
                                                 int64_t* cu_seqlens, int32_t* n_survivors,
                                                 int64_t* total_tokens, int32_t* max_seqlen,
                                                 void* cuda_stream) {
    if (Q < 0 || !cu_seqlens || !n_survivors || !total_tokens || !max_seqlen)
        return MOSAIC_ERR_INVALID_ARG;
    if (Q > MOSAIC_COMPACT_STATIC_MAX_Q) return MOSAIC_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    if (Q == 0) {
        MOSAIC_CUDA_TRY(cudaMemsetAsync(cu_seqlens, 0, sizeof(int64_t), s));
        MOSAIC_CUDA_TRY(cudaMemsetAsync(n_survivors, 0, sizeof(int32_t), s));
        MOSAIC_CUDA_TRY(cudaMemsetAsync(total_tokens, 0, sizeof(int64_t), s));
        MOSAIC_CUDA_TRY(cudaMemsetAsync(max_seqlen, 0, sizeof(int32_t), s));
        return MOSAIC_OK;
    }
    if (!bypass || !ctx_len || !survivor_idx) return MOSAIC_ERR_INVALID_ARG;
    void* scratch = nullptr;
    mosaic_status_t st = static_scratch(&scratch);
    if (st != MOSAIC_OK) return st;
    GateArgs a{};
    a.bypass_in = bypass;
    a.ctx_len = ctx_len;
    a.Q = Q;
    a.E = 1;
    a.survivor_idx = survivor_idx;
    a.cu_seqlens = cu_seqlens;
    a.n_survivors = n_survivors;
    a.total_tokens = total_tokens;
    a.max_seqlen = max_seqlen;
    return launch<1, MOSAIC_CONF_VOTE, kSrcBypass, 4, kLightBlocksStatic>(a, kStaticScratchBytes,
                                                                         scratch, s);
}
