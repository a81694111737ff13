// attn.cu -- step 2 of the confidence-gated aggregator stage: the aggregator's prefill attention
// over the survivors' packed contexts ("process the combined output or reasoning
// traces of its experts"; math fixed by BASELINE.json north_star: variable-length causal
// grouped-query attention, bf16 O + fp32 row logsumexp).
//
// A5  schedule_kernel : (sequence, q tile) work items, longest (most KV tiles) first.
// A1-A4 attn_fwd      : tcgen05 / TMEM / TMA flash-attention forward, one q tile of 128 rows per
//                       work item and q head; S = Q K^T and O += P V on the 5th-gen tensor cores
//                       with fp32 accumulators in tensor memory, K/V tiles staged by TMA with the
//                       128-byte swizzle, online softmax with one thread per query row.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "common.cuh"
#include "ptx.cuh"

namespace mosaic {
namespace {

constexpr int BM = 128;  // query rows per tile  (UMMA M)
constexpr int BN = 128;  // key rows per tile    (UMMA N of S, UMMA K of PV)
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

// ------------------------------------------------------------------------------- A5: schedule
struct SchedHeader {
    int n_items;  // number of (sequence, q tile) entries
    int pad[3];
};

struct Workspace {
    SchedHeader* header;
    int* cnt;     // [levels]  sequences with exactly c+1 q tiles -> sequences with more than c
    int* start;   // [levels]  first entry of level c (levels in descending order)
    int* cursor;  // [levels]
    int2* items;  // [capacity] (sequence, q tile)
    size_t zero_bytes;  // prefix that must be zeroed before schedule_kernel
    size_t total_bytes;
};

inline Workspace carve(void* base, int32_t n_seqs, int64_t total_tokens) {
    Workspace w;
    const size_t levels = (size_t)(total_tokens / BM) + 2;
    const size_t cap = (size_t)(total_tokens / BM) + (size_t)n_seqs + 1;
    char* p = static_cast<char*>(base);
    size_t off = 0;
    w.header = reinterpret_cast<SchedHeader*>(p + off);
    off += 64;
    w.cnt = reinterpret_cast<int*>(p + off);
    off += levels * sizeof(int);
    w.cursor = reinterpret_cast<int*>(p + off);
    off += levels * sizeof(int);
    w.zero_bytes = off;
    w.start = reinterpret_cast<int*>(p + off);
    off += levels * sizeof(int);
    off = (off + 15) & ~size_t(15);
    w.items = reinterpret_cast<int2*>(p + off);
    off += cap * sizeof(int2);
    w.total_bytes = (off + 255) & ~size_t(255);
    return w;
}

// Work items in descending cost order.  The cost of (sequence s, q tile c) is its number of KV
// tiles, c + 1, so "longest first" is "descending c": level c holds one entry for every sequence
// with more than c tiles.  Counting sort over levels; order inside a level is arbitrary (the
// results do not depend on the schedule).  One block.
__global__ void __launch_bounds__(1024) schedule_kernel(const int64_t* __restrict__ cu_seqlens,
                                                        int n_seqs, int levels, SchedHeader* header,
                                                        int* cnt, int* start, int* cursor,
                                                        int2* items) {
    for (int s = threadIdx.x; s < n_seqs; s += blockDim.x) {
        const int64_t L = cu_seqlens[s + 1] - cu_seqlens[s];
        const int nt = (int)((L + BM - 1) / BM);
        if (nt > 0) atomicAdd(&cnt[min(nt, levels) - 1], 1);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        // cnt[c] <- number of sequences with more than c tiles (suffix sum)
        int run = 0;
        for (int c = levels - 1; c >= 0; --c) {
            run += cnt[c];
            cnt[c] = run;
        }
        int pos = 0;
        for (int c = levels - 1; c >= 0; --c) {
            start[c] = pos;
            pos += cnt[c];
        }
        header->n_items = pos;
    }
    __syncthreads();
    for (int s = threadIdx.x; s < n_seqs; s += blockDim.x) {
        const int64_t L = cu_seqlens[s + 1] - cu_seqlens[s];
        const int nt = min((int)((L + BM - 1) / BM), levels);
        for (int c = 0; c < nt; ++c) {
            const int pos = start[c] + atomicAdd(&cursor[c], 1);
            items[pos] = make_int2(s, c);
        }
    }
}

// ------------------------------------------------------------------------------ A1-A4: forward
struct AttnParams {
    const int64_t* cu_seqlens;
    const int2* items;
    const SchedHeader* header;
    __nv_bfloat16* o;
    float* lse;
    int64_t T;
    int Hq, Hkv;
    float scale_log2;  // softmax_scale * log2(e)
};

template <int D>
struct SmemLayout {
    static constexpr int kTileBytes = BM * D * 2;        // one [128, D] bf16 tile
    static constexpr int kBlockBytes = BM * 128;         // one [128 rows, 64 cols] swizzled block
    static constexpr int kQ = 0;
    static constexpr int kK = kTileBytes;
    static constexpr int kV = 2 * kTileBytes;
    static constexpr int kBars = 3 * kTileBytes;         // 4 mbarriers + tmem base
    static constexpr int kTotal = kBars + 64;
    static constexpr int kDynamic = kTotal + 1024;       // slack for the 1024-byte alignment
};

template <int D>
__global__ void __launch_bounds__(128) attn_fwd(const __grid_constant__ CUtensorMap tm_q,
                                                const __grid_constant__ CUtensorMap tm_k,
                                                const __grid_constant__ CUtensorMap tm_v,
                                                const AttnParams p) {
    using SL = SmemLayout<D>;
    constexpr int kTmemCols = 256;          // S/P: columns [0,128), O: columns [128, 128 + D)
    constexpr uint32_t kIdescS = ptx::umma_idesc_bf16(BM, BN, false, false);
    constexpr uint32_t kIdescPV = ptx::umma_idesc_bf16(BM, D, false, true);

    const int item = blockIdx.x / p.Hq;
    if (item >= p.header->n_items) return;
    const int h = blockIdx.x - item * p.Hq;
    const int g = h / (p.Hq / p.Hkv);
    const int2 it = p.items[item];
    const int seq = it.x, mt = it.y;
    const int64_t t0 = p.cu_seqlens[seq];
    const int L = (int)(p.cu_seqlens[seq + 1] - t0);
    const int row0 = mt * BM;

    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem = smem_raw + (smem_base - ptx::smem_u32(smem_raw));
    const uint32_t sQ = smem_base + SL::kQ, sK = smem_base + SL::kK, sV = smem_base + SL::kV;
    const uint32_t bar_q = smem_base + SL::kBars, bar_kv = bar_q + 8, bar_s = bar_q + 16,
                   bar_o = bar_q + 24;
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + SL::kBars + 32);

    const int tid = threadIdx.x, warp = tid >> 5;

    if (tid == 0) {
        ptx::prefetch_tensormap(&tm_q);
        ptx::prefetch_tensormap(&tm_k);
        ptx::prefetch_tensormap(&tm_v);
        ptx::mbar_init(bar_q, 1);
        ptx::mbar_init(bar_kv, 1);
        ptx::mbar_init(bar_s, 1);
        ptx::mbar_init(bar_o, 1);
        ptx::fence_barrier_init();
    }
    if (warp == 0) {
        ptx::tmem_alloc<kTmemCols>(ptx::smem_u32(const_cast<uint32_t*>(tmem_slot)));
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t lane_off = (uint32_t)(warp * 32) << 16;
    const uint32_t tS = tmem, tP = tmem, tO = tmem + 128;

    if (tid == 0) {
        ptx::mbar_arrive_expect_tx(bar_q, SL::kTileBytes);
#pragma unroll
        for (int c = 0; c < D / 64; ++c)
            ptx::tma_load_3d(sQ + c * SL::kBlockBytes, &tm_q, bar_q, c * 64, h, (int)(t0 + row0));
    }

    const int row = tid;  // this thread's TMEM lane == query row inside the tile
    float m_run = -INFINITY, l_run = 0.f;
    const int n_kv = mt + 1;

    for (int j = 0; j < n_kv; ++j) {
        const uint32_t ph = j & 1;
        if (tid == 0) {
            ptx::mbar_arrive_expect_tx(bar_kv, 2 * SL::kTileBytes);
#pragma unroll
            for (int c = 0; c < D / 64; ++c) {
                ptx::tma_load_3d(sK + c * SL::kBlockBytes, &tm_k, bar_kv, c * 64, g,
                                 (int)(t0 + j * BN));
                ptx::tma_load_3d(sV + c * SL::kBlockBytes, &tm_v, bar_kv, c * 64, g,
                                 (int)(t0 + j * BN));
            }
            if (j == 0) ptx::mbar_wait(bar_q, 0);
            ptx::mbar_wait(bar_kv, ph);
            ptx::tc_fence_after();
            // S = Q K^T : both operands K-major (D contiguous), 128-byte swizzle
#pragma unroll
            for (int kk = 0; kk < D / 16; ++kk) {
                const uint32_t off = (kk / 4) * SL::kBlockBytes + (kk % 4) * 32;
                ptx::umma_ss(tS, ptx::umma_smem_desc_sw128(sQ + off, 16, 1024),
                             ptx::umma_smem_desc_sw128(sK + off, 16, 1024), kIdescS, kk > 0);
            }
            ptx::umma_commit(bar_s);
        }
        ptx::mbar_wait(bar_s, ph);
        ptx::tc_fence_after();

        // ---- A2: online softmax, one thread per row -------------------------------------------
        const bool diag = (j == mt);
        float mx = -INFINITY;
#pragma unroll
        for (int c = 0; c < BN / 32; ++c) {
            uint32_t r[32];
            ptx::tmem_ld32(tS + lane_off + c * 32, r);
            ptx::tmem_wait_ld();
#pragma unroll
            for (int i = 0; i < 32; ++i) {
                float t = __uint_as_float(r[i]) * p.scale_log2;
                if (diag && (c * 32 + i > row)) t = -INFINITY;
                mx = fmaxf(mx, t);
            }
        }
        const float m_new = fmaxf(m_run, mx);
        const float alpha = exp2f(m_run - m_new);
        float l_sum = 0.f;
#pragma unroll
        for (int c = 0; c < BN / 32; ++c) {
            uint32_t r[32];
            ptx::tmem_ld32(tS + lane_off + c * 32, r);
            ptx::tmem_wait_ld();
            uint32_t pk[16];
#pragma unroll
            for (int i = 0; i < 32; i += 2) {
                float t0f = __uint_as_float(r[i]) * p.scale_log2;
                float t1f = __uint_as_float(r[i + 1]) * p.scale_log2;
                float p0 = exp2f(t0f - m_new), p1 = exp2f(t1f - m_new);
                if (diag && (c * 32 + i > row)) p0 = 0.f;
                if (diag && (c * 32 + i + 1 > row)) p1 = 0.f;
                l_sum += p0 + p1;
                __nv_bfloat162 hh = __floats2bfloat162_rn(p0, p1);
                pk[i / 2] = *reinterpret_cast<uint32_t*>(&hh);
            }
            ptx::tmem_st16(tP + lane_off + c * 16, pk);
        }
        if (j > 0) {
#pragma unroll
            for (int c = 0; c < D / 32; ++c) {
                uint32_t r[32];
                ptx::tmem_ld32(tO + lane_off + c * 32, r);
                ptx::tmem_wait_ld();
#pragma unroll
                for (int i = 0; i < 32; ++i) r[i] = __float_as_uint(__uint_as_float(r[i]) * alpha);
                ptx::tmem_st32(tO + lane_off + c * 32, r);
            }
        }
        l_run = l_run * alpha + l_sum;
        m_run = m_new;
        ptx::tmem_wait_st();
        ptx::tc_fence_before();
        __syncthreads();

        // ---- A3: O += P V : A = P from tensor memory, B = V (MN-major: D contiguous) ----------
        if (tid == 0) {
            ptx::tc_fence_after();
#pragma unroll
            for (int kk = 0; kk < BN / 16; ++kk) {
                ptx::umma_ts(tO, tP + kk * 8,
                             ptx::umma_smem_desc_sw128(sV + kk * 2048, SL::kBlockBytes, 1024),
                             kIdescPV, (j > 0 || kk > 0) ? 1u : 0u);
            }
            ptx::umma_commit(bar_o);
        }
        ptx::mbar_wait(bar_o, ph);
        ptx::tc_fence_after();
    }

    // ---- epilogue: normalise, round to bf16, store; A4: logsumexp ---------------------------------
    const int row_g = row0 + row;
    const float inv_l = 1.f / l_run;
    __nv_bfloat16* orow = p.o + ((t0 + row_g) * p.Hq + h) * (int64_t)D;
#pragma unroll
    for (int c = 0; c < D / 32; ++c) {
        uint32_t r[32];
        ptx::tmem_ld32(tO + lane_off + c * 32, r);
        ptx::tmem_wait_ld();
        if (row_g < L) {
#pragma unroll
            for (int i = 0; i < 32; i += 8) {
                uint4 v;
                __nv_bfloat162 h0 = __floats2bfloat162_rn(__uint_as_float(r[i + 0]) * inv_l,
                                                          __uint_as_float(r[i + 1]) * inv_l);
                __nv_bfloat162 h1 = __floats2bfloat162_rn(__uint_as_float(r[i + 2]) * inv_l,
                                                          __uint_as_float(r[i + 3]) * inv_l);
                __nv_bfloat162 h2 = __floats2bfloat162_rn(__uint_as_float(r[i + 4]) * inv_l,
                                                          __uint_as_float(r[i + 5]) * inv_l);
                __nv_bfloat162 h3 = __floats2bfloat162_rn(__uint_as_float(r[i + 6]) * inv_l,
                                                          __uint_as_float(r[i + 7]) * inv_l);
                v.x = *reinterpret_cast<uint32_t*>(&h0);
                v.y = *reinterpret_cast<uint32_t*>(&h1);
                v.z = *reinterpret_cast<uint32_t*>(&h2);
                v.w = *reinterpret_cast<uint32_t*>(&h3);
                *reinterpret_cast<uint4*>(orow + c * 32 + i) = v;
            }
        }
    }
    if (row_g < L) p.lse[(int64_t)h * p.T + t0 + row_g] = (m_run + log2f(l_run)) * kLn2;

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 0) ptx::tmem_dealloc<kTmemCols>(tmem);
}

// ------------------------------------------------------------------------------------ host side
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                   const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                   const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = [] {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &qres) !=
                cudaSuccess ||
            qres != cudaDriverEntryPointSuccess)
            f = nullptr;
        return reinterpret_cast<EncodeTiledFn>(f);
    }();
    return fn;
}

// Tensor map over a packed [T, H, D] bf16 tensor; box = 64 columns (128 bytes, one swizzle row)
// x 1 head x `rows` tokens.  Rows past T are zero-filled.
bool make_tensor_map(CUtensorMap* map, const void* base, int64_t T, int H, int D, int rows) {
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return false;
    cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)H, (cuuint64_t)T};
    cuuint64_t strides[2] = {(cuuint64_t)D * 2, (cuuint64_t)H * D * 2};
    cuuint32_t box[3] = {64, 1, (cuuint32_t)rows};
    cuuint32_t estr[3] = {1, 1, 1};
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides,
               box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
               CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int D>
mosaic_status_t launch_attn(const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv,
                            const AttnParams& p, int grid, cudaStream_t s) {
    using SL = SmemLayout<D>;
    static bool configured = false;
    if (!configured) {
        MOSAIC_CUDA_TRY(cudaFuncSetAttribute(attn_fwd<D>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             SL::kDynamic));
        configured = true;
    }
    attn_fwd<D><<<grid, 128, SL::kDynamic, s>>>(tq, tk, tv, p);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());
    return MOSAIC_OK;
}

}  // namespace
}  // namespace mosaic

using namespace mosaic;

extern "C" size_t mosaic_agg_prefill_attn_workspace_bytes(int32_t n_seqs, int64_t total_tokens,
                                                          int32_t Hq, int32_t Hkv, int32_t D) {
    (void)Hq;
    (void)Hkv;
    (void)D;
    if (n_seqs < 0 || total_tokens < 0) return 0;
    return carve(nullptr, n_seqs, total_tokens).total_bytes;
}

extern "C" mosaic_status_t mosaic_agg_prefill_attn(const void* q, const void* k, const void* v,
                                                   const int64_t* cu_seqlens, int32_t n_seqs,
                                                   int64_t total_tokens, int32_t max_seqlen,
                                                   int32_t Hq, int32_t Hkv, int32_t D,
                                                   float softmax_scale, void* o, float* lse,
                                                   void* workspace, size_t workspace_bytes,
                                                   void* cuda_stream) {
    if (n_seqs < 0 || total_tokens < 0 || total_tokens >= (1ll << 31) || max_seqlen < 0 ||
        Hq < 1 || Hkv < 1 || Hq % Hkv != 0 || !isfinite(softmax_scale))
        return MOSAIC_ERR_INVALID_ARG;
    if (D != 64 && D != 128) return MOSAIC_ERR_UNSUPPORTED;
    if (n_seqs == 0 || total_tokens == 0) return MOSAIC_OK;
    if (!q || !k || !v || !o || !lse || !cu_seqlens || !workspace || !aligned16(q) ||
        !aligned16(k) || !aligned16(v) || !aligned16(o) || !aligned16(workspace))
        return MOSAIC_ERR_INVALID_ARG;
    // TODO(negative scale): the row max is taken after scaling, so any finite scale is handled.
    Workspace w = carve(workspace, n_seqs, total_tokens);
    if (workspace_bytes < w.total_bytes) return MOSAIC_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);

    CUtensorMap tq, tk, tv;
    if (!make_tensor_map(&tq, q, total_tokens, Hq, D, BM) ||
        !make_tensor_map(&tk, k, total_tokens, Hkv, D, BN) ||
        !make_tensor_map(&tv, v, total_tokens, Hkv, D, BN))
        return MOSAIC_ERR_CUDA;

    const int levels = (int)(total_tokens / BM) + 2;
    MOSAIC_CUDA_TRY(cudaMemsetAsync(workspace, 0, w.zero_bytes, s));
    schedule_kernel<<<1, 1024, 0, s>>>(cu_seqlens, n_seqs, levels, w.header, w.cnt, w.start,
                                       w.cursor, w.items);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());

    AttnParams p{};
    p.cu_seqlens = cu_seqlens;
    p.items = w.items;
    p.header = w.header;
    p.o = static_cast<__nv_bfloat16*>(o);
    p.lse = lse;
    p.T = total_tokens;
    p.Hq = Hq;
    p.Hkv = Hkv;
    p.scale_log2 = softmax_scale * kLog2e;
    const int64_t max_items = total_tokens / BM + n_seqs;
    const int64_t grid = max_items * Hq;
    if (grid >= (1ll << 31)) return MOSAIC_ERR_UNSUPPORTED;
    return D == 64 ? launch_attn<64>(tq, tk, tv, p, (int)grid, s)
                   : launch_attn<128>(tq, tk, tv, p, (int)grid, s);
}
