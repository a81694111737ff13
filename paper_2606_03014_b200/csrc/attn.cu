// attn.cu -- step 2 of the confidence-gated aggregator stage: the aggregator's prefill attention
// over the survivors' packed contexts ("process the combined output or reasoning
// traces of its experts"; math fixed by BASELINE.json north_star: variable-length causal
// grouped-query attention, bf16 O + fp32 row logsumexp).
//
// A5    schedule_kernel : (sequence, 256-row q block) work items, longest (most KV tiles) first.
// A1-A4 attn_fwd        : persistent, warp-specialised tcgen05 / TMEM / TMA flash attention.
//   One CTA per SM works through (item, q head) pairs.  A q block is two 128-row tiles; for each
//   128-key tile j the tensor core computes S_t = Q_t K_j^T into tensor memory, a 128-thread
//   softmax group per tile (one thread per query row) turns S_t into P_t in place (bf16, same
//   TMEM columns), and O_t += P_t V_j accumulates in tensor memory.  While one tile is in
//   softmax the tensor core runs the other tile's MMAs.
//     warp 0      : TMA producer (Q tiles, K/V ring of kSlots 128-key tiles, 128-byte swizzle)
//     warp 1      : tcgen05.mma issuer (one elected thread)
//     warp 2      : TMEM allocation / release
//     warps 4-7   : softmax + epilogue of tile 0        warps 8-11 : ... of tile 1
//   The running row max is only moved (and O rescaled) when it grows by more than 2^8, so the
//   rescale of the accumulator is rare; the final 1/l normalisation makes the result exact.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <type_traits>

#include "common.cuh"
#include "ptx.cuh"

namespace mosaic {
namespace {

constexpr int BM = 128;       // query rows per tile  (UMMA M)
constexpr int BN = 128;       // key rows per tile    (UMMA N of S, UMMA K of PV)
constexpr int BQ = 2 * BM;    // query rows per work item (two tiles)
constexpr int kSlots = 4;     // K/V ring depth (tiles)
constexpr int kThreadsAttn = 384;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr float kRescaleThreshold = 8.0f;  // log2 units

// ------------------------------------------------------------------------------- A5: schedule
struct SchedHeader {
    int n_items;  // number of (sequence, q block) entries
    int pad[3];
};

struct Workspace {
    SchedHeader* header;
    int* cnt;     // [levels]  sequences with exactly c+1 q blocks -> sequences with more than c
    int* start;   // [levels]  first entry of level c (levels in descending order)
    int* cursor;  // [levels]
    int2* items;  // [capacity] (sequence, q block)
    size_t zero_bytes;  // prefix that must be zeroed before schedule_kernel
    size_t total_bytes;
};

inline Workspace carve(void* base, int32_t n_seqs, int64_t total_tokens) {
    Workspace w;
    const size_t levels = (size_t)(total_tokens / BQ) + 2;
    const size_t cap = (size_t)(total_tokens / BQ) + (size_t)n_seqs + 1;
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

// Work items in descending cost order.  The cost of (sequence s, q block c) is its number of KV
// tiles, ~2c + 2, so "longest first" is "descending c": level c holds one entry for every
// sequence with more than c blocks.  Counting sort over levels; order inside a level is arbitrary
// (the results do not depend on the schedule).  One block.
__global__ void __launch_bounds__(1024) schedule_kernel(const int64_t* __restrict__ cu_seqlens,
                                                        int n_seqs, int levels, SchedHeader* header,
                                                        int* cnt, int* start, int* cursor,
                                                        int2* items) {
    for (int s = threadIdx.x; s < n_seqs; s += blockDim.x) {
        const int64_t L = cu_seqlens[s + 1] - cu_seqlens[s];
        const int nb = (int)((L + BQ - 1) / BQ);
        if (nb > 0) atomicAdd(&cnt[min(nb, levels) - 1], 1);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int run = 0;
        for (int c = levels - 1; c >= 0; --c) {  // suffix sum: sequences with more than c blocks
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
        const int nb = min((int)((L + BQ - 1) / BQ), levels);
        for (int c = 0; c < nb; ++c) {
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
    float scale_log2;  // |softmax_scale| * log2(e); a negative scale negates Q inside the MMA
};

template <int D>
struct SmemLayout {
    static constexpr int kTileBytes = BM * D * 2;   // one [128, D] bf16 tile (Q_t, K_j or V_j)
    static constexpr int kBlockBytes = BM * 128;    // one [128 rows, 64 cols] swizzled block
    static constexpr int kQ = 0;                    // Q_0, Q_1
    static constexpr int kKV = 2 * kTileBytes;      // ring of kSlots tiles
    static constexpr int kBars = kKV + kSlots * kTileBytes;
    static constexpr int kTotal = kBars + 256;
    static constexpr int kDynamic = kTotal + 1024;  // slack for the 1024-byte alignment
};

// One (work item, q head) pair as every warp role sees it.
struct Work {
    int h, g;        // q head, kv head
    int64_t t0;      // first token of the sequence
    int L;           // sequence length
    int row0;        // first row of the block inside the sequence
    int n[2];        // KV tiles of tile 0 / tile 1 (0 = tile has no rows)
    int n_kv;        // max of the two
};

__device__ __forceinline__ Work decode_work(const AttnParams& p, int w) {
    Work k;
    const int item = w / p.Hq;
    k.h = w - item * p.Hq;
    k.g = k.h / (p.Hq / p.Hkv);
    const int2 it = p.items[item];
    k.t0 = p.cu_seqlens[it.x];
    k.L = (int)(p.cu_seqlens[it.x + 1] - k.t0);
    k.row0 = it.y * BQ;
    k.n[0] = 2 * it.y + 1;
    k.n[1] = (k.row0 + BM < k.L) ? 2 * it.y + 2 : 0;
    k.n_kv = max(k.n[0], k.n[1]);
    return k;
}

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
template <int N>
__device__ __forceinline__ void setmaxnreg_inc() {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N));
}
template <int N>
__device__ __forceinline__ void setmaxnreg_dec() {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N));
}

template <int D>
__global__ void __launch_bounds__(kThreadsAttn, 1)
attn_fwd(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
         const __grid_constant__ CUtensorMap tm_v, const AttnParams p, const int negate_q) {
    using SL = SmemLayout<D>;
    constexpr int kTmemCols = 512;  // S_0/P_0: [0,128)  S_1/P_1: [128,256)  O_0: [256,..)  O_1: [384,..)

    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem = smem_raw + (smem_base - ptx::smem_u32(smem_raw));
    const uint32_t sQ = smem_base + SL::kQ, sKV = smem_base + SL::kKV;
    const uint32_t bars = smem_base + SL::kBars;
    const uint32_t bar_q_full = bars, bar_q_empty = bars + 8;
    auto bar_kv_full = [&](int s) { return bars + 16 + 8 * s; };
    auto bar_kv_empty = [&](int s) { return bars + 16 + 8 * kSlots + 8 * s; };
    auto bar_s_full = [&](int t) { return bars + 16 + 16 * kSlots + 8 * t; };
    auto bar_p_full = [&](int t) { return bars + 32 + 16 * kSlots + 8 * t; };
    auto bar_o_done = [&](int t) { return bars + 48 + 16 * kSlots + 8 * t; };
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + SL::kBars + 192);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int n_work = p.header->n_items * p.Hq;

    if (tid == 0) {
        ptx::prefetch_tensormap(&tm_q);
        ptx::prefetch_tensormap(&tm_k);
        ptx::prefetch_tensormap(&tm_v);
        ptx::mbar_init(bar_q_full, 1);
        ptx::mbar_init(bar_q_empty, 1);
        for (int s = 0; s < kSlots; ++s) {
            ptx::mbar_init(bar_kv_full(s), 1);
            ptx::mbar_init(bar_kv_empty(s), 1);
        }
        for (int t = 0; t < 2; ++t) {
            ptx::mbar_init(bar_s_full(t), 1);
            ptx::mbar_init(bar_p_full(t), BM);
            ptx::mbar_init(bar_o_done(t), 1);
        }
        ptx::fence_barrier_init();
    }
    if (warp == 2) {
        ptx::tmem_alloc<kTmemCols>(ptx::smem_u32(const_cast<uint32_t*>(tmem_slot)));
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp < 4) {
        setmaxnreg_dec<80>();
        if (warp == 0 && lane == 0) {
            // ================================ TMA producer ================================
            int slot = 0;
            uint32_t ph_kv = 0, ph_q = 0;
            for (int w = blockIdx.x; w < n_work; w += gridDim.x) {
                const Work k = decode_work(p, w);
                ptx::mbar_wait(bar_q_empty, ph_q ^ 1);
                ph_q ^= 1;
                const int nq = k.n[1] ? 2 : 1;
                ptx::mbar_arrive_expect_tx(bar_q_full, nq * SL::kTileBytes);
                for (int t = 0; t < nq; ++t)
#pragma unroll
                    for (int c = 0; c < D / 64; ++c)
                        ptx::tma_load_3d(sQ + t * SL::kTileBytes + c * SL::kBlockBytes, &tm_q,
                                         bar_q_full, c * 64, k.h, (int)(k.t0 + k.row0 + t * BM));
                for (int j = 0; j < k.n_kv; ++j) {
#pragma unroll
                    for (int kv = 0; kv < 2; ++kv) {  // K_j then V_j
                        ptx::mbar_wait(bar_kv_empty(slot), ph_kv ^ 1);
                        ptx::mbar_arrive_expect_tx(bar_kv_full(slot), SL::kTileBytes);
#pragma unroll
                        for (int c = 0; c < D / 64; ++c)
                            ptx::tma_load_3d(sKV + slot * SL::kTileBytes + c * SL::kBlockBytes,
                                             kv == 0 ? &tm_k : &tm_v, bar_kv_full(slot), c * 64,
                                             k.g, (int)(k.t0 + j * BN));
                        if (++slot == kSlots) {
                            slot = 0;
                            ph_kv ^= 1;
                        }
                    }
                }
            }
        } else if (warp == 1 && lane == 0) {
            // ================================ MMA issuer ==================================
            const uint32_t idesc_s =
                ptx::umma_idesc_bf16(BM, BN, false, false) | (negate_q ? (1u << 13) : 0u);
            constexpr uint32_t idesc_pv = ptx::umma_idesc_bf16(BM, D, false, true);
            int slot = 0;
            uint32_t ph_kv = 0, ph_q = 0, ph_p[2] = {0, 0};
            auto advance = [&]() {
                if (++slot == kSlots) {
                    slot = 0;
                    ph_kv ^= 1;
                }
            };
            // S_t = Q_t K^T : both operands K-major (D contiguous), 128-byte swizzle
            auto issue_qk = [&](int t, int kslot) {
                const uint32_t a = sQ + t * SL::kTileBytes, b = sKV + kslot * SL::kTileBytes;
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk) {
                    const uint32_t off = (kk / 4) * SL::kBlockBytes + (kk % 4) * 32;
                    ptx::umma_ss(tmem + t * 128, ptx::umma_smem_desc_sw128(a + off, 16, 1024),
                                 ptx::umma_smem_desc_sw128(b + off, 16, 1024), idesc_s, kk > 0);
                }
                ptx::umma_commit(bar_s_full(t));
            };
            // O_t (+)= P_t V : A = P_t from tensor memory, B = V (MN-major: D contiguous)
            auto issue_pv = [&](int t, int vslot, bool accumulate) {
                const uint32_t b = sKV + vslot * SL::kTileBytes;
#pragma unroll
                for (int kk = 0; kk < BN / 16; ++kk)
                    ptx::umma_ts(tmem + 256 + t * 128, tmem + t * 128 + kk * 8,
                                 ptx::umma_smem_desc_sw128(b + kk * 2048, SL::kBlockBytes, 1024),
                                 idesc_pv, (accumulate || kk > 0) ? 1u : 0u);
            };
            for (int w = blockIdx.x; w < n_work; w += gridDim.x) {
                const Work k = decode_work(p, w);
                ptx::mbar_wait(bar_q_full, ph_q);
                ph_q ^= 1;
                ptx::mbar_wait(bar_kv_full(slot), ph_kv);  // K_0
                ptx::tc_fence_after();
                issue_qk(0, slot);
                if (k.n[1]) issue_qk(1, slot);
                ptx::umma_commit(bar_kv_empty(slot));
                advance();
                for (int j = 0; j < k.n_kv; ++j) {
                    const int vslot = slot;
                    const uint32_t vph = ph_kv;
                    advance();
                    const int kslot = slot;  // K_{j+1}, if any
                    const bool has_next = j + 1 < k.n_kv;
                    ptx::mbar_wait(bar_kv_full(vslot), vph);
                    if (has_next) ptx::mbar_wait(bar_kv_full(kslot), ph_kv);
#pragma unroll
                    for (int t = 0; t < 2; ++t) {
                        if (j < k.n[t]) {
                            ptx::mbar_wait(bar_p_full(t), ph_p[t]);
                            ph_p[t] ^= 1;
                            ptx::tc_fence_after();
                            issue_pv(t, vslot, j > 0);
                            if (j + 1 < k.n[t]) issue_qk(t, kslot);
                            if (j == k.n[t] - 1) ptx::umma_commit(bar_o_done(t));
                        }
                    }
                    ptx::umma_commit(bar_kv_empty(vslot));
                    if (has_next) {
                        ptx::umma_commit(bar_kv_empty(kslot));
                        advance();
                    }
                }
                ptx::umma_commit(bar_q_empty);
            }
        }
    } else {
        // ============================ softmax + epilogue groups ===========================
        setmaxnreg_inc<208>();
        const int t = (warp >> 2) - 1;             // tile of this group (0 or 1)
        const int row = tid - (t + 1) * BM;        // query row inside the tile == TMEM lane
        const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t tS = tmem + t * 128 + lane_off;        // S_t, overwritten by P_t (bf16)
        const uint32_t tO = tmem + 256 + t * 128 + lane_off;  // O_t
        const float sc = p.scale_log2;
        uint32_t ph_s = 0, ph_o = 0;

        for (int w = blockIdx.x; w < n_work; w += gridDim.x) {
            const Work k = decode_work(p, w);
            const int n_t = k.n[t];
            if (n_t == 0) continue;  // this tile has no rows in this block
            float m_used = 0.f, l_run = 0.f;
            for (int j = 0; j < n_t; ++j) {
                ptx::mbar_wait(bar_s_full(t), ph_s);
                ph_s ^= 1;
                ptx::tc_fence_after();
                // ---- A2: scores of this row, running max -------------------------------------
                float s[BN];
#pragma unroll
                for (int c = 0; c < BN / 32; ++c)
                    ptx::tmem_ld32(tS + c * 32, *reinterpret_cast<uint32_t(*)[32]>(&s[c * 32]));
                ptx::tmem_wait_ld();
                const bool diag = (j == n_t - 1);  // diagonal tile: keys after the query are masked
                if (diag) {
#pragma unroll
                    for (int c = 0; c < BN; ++c)
                        if (c > row) s[c] = -INFINITY;
                }
                float mx0 = s[0], mx1 = s[1], mx2 = s[2], mx3 = s[3];
#pragma unroll
                for (int c = 4; c < BN; c += 4) {
                    mx0 = fmaxf(mx0, s[c]);
                    mx1 = fmaxf(mx1, s[c + 1]);
                    mx2 = fmaxf(mx2, s[c + 2]);
                    mx3 = fmaxf(mx3, s[c + 3]);
                }
                const float m_new = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * sc;
                if (j == 0) {
                    m_used = m_new;
                } else {
                    // move the max (and rescale l, O) only when it grew by more than 2^8
                    const bool need = m_new > m_used + kRescaleThreshold;
                    if (__any_sync(0xffffffffu, need)) {
                        const float alpha = need ? ex2_approx(m_used - m_new) : 1.f;
                        if (need) m_used = m_new;
                        l_run *= alpha;
#pragma unroll
                        for (int c = 0; c < D / 32; ++c) {
                            uint32_t r[32];
                            ptx::tmem_ld32(tO + c * 32, r);
                            ptx::tmem_wait_ld();
#pragma unroll
                            for (int i = 0; i < 32; ++i)
                                r[i] = __float_as_uint(__uint_as_float(r[i]) * alpha);
                            ptx::tmem_st32(tO + c * 32, r);
                        }
                    }
                }
                // ---- P = exp2(s * scale_log2 - m), row sum, bf16 pairs into the S columns ------
                float l0 = 0.f, l1 = 0.f, l2 = 0.f, l3 = 0.f;
                auto exp_pass = [&](auto is_diag) {
                    constexpr bool kDiag = decltype(is_diag)::value;
                    auto arg = [&](float x) {
                        const float a = fmaf(x, sc, -m_used);
                        // a masked key must give exactly 0 even when scale_log2 == 0 (-inf * 0)
                        return (kDiag && x == -INFINITY) ? -INFINITY : a;
                    };
#pragma unroll
                    for (int c = 0; c < BN / 32; ++c) {
                        uint32_t pk[16];
#pragma unroll
                        for (int i = 0; i < 32; i += 4) {
                            const float p0 = ex2_approx(arg(s[c * 32 + i + 0]));
                            const float p1 = ex2_approx(arg(s[c * 32 + i + 1]));
                            const float p2 = ex2_approx(arg(s[c * 32 + i + 2]));
                            const float p3 = ex2_approx(arg(s[c * 32 + i + 3]));
                            l0 += p0;
                            l1 += p1;
                            l2 += p2;
                            l3 += p3;
                            __nv_bfloat162 h0 = __floats2bfloat162_rn(p0, p1);
                            __nv_bfloat162 h1 = __floats2bfloat162_rn(p2, p3);
                            pk[i / 2] = *reinterpret_cast<uint32_t*>(&h0);
                            pk[i / 2 + 1] = *reinterpret_cast<uint32_t*>(&h1);
                        }
                        ptx::tmem_st16(tS + c * 16, pk);
                    }
                };
                if (diag)
                    exp_pass(std::true_type{});
                else
                    exp_pass(std::false_type{});
                l_run += (l0 + l1) + (l2 + l3);
                ptx::tmem_wait_st();
                ptx::tc_fence_before();
                ptx::mbar_arrive(bar_p_full(t));
            }
            // ---- epilogue: O_t / l -> bf16 -> global; A4: logsumexp ---------------------------------
            ptx::mbar_wait(bar_o_done(t), ph_o);
            ph_o ^= 1;
            ptx::tc_fence_after();
            const int row_g = k.row0 + t * BM + row;
            const float inv_l = 1.f / l_run;
            __nv_bfloat16* orow = p.o + ((k.t0 + row_g) * p.Hq + k.h) * (int64_t)D;
#pragma unroll
            for (int c = 0; c < D / 32; ++c) {
                uint32_t r[32];
                ptx::tmem_ld32(tO + c * 32, r);
                ptx::tmem_wait_ld();
                if (row_g < k.L) {
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
            if (row_g < k.L)
                p.lse[(int64_t)k.h * p.T + k.t0 + row_g] = (m_used + log2f(l_run)) * kLn2;
            ptx::tc_fence_before();
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 2) ptx::tmem_dealloc<kTmemCols>(tmem);
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
                            const AttnParams& p, int negate_q, int grid, cudaStream_t s) {
    using SL = SmemLayout<D>;
    static bool configured = false;
    if (!configured) {
        MOSAIC_CUDA_TRY(cudaFuncSetAttribute(attn_fwd<D>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             SL::kDynamic));
        configured = true;
    }
    attn_fwd<D><<<grid, kThreadsAttn, SL::kDynamic, s>>>(tq, tk, tv, p, negate_q);
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
    Workspace w = carve(workspace, n_seqs, total_tokens);
    if (workspace_bytes < w.total_bytes) return MOSAIC_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);

    CUtensorMap tq, tk, tv;
    if (!make_tensor_map(&tq, q, total_tokens, Hq, D, BM) ||
        !make_tensor_map(&tk, k, total_tokens, Hkv, D, BN) ||
        !make_tensor_map(&tv, v, total_tokens, Hkv, D, BN))
        return MOSAIC_ERR_CUDA;

    const int levels = (int)(total_tokens / BQ) + 2;
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
    p.scale_log2 = fabsf(softmax_scale) * kLog2e;
    const int negate_q = softmax_scale < 0.f ? 1 : 0;
    const int64_t max_work = (total_tokens / BQ + n_seqs) * (int64_t)Hq;
    if (max_work >= (1ll << 31)) return MOSAIC_ERR_UNSUPPORTED;
    const int grid = (int)(max_work < num_sms() ? max_work : num_sms());
    return D == 64 ? launch_attn<64>(tq, tk, tv, p, negate_q, grid, s)
                   : launch_attn<128>(tq, tk, tv, p, negate_q, grid, s);
}
