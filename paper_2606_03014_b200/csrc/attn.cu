// attn.cu -- step 2 of the confidence-gated aggregator stage: the aggregator's prefill attention
// over the survivors' packed contexts ("process the combined output or reasoning
// traces of its experts"; math fixed by BASELINE.json north_star: variable-length causal
// grouped-query attention, bf16 O + fp32 row logsumexp).
//
// A5    schedule_kernel : (sequence, 256-row q block) work items, longest (most KV tiles) first.
// A1-A4 attn_fwd        : persistent, warp-specialised tcgen05 / TMEM / TMA flash attention.
//   One CTA per SM works through (item, q head) pairs.  A q block is two 128-row tiles.  Each
//   128-key tile j is taken in two steps of 64 keys: the tensor core computes S_t = Q_t K^T for
//   64 keys into one of TWO 64-column score buffers of the tile in tensor memory, a 128-thread
//   softmax group per tile (one thread per query row) turns it into P_t in place (bf16, same
//   TMEM columns), and O_t += P_t V accumulates in tensor memory.  While the group works on one
//   buffer the scores of the next step are already being computed into the other, so a softmax
//   group never waits for the tensor pipe in the steady state.  The two tiles are two
//   independent streams that share only the K/V ring: each has its own MMA-issuing thread and
//   its own softmax group, and a tile that finishes its item first starts the next item
//   without waiting.
//     warps 0-3   : softmax of tile 0                   warps 4-7 : ... of tile 1
//     warps 8-11  : epilogue of both tiles (O_t / l -> bf16 -> global, logsumexp), so that the
//                   softmax groups go straight on to the next item
//     warp 12     : TMA producer (Q tiles, K/V ring of kSlots 128-key tiles, 128-byte swizzle);
//                   it also takes the CTA's next work unit from a global counter and publishes
//                   it to the other roles through a small shared-memory ring
//     warp 13, 14 : tcgen05.mma issuer of tile 0 / tile 1 (one elected thread each);
//                   warp 14 also allocates / releases tensor memory
//   Both softmax groups are busy all the time, so the FMA / ALU issue slots are as scarce as the
//   MUFU unit: all exponentials go to MUFU (MOSAIC_POLY_PAIRS = n evaluates n of every 4 element
//   pairs on the FMA pipe instead, exp2_poly2; measured slower here), and the two issuers do not
//   take turns (MOSAIC_MMA_LOCK = 1 makes them; it paid when S and P shared one buffer).
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
constexpr int BN = 128;       // key rows per K/V tile (one TMA load, one ring slot)
constexpr int BS = 64;        // keys per step         (UMMA N of S; two steps per K/V tile)
constexpr int BQ = 2 * BM;    // query rows per work item (two tiles)
#ifndef MOSAIC_KV_SLOTS
#define MOSAIC_KV_SLOTS 5
#endif
constexpr int kSlots = MOSAIC_KV_SLOTS;  // K/V ring depth (tiles)
constexpr int kThreadsAttn = 512;
constexpr int kUnitSlots = 4;  // work units the producer may publish ahead of the other roles
// Warp roles.  The softmax groups take the LOW warp ids (TMEM lane quarter = warp % 4) and the
// single-thread roles the HIGH ones: the warp schedulers favour the highest warp id among the
// eligible warps, and the MMA issuers are the threads everything else waits for.
constexpr int kWarpEpilogue = 8;  // warps 8-11: O_t / l -> global, for both tiles
constexpr int kWarpProducer = 12, kWarpMma0 = 13, kWarpMma1 = 14;  // warp 15: idle
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr float kRescaleThreshold = 8.0f;  // log2 units
#ifndef MOSAIC_POLY_PAIRS
#define MOSAIC_POLY_PAIRS 0
#endif
#ifndef MOSAIC_MMA_LOCK
#define MOSAIC_MMA_LOCK 0
#endif
constexpr int kPolyPairs = MOSAIC_POLY_PAIRS;  // of every 4 element pairs: exp2 on the FMA pipe

// ------------------------------------------------------------------------------- A5: schedule
struct SchedHeader {
    int n_items;    // number of (sequence, q block) entries
    int next_unit;  // work units handed out so far (attn_fwd's CTAs take them in cost order)
    int pad[2];
};

struct Workspace {
    SchedHeader* header;
    int* cnt;     // [levels]  sequences whose costliest block sits at the level
    int* cursor;  // [levels]
    int* start;   // [levels]  sequences at higher levels (= the first rank of the level)
    int* rank;    // [n_seqs]      rank of sequence s in descending cost order
    int* first;   // [n_seqs + 1]  blocks of the sequences of lower rank (indexed by rank)
    int4* items;  // [capacity] (first q token of the sequence, its q length, q block, first k token)
    int* items_lk;  // [capacity] its k length
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
    w.rank = reinterpret_cast<int*>(p + off);
    off += ((size_t)n_seqs + 1) * sizeof(int);
    w.first = reinterpret_cast<int*>(p + off);
    off += ((size_t)n_seqs + 2) * sizeof(int);
    off = (off + 15) & ~size_t(15);
    w.items = reinterpret_cast<int4*>(p + off);
    off += cap * sizeof(int4);
    w.items_lk = reinterpret_cast<int*>(p + off);
    off += cap * sizeof(int);
    w.total_bytes = (off + 255) & ~size_t(255);
    return w;
}

// A5, the length-sorted work list.  Sequences are ranked by the cost of their costliest q block --
// level = ceil(visible keys / 256) of the LAST block, relative to the cheapest sequence of the batch:
// for the plain prefill simply the length -- longest first (counting sort over the levels; order
// inside a level is arbitrary, the results do not depend on the schedule), and a sequence's blocks
// follow one another from the last (most KV tiles) to the first.  attn_fwd walks the list once per
// KV head (KV head outermost, the q heads of its group innermost): the ~148 units in flight are then
// neighbouring q blocks of ONE (sequence, KV head) -- they stream the same K / V, which stays in
// L2 (16.8 MB for a 32 k-token head) -- instead of the same q block of every KV head (134 MB for a
// 32 k-token sequence, more than the L2: round 1's order re-read K / V from DRAM 4.5-6x).  The
// hand-out is dynamic, and the last units of the launch are the first blocks of the shortest
// sequences, so the CTAs still finish together.  One block; the scans are chunked over its threads.

// Sum of v over the threads with a larger thread index (whole block calls).
__device__ __forceinline__ int block_suffix_exclusive(int v, int* warp_tot /* [32] shared */) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    int x = v;  // inclusive suffix inside the warp
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_down_sync(0xffffffffu, x, o);
        if (lane + o < 32) x += y;
    }
    __syncthreads();  // warp_tot may still be read from a previous call
    if (lane == 0) warp_tot[warp] = x;
    __syncthreads();
    int above = 0;
    for (int w = warp + 1; w < nwarp; ++w) above += warp_tot[w];
    return above + x - v;
}
// Sum of v over the threads with a smaller thread index (whole block calls).
__device__ __forceinline__ int block_prefix_exclusive(int v, int* warp_tot /* [32] shared */) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int x = v;  // inclusive prefix inside the warp
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    __syncthreads();
    if (lane == 31) warp_tot[warp] = x;
    __syncthreads();
    int below = 0;
    for (int w = 0; w < warp; ++w) below += warp_tot[w];
    return below + x - v;
}

// A sequence's q rows and keys come either from the two cu_seqlens arrays (rows / keys of
// sequence s = [cu[s], cu[s+1])) or, when `desc` is given, from explicit per-sequence views -- q
// rows and key ranges that need not be adjacent or disjoint (the chunks of a chunked prefill all
// start at their sequence's first key).
__device__ __forceinline__ void seq_view(const int64_t* cu_q, const int64_t* cu_k, const SeqDesc* desc,
                                         int s, int64_t& q0, int64_t& L, int64_t& k0, int64_t& Lk) {
    if (desc) {
        const SeqDesc d = desc[s];
        q0 = d.q_start;
        L = d.q_len;
        k0 = d.k_start;
        Lk = d.k_len;
    } else {
        q0 = cu_q[s];
        L = cu_q[s + 1] - q0;
        k0 = cu_k[s];
        Lk = cu_k[s + 1] - k0;
    }
}

// Cost level of a sequence = that of its last q block: all its keys when causal (the last row sees
// them all) or not, in 256-key units.
__device__ __forceinline__ int seq_level(int64_t L, int64_t Lk) {
    return (L > 0 && Lk > 0) ? (int)((Lk - 1) / BQ) : 0;
}

__global__ void __launch_bounds__(1024) schedule_kernel(const int64_t* __restrict__ cu_seqlens,
                                                        const int64_t* __restrict__ cu_seqlens_k,
                                                        const SeqDesc* __restrict__ desc,
                                                        int n_seqs, int levels, SchedHeader* header,
                                                        int* cnt, int* start, int* cursor, int* rank,
                                                        int* first, int4* items, int* items_lk) {
    __shared__ int warp_tot[32];
    __shared__ int lv_min;  // levels are counted from the cheapest sequence of the batch: the arrays
                            // hold total_q_tokens / 256 + 2 levels however long the keys are
    __shared__ int carry;
    const int tid = threadIdx.x;
    if (tid == 0) lv_min = 0x7fffffff;
    __syncthreads();
    for (int s = tid; s < n_seqs; s += blockDim.x) {
        int64_t q0, L, k0, Lk;
        seq_view(cu_seqlens, cu_seqlens_k, desc, s, q0, L, k0, Lk);
        if (L > 0) atomicMin(&lv_min, seq_level(L, Lk));
    }
    __syncthreads();
    const int base = lv_min == 0x7fffffff ? 0 : lv_min;
    for (int s = tid; s < n_seqs; s += blockDim.x) {
        int64_t q0, L, k0, Lk;
        seq_view(cu_seqlens, cu_seqlens_k, desc, s, q0, L, k0, Lk);
        if (L > 0) atomicAdd(&cnt[min(levels - 1, seq_level(L, Lk) - base)], 1);
    }
    __syncthreads();
    // start[c] <- sequences at the levels above c (exclusive suffix sum of the counts)
    const int chunk = (levels + (int)blockDim.x - 1) / (int)blockDim.x;
    const int lo = min(levels, tid * chunk), hi = min(levels, lo + chunk);
    int local = 0;
    for (int c = lo; c < hi; ++c) local += cnt[c];
    int pos = block_suffix_exclusive(local, warp_tot);
    for (int c = hi - 1; c >= lo; --c) {
        start[c] = pos;
        pos += cnt[c];
    }
    __syncthreads();
    // rank of every sequence (empty ones are not ranked), its block count by rank
    const int n_ranked = start[0] + cnt[0];
    for (int s = tid; s < n_seqs; s += blockDim.x) {
        int64_t q0, L, k0, Lk;
        seq_view(cu_seqlens, cu_seqlens_k, desc, s, q0, L, k0, Lk);
        int r = -1;
        if (L > 0) {
            const int lv = min(levels - 1, seq_level(L, Lk) - base);
            r = start[lv] + atomicAdd(&cursor[lv], 1);
            first[r] = (int)((L + BQ - 1) / BQ);
        }
        rank[s] = r;
    }
    if (tid == 0) carry = 0;
    __syncthreads();
    // first[r] <- blocks of the sequences of lower rank (exclusive prefix sum, 1024 ranks a round)
    for (int r0 = 0; r0 < n_ranked; r0 += (int)blockDim.x) {
        const int r = r0 + tid;
        const int nb = r < n_ranked ? first[r] : 0;
        const int before = carry + block_prefix_exclusive(nb, warp_tot);
        if (r < n_ranked) first[r] = before;
        __syncthreads();
        if (tid == (int)blockDim.x - 1) carry = before + nb;
        __syncthreads();
    }
    if (tid == 0) header->n_items = carry;
    for (int s = tid; s < n_seqs; s += blockDim.x) {
        const int r = rank[s];
        if (r < 0) continue;
        int64_t q0, L, k0, Lk;
        seq_view(cu_seqlens, cu_seqlens_k, desc, s, q0, L, k0, Lk);
        const int nb = (int)((L + BQ - 1) / BQ);
        const int at0 = first[r];
        for (int c = 0; c < nb; ++c) {
            const int at = at0 + (nb - 1 - c);  // the last block (most KV tiles) first
            items[at] = make_int4((int)q0, (int)L, c, (int)k0);  // (token counts are < 2^31)
            items_lk[at] = (int)Lk;
        }
    }
}

// ------------------------------------------------------------------------------ A1-A4: forward
struct AttnParams {
    const int64_t* cu_seqlens;
    const int4* items;
    const int* items_lk;
    SchedHeader* header;
    __nv_bfloat16* o;
    float* lse;
    int64_t T;
    int Hq, Hkv;
    float scale_log2;  // |softmax_scale| * log2(e); a negative scale negates Q inside the MMA
    float inv_group;   // 1 / (Hq / Hkv)
    int group;         // Hq / Hkv
    int prefix_len;    // shared-prefix cascade: every sequence's keys are prefix_len shared keys (their
    int prefix_pad;    // own tensor maps) followed by its own; prefix_pad = prefix_len rounded up to 128
    int causal;        // 0: every q row sees all the keys of its sequence
    int o_align32;     // o is 32-byte aligned: the epilogue may use 256-bit stores
};

template <int D>
struct SmemLayout {
    static constexpr int kTileBytes = BM * D * 2;   // one [128, D] bf16 tile (Q_t, K_j or V_j)
    static constexpr int kBlockBytes = BM * 128;    // one [128 rows, 64 cols] swizzled block
    static constexpr int kQ = 0;                    // Q_0, Q_1
    static constexpr int kKV = 2 * kTileBytes;      // ring of kSlots tiles
    static constexpr int kBars = kKV + kSlots * kTileBytes;
    static constexpr int kStat = kBars + 512;       // (logsumexp, 1 / normaliser) of every row of both tiles, for the epilogue
    static constexpr int kUnits = kStat + 2 * BM * 8;  // ring of work-unit descriptors (32 bytes each)
    static constexpr int kTotal = kUnits + kUnitSlots * 32;
    static constexpr int kDynamic = kTotal;         // the base is 1024-byte aligned (checked)
    static_assert(kDynamic <= 227 * 1024, "shared memory of one CTA");
};

// mbarriers (8 bytes each) inside the kBars region
enum Bar : uint32_t {
    kBarQFull = 0,                          // [2]  Q_t landed                       (TMA tx)
    kBarQEmpty = 2,                         // [2]  last S_t of the item has read Q_t (commit)
    kBarKvFull = 4,                         // [kSlots] K_j / V_j landed             (TMA tx)
    kBarKvEmpty = 4 + kSlots,               // [2][kSlots] stream t is done with the slot
    kBarSFull = 4 + 3 * kSlots,             // [2][2] score buffer b of tile t complete (commit)
    kBarPFull = kBarSFull + 4,              // [2][2] P_t written over buffer b      (4 warps)
    kBarPvDone = kBarSFull + 8,             // [2]  a PV_t step complete             (commit)
    kBarODone = kBarSFull + 10,             // [2]  last PV_t of the item complete   (commit)
    kBarStat = kBarSFull + 12,              // [2]  (logsumexp, 1/normaliser) of the tile's rows are in shared memory (4 warps)
    kBarOFree = kBarSFull + 14,             // [2]  the epilogue has read O_t        (4 warps)
    kBarUnitFull = kBarSFull + 16,          // [kUnitSlots] the producer has published a work unit
    kBarUnitEmpty = kBarSFull + 16 + kUnitSlots,  // [kUnitSlots] every other role has read it (14 warps)
    kNumBars = kBarSFull + 16 + 2 * kUnitSlots
};
static_assert(kNumBars * 8 + 8 <= 512, "barrier region");

// One (work item, q head) pair as every warp role sees it.
struct Work {
    int h, g;        // q head, kv head
    int64_t t0;      // first q token of the sequence
    int64_t tk0;     // first k token of the sequence
    int L;           // q rows of the sequence
    int off;         // row i sees keys j <= min(i + off, lk - 1): k length - q length when causal
                     // (0 for the plain prefill), huge when not
    int lk;          // keys of the sequence
    int row0;        // first row of the block inside the sequence
    int n0, n1;      // KV tiles of tile 0 / tile 1 (0 = tile has no rows)
    int n_kv;        // max of the two
    __device__ __forceinline__ int n(int t) const { return t ? n1 : n0; }
    __device__ __forceinline__ int tile_of(int t) const { return t; }
};

// Work units (unit w = q head w % Hq of entry w / Hq of the cost-sorted work list) are handed out
// dynamically: the producer warp of a CTA takes the next unit from a global counter, loads its
// descriptor and publishes both in a small shared-memory ring that every other warp role reads,
// so all roles of a CTA walk the same sequence, and a CTA that runs faster (the per-CTA finish
// times of a static assignment spread over 5 % of the kernel) simply takes more units.
constexpr int kUnitConsumers = 14;  // 8 softmax + 4 epilogue + 2 issuer warps
struct UnitEntry {  // 32 bytes in shared memory
    int4 it;        // (first q token, q length, q block, first k token) of the entry
    int h;          // q head; < 0: no more work
    int lk;         // k length of the entry
    int pad[2];
};
__device__ __forceinline__ Work make_work(const AttnParams& p, const int4 it, int h, int lk) {
    Work k;
    k.h = h;
    k.g = __float2int_rd(((float)h + 0.5f) * p.inv_group);  // h / (Hq / Hkv)
    k.t0 = it.x;
    k.tk0 = it.w;
    k.L = it.y;
    // (with a shared prefix the keys are [prefix, padded to whole tiles][own keys]: every row sees
    //  the whole prefix, so the offset and the key count simply grow by prefix_pad)
    k.off = p.causal ? lk - it.y + p.prefix_pad : (1 << 29);
    k.lk = lk + p.prefix_pad;
    k.row0 = it.z * BQ;
    // KV tiles of a q tile: up to the last key its last row sees (2c+1 and 2c+2 when off = 0)
    // (clamped at 0: a sequence without keys -- mosaic_agg_decode_attn makes those -- or, against
    //  the contract, with fewer keys than q rows when causal, has tiles that visit nothing)
    const int last0 = max(0, min(min(k.row0 + BM, k.L) + k.off, k.lk));
    const int last1 = max(0, min(min(k.row0 + BQ, k.L) + k.off, k.lk));
    k.n0 = (last0 + BN - 1) / BN;
    k.n1 = (k.row0 + BM < k.L) ? (last1 + BN - 1) / BN : 0;
    k.n_kv = max(k.n0, k.n1);
    return k;
}

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// 2^x for two x <= ~100 on the FMA pipe: x = n + f with n = round(x) taken from the low mantissa
// bits of x + 1.5 * 2^23, 2^f on [-0.5, 0.5] by a degree-3 minimax polynomial (relative error
// 7.5e-5, far below the 2^-9 rounding of P to bf16), 2^n added into the exponent field.
__device__ __forceinline__ float2 exp2_poly2(float2 x) {
    x.x = fmaxf(x.x, -126.f);
    x.y = fmaxf(x.y, -126.f);
    const float2 t = __fadd2_rn(x, make_float2(12582912.f, 12582912.f));
    const float2 n = __fadd2_rn(t, make_float2(-12582912.f, -12582912.f));
    const float2 f = __ffma2_rn(n, make_float2(-1.f, -1.f), x);
    float2 p = __ffma2_rn(make_float2(0.055172015f, 0.055172015f), f,
                          make_float2(0.24261113f, 0.24261113f));
    p = __ffma2_rn(p, f, make_float2(0.69326091f, 0.69326091f));
    p = __ffma2_rn(p, f, make_float2(0.99992806f, 0.99992806f));
    p.x = __int_as_float(__float_as_int(p.x) + (__float_as_int(t.x) << 23));
    p.y = __int_as_float(__float_as_int(p.y) + (__float_as_int(t.y) << 23));
    return p;
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
         const __grid_constant__ CUtensorMap tm_v, const __grid_constant__ CUtensorMap tm_kp,
         const __grid_constant__ CUtensorMap tm_vp, const AttnParams p, const int negate_q) {
    using SL = SmemLayout<D>;
    // tile t: score buffers [128 t, 128 t + 64) and [128 t + 64, 128 t + 128), each overwritten by
    // its P (bf16, 32 columns); O_t: [256 + 128 t, ..)
    constexpr int kTmemCols = 512;

    extern __shared__ __align__(1024) uint8_t smem[];  // 128-byte swizzle wants 1024-byte alignment
    const uint32_t smem_base = ptx::smem_u32(smem);
    if (smem_base & 1023u) __trap();
    const uint32_t sQ = smem_base + SL::kQ, sKV = smem_base + SL::kKV;
    const uint32_t bars = smem_base + SL::kBars;
    auto bar = [&](uint32_t which, int i = 0) { return bars + 8u * (which + (uint32_t)i); };
    auto bar_kv_empty = [&](int t, uint32_t slot) { return bar(kBarKvEmpty, t * kSlots + (int)slot); };
    volatile uint32_t* tmem_slot =
        reinterpret_cast<volatile uint32_t*>(smem + SL::kBars + 8 * kNumBars);
    const uint32_t mma_lock = bars + 8 * kNumBars + 4;  // the two issuers take turns (see below)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int n_items = p.header->n_items;
    const int n_work = n_items * p.Hq;

    if (tid == 0) {
        ptx::prefetch_tensormap(&tm_q);
        ptx::prefetch_tensormap(&tm_k);
        ptx::prefetch_tensormap(&tm_v);
        if (p.prefix_pad) {
            ptx::prefetch_tensormap(&tm_kp);
            ptx::prefetch_tensormap(&tm_vp);
        }
        for (int t = 0; t < 2; ++t) {
            ptx::mbar_init(bar(kBarQFull, t), 1);
            ptx::mbar_init(bar(kBarQEmpty, t), 1);
            for (int b = 0; b < 2; ++b) {
                ptx::mbar_init(bar(kBarSFull, 2 * t + b), 1);
                ptx::mbar_init(bar(kBarPFull, 2 * t + b), BM / 32);
            }
            ptx::mbar_init(bar(kBarPvDone, t), 1);
            ptx::mbar_init(bar(kBarODone, t), 1);
            ptx::mbar_init(bar(kBarStat, t), BM / 32);
            ptx::mbar_init(bar(kBarOFree, t), BM / 32);
            for (int s = 0; s < kSlots; ++s) ptx::mbar_init(bar_kv_empty(t, s), 1);
        }
        for (int s = 0; s < kSlots; ++s) ptx::mbar_init(bar(kBarKvFull, s), 1);
        for (int s = 0; s < kUnitSlots; ++s) {
            ptx::mbar_init(bar(kBarUnitFull, s), 1);
            ptx::mbar_init(bar(kBarUnitEmpty, s), kUnitConsumers);
        }
        asm volatile("st.shared.u32 [%0], %1;" ::"r"(mma_lock), "r"(0u) : "memory");
        ptx::fence_barrier_init();
    }
    if (warp == kWarpMma1) {
        ptx::tmem_alloc<kTmemCols>(ptx::smem_u32(const_cast<uint32_t*>(tmem_slot)));
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    // The next work unit of this CTA, as published by the producer warp (whole warp calls; false
    // when there is no more work).  n counts the units this warp has read.
    volatile UnitEntry* unit_ring = reinterpret_cast<volatile UnitEntry*>(smem + SL::kUnits);
    auto next_unit = [&](uint32_t& n, Work& k) -> bool {
        const uint32_t slot = n % kUnitSlots, ph = (n / kUnitSlots) & 1u;
        ++n;
        ptx::mbar_wait(bar(kBarUnitFull, (int)slot), ph);
        int4 it;
        it.x = unit_ring[slot].it.x;
        it.y = unit_ring[slot].it.y;
        it.z = unit_ring[slot].it.z;
        it.w = unit_ring[slot].it.w;
        const int h = unit_ring[slot].h;
        const int lk = unit_ring[slot].lk;
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(bar(kBarUnitEmpty, (int)slot));
        if (h < 0) return false;
        k = make_work(p, it, h, lk);
        return true;
    };

    // Position q of the K/V ring sequence (K_0, V_0, K_1, V_1, ... of one item after the other)
    // lives in slot q % kSlots; its full / empty barriers are in phase (q / kSlots) & 1.
    auto slot_of = [](uint32_t q) { return q % kSlots; };
    auto phase_of = [](uint32_t q) { return (q / kSlots) & 1u; };

    if (warp >= kWarpEpilogue) {
        setmaxnreg_dec<48>();
        if (warp < kWarpProducer) {
            // ====================== epilogue: O_t / l -> bf16 -> global; A4: logsumexp ======================
            const int row = tid & (BM - 1);  // query row inside the tile == TMEM lane (warp % 4 quarter)
            const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
            const float2* stat = reinterpret_cast<const float2*>(smem + SL::kStat);
            uint32_t ph[2] = {0, 0};
            uint32_t n_units = 0;
            for (Work k; next_unit(n_units, k);) {
#pragma unroll 1
                for (int t = 0; t < 2; ++t) {
                    if (k.n(t) == 0) continue;
                    ptx::mbar_wait(bar(kBarStat, t), ph[t]);   // the softmax group is done with the item
                    ptx::mbar_wait(bar(kBarODone, t), ph[t]);  // ... and so is the last PV_t
                    ph[t] ^= 1;
                    ptx::tc_fence_after();
                    const float2 ml = stat[t * BM + row];  // (logsumexp, 1 / normaliser) of the row
                    const uint32_t tO = tmem + 256 + t * 128 + lane_off;
                    const int row_g = k.row0 + t * BM + row;
                    const float inv_l = ml.y;
                    __nv_bfloat16* orow = p.o + ((k.t0 + row_g) * p.Hq + k.h) * (int64_t)D;
#pragma unroll 2
                    for (int c = 0; c < D / 16; ++c) {
                        uint32_t r[16];
                        ptx::tmem_ld16(tO + c * 16, r);
                        ptx::tmem_wait_ld();
                        if (row_g < k.L) {
                            uint32_t pk[8];
#pragma unroll
                            for (int i = 0; i < 16; i += 2) {
                                __nv_bfloat162 h = __floats2bfloat162_rn(
                                    __uint_as_float(r[i]) * inv_l, __uint_as_float(r[i + 1]) * inv_l);
                                pk[i / 2] = *reinterpret_cast<uint32_t*>(&h);
                            }
                            // one full 32-byte sector per store when the row is 32-byte aligned; O is
                            // written once and never read here: do not let it displace K/V in L2
                            if (p.o_align32) {
                                asm volatile("st.global.L1::no_allocate.L2::evict_first.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(
                                                 orow + c * 16),
                                             "r"(pk[0]), "r"(pk[1]), "r"(pk[2]), "r"(pk[3]), "r"(pk[4]),
                                             "r"(pk[5]), "r"(pk[6]), "r"(pk[7])
                                             : "memory");
                            } else {
                                *reinterpret_cast<uint4*>(orow + c * 16) =
                                    make_uint4(pk[0], pk[1], pk[2], pk[3]);
                                *reinterpret_cast<uint4*>(orow + c * 16 + 8) =
                                    make_uint4(pk[4], pk[5], pk[6], pk[7]);
                            }
                        }
                    }
                    // O_t and the row statistics have been read: the next item may overwrite them
                    ptx::tc_fence_before();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(bar(kBarOFree, t));
                    if (row_g < k.L) p.lse[(int64_t)k.h * p.T + k.t0 + row_g] = ml.x;
                }
            }
        } else if (warp == kWarpProducer) {
            // ================================ TMA producer ================================
            uint32_t pos = 0, ph_q[2] = {0, 0};
            // Units are fetched one ahead (counter and descriptor: two L2 round trips that hide
            // behind the unit in progress) and published when their turn comes.
            uint32_t n_pub = 0;
            int4 f_it = make_int4(0, 0, 0, 0);
            int f_h = -1, f_lk = 0;
            auto fetch = [&]() {
                int w = 0;
                if (lane == 0) w = atomicAdd(&p.header->next_unit, 1);
                w = __shfl_sync(0xffffffffu, w, 0);
                f_h = -1;
                if (w < n_work) {
                    // unit w = (KV head g, work-list entry, q head r of g's group), r fastest
                    const int per_g = n_items * p.group;
                    const int g = w / per_g, rem = w - g * per_g;
                    const int item = rem / p.group;
                    f_h = g * p.group + (rem - item * p.group);
                    f_it = __ldg(p.items + item);
                    f_lk = __ldg(p.items_lk + item);
                }
            };
            auto publish = [&]() {  // the fetched unit (or the end marker) to every other role
                const uint32_t slot = n_pub % kUnitSlots, ph = (n_pub / kUnitSlots) & 1u;
                ++n_pub;
                ptx::mbar_wait(bar(kBarUnitEmpty, (int)slot), ph ^ 1);
                if (lane == 0) {
                    unit_ring[slot].it.x = f_it.x;
                    unit_ring[slot].it.y = f_it.y;
                    unit_ring[slot].it.z = f_it.z;
                    unit_ring[slot].it.w = f_it.w;
                    unit_ring[slot].h = f_h;
                    unit_ring[slot].lk = f_lk;
                    ptx::mbar_arrive(bar(kBarUnitFull, (int)slot));
                }
                __syncwarp();
            };
            fetch();
            for (;;) {
                publish();
                if (f_h < 0) break;
                const Work k = make_work(p, f_it, f_h, f_lk);
                fetch();  // the unit after this one
                auto load_q = [&](int t) {
                    ptx::mbar_wait(bar(kBarQEmpty, t), ph_q[t] ^ 1);
                    ph_q[t] ^= 1;
                    if (ptx::elect_one()) {
                        ptx::mbar_arrive_expect_tx(bar(kBarQFull, t), SL::kTileBytes);
#pragma unroll
                        for (int c = 0; c < D / 64; ++c)
                            ptx::tma_load_3d(sQ + t * SL::kTileBytes + c * SL::kBlockBytes, &tm_q,
                                             bar(kBarQFull, t), c * 64, k.h,
                                             (int)(k.t0 + k.row0 + t * BM));
                    }
                    __syncwarp();
                };
                // KV tile j of the unit: one of the shared prefix's tiles first (rows past prefix_len
                // are outside that tensor map and arrive as zeros; the softmax groups mask them),
                // then the sequence's own keys
                const int jp = p.prefix_pad / BN;
                auto load_kv = [&](bool is_v, int j) {
                    const uint32_t slot = slot_of(pos), ph = phase_of(pos);
                    ++pos;
                    ptx::mbar_wait(bar_kv_empty(0, slot), ph ^ 1);
                    ptx::mbar_wait(bar_kv_empty(1, slot), ph ^ 1);
                    if (ptx::elect_one()) {
                        const CUtensorMap* tm = j < jp ? (is_v ? &tm_vp : &tm_kp) : (is_v ? &tm_v : &tm_k);
                        const int row = j < jp ? j * BN : (int)(k.tk0 + (j - jp) * BN);
                        ptx::mbar_arrive_expect_tx(bar(kBarKvFull, slot), SL::kTileBytes);
#pragma unroll
                        for (int c = 0; c < D / 64; ++c)
                            ptx::tma_load_3d(sKV + slot * SL::kTileBytes + c * SL::kBlockBytes, tm,
                                             bar(kBarKvFull, slot), c * 64, k.g, row);
                    }
                    __syncwarp();
                };
                // A tile without KV tiles (n_t = 0) is skipped by its issuer, softmax group and
                // epilogue: its Q must not be loaded either (nobody would release the buffer), and
                // a unit without any KV tile takes no ring position at all.
                if (k.n_kv == 0) continue;
                if (k.n0) load_q(0);
                load_kv(false, 0);
                if (k.n1) load_q(1);
                load_kv(true, 0);
                for (int j = 1; j < k.n_kv; ++j) {
                    load_kv(false, j);
                    load_kv(true, j);
                }
            }
        } else if (warp == kWarpMma0 || warp == kWarpMma1) {
            // ===================== MMA issuer of tile t = warp - kWarpMma0 =====================
            const int t = warp - kWarpMma0;
            const uint32_t idesc_s =
                ptx::umma_idesc_bf16(BM, BS, false, false) | (negate_q ? (1u << 13) : 0u);
            constexpr uint32_t idesc_pv = ptx::umma_idesc_bf16(BM, D, false, true);
            const uint32_t tS = tmem + t * 128, tO = tmem + 256 + t * 128;
            const uint32_t q_smem = sQ + t * SL::kTileBytes;
            auto kv_wait = [&](uint32_t q) { ptx::mbar_wait(bar(kBarKvFull, slot_of(q)), phase_of(q)); };
            // S_t[b] = Q_t K[64 b, 64 b + 64)^T : both operands K-major (D contiguous), 128-byte swizzle
            // (descriptors of the k-th 16-wide slice = descriptor of the tile + a constant in the
            //  14-bit start-address field; tiles are 1024-byte aligned and < 256 KB, so no carry;
            //  64 key rows are 8 swizzle atoms = 8192 bytes further on)
            const uint64_t q_desc = ptx::umma_smem_desc_sw128(q_smem, 16, 1024);
            auto issue_qk = [&](uint32_t kslot, int b) {
                const uint64_t k_desc = ptx::umma_smem_desc_sw128(
                    sKV + kslot * SL::kTileBytes + b * (BS * 128), 16, 1024);
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk) {
                    constexpr int kBlk = SL::kBlockBytes;
                    const uint64_t off = (uint64_t)(((kk / 4) * kBlk + (kk % 4) * 32) >> 4);
                    ptx::umma_ss(tS + b * BS, q_desc + off, k_desc + off, idesc_s, kk > 0);
                }
            };
            // O_t (+)= P_t[b] V[64 b, 64 b + 64) : A = P_t[b] from tensor memory, B = V (MN-major)
            auto issue_pv = [&](uint32_t vslot, int b, bool accumulate) {
                const uint64_t v_desc =
                    ptx::umma_smem_desc_sw128(sKV + vslot * SL::kTileBytes, SL::kBlockBytes, 1024);
#pragma unroll
                for (int kk = 0; kk < BS / 16; ++kk)
                    ptx::umma_ts(tO, tS + b * BS + kk * 8,
                                 v_desc + (uint64_t)(((b * (BS / 16) + kk) * 2048) >> 4), idesc_pv,
                                 (accumulate || kk > 0) ? 1u : 0u);
            };
            // The tensor pipe runs MMAs in issue order.  With MOSAIC_MMA_LOCK an issuer holds this
            // lock while it issues one group of MMAs, so that the groups of the two tiles alternate
            // instead of interleaving instruction by instruction (off: see the file header).
            auto lock = [&]() {
#if MOSAIC_MMA_LOCK
                uint32_t old;
                do {
                    asm volatile("atom.shared.relaxed.cta.cas.b32 %0, [%1], 0, 1;"
                                 : "=r"(old) : "r"(mma_lock) : "memory");
                } while (old != 0);
#endif
            };
            auto unlock = [&]() {
#if MOSAIC_MMA_LOCK
                asm volatile("st.shared.relaxed.cta.u32 [%0], %1;" ::"r"(mma_lock), "r"(0u) : "memory");
#endif
            };
            // The whole warp walks the work list (uniform control flow keeps the descriptors in
            // uniform registers); one elected lane issues the MMAs and their commits.
            // Steps u = 2 j + b (KV tile j, half b) of an item use score buffer b.  The scores run
            // two steps ahead of the PVs:
            //   S(0) S(1) | PV(0) S(2) | PV(1) S(3) | ... | PV(U-2) | PV(U-1)
            // so S(u+2) overwrites P(u) right behind PV(u) in the (in-order) tensor pipe and is
            // ready, as a rule, before the softmax group has finished step u + 1.
            uint32_t pos = 0, ph_q = 0, ph_p = 0, ph_f = 0;
            uint32_t n_units = 0;
            for (Work k; next_unit(n_units, k);) {
                const int n_t = k.n(t);
                const uint32_t base = pos;
                if (n_t > 0) {
                    ptx::mbar_wait(bar(kBarQFull, t), ph_q);
                    ph_q ^= 1;
                    kv_wait(base);  // K_0
                    ptx::tc_fence_after();
                    if (ptx::elect_one()) {
                        lock();
                        issue_qk(slot_of(base), 0);
                        ptx::umma_commit(bar(kBarSFull, 2 * t));
                        issue_qk(slot_of(base), 1);
                        ptx::umma_commit(bar(kBarSFull, 2 * t + 1));
                        ptx::umma_commit(bar_kv_empty(t, slot_of(base)));
                        if (n_t == 1) ptx::umma_commit(bar(kBarQEmpty, t));
                        unlock();
                    }
                    __syncwarp();
                    for (int j = 0; j < n_t; ++j) {
                        const uint32_t vpos = base + 2 * j + 1, kpos = vpos + 1;  // V_j, K_{j+1}
                        const bool more = j + 1 < n_t;
                        kv_wait(vpos);
                        if (more) kv_wait(kpos);
                        if (j == 0) {  // PV_t(0) overwrites O_t: the epilogue of the previous item is done
                            ptx::mbar_wait(bar(kBarOFree, t), ph_f ^ 1);
                            ph_f ^= 1;
                        }
                        ptx::mbar_wait(bar(kBarPFull, 2 * t), ph_p);
                        ptx::tc_fence_after();
                        if (ptx::elect_one()) {
                            lock();
                            issue_pv(slot_of(vpos), 0, j > 0);
                            ptx::umma_commit(bar(kBarPvDone, t));
                            if (more) {
                                issue_qk(slot_of(kpos), 0);
                                ptx::umma_commit(bar(kBarSFull, 2 * t));
                            }
                            unlock();
                        }
                        __syncwarp();
                        ptx::mbar_wait(bar(kBarPFull, 2 * t + 1), ph_p);
                        ph_p ^= 1;
                        ptx::tc_fence_after();
                        if (ptx::elect_one()) {
                            lock();
                            issue_pv(slot_of(vpos), 1, true);
                            ptx::umma_commit(bar_kv_empty(t, slot_of(vpos)));
                            ptx::umma_commit(bar(kBarPvDone, t));
                            if (more) {
                                issue_qk(slot_of(kpos), 1);
                                ptx::umma_commit(bar(kBarSFull, 2 * t + 1));
                                ptx::umma_commit(bar_kv_empty(t, slot_of(kpos)));
                                if (j + 2 == n_t) ptx::umma_commit(bar(kBarQEmpty, t));
                            } else {
                                ptx::umma_commit(bar(kBarODone, t));
                            }
                            unlock();
                        }
                        __syncwarp();
                    }
                }
                // ring positions of this item that tile t does not use: consume and release
                pos = base + 2 * k.n_kv;
                for (uint32_t q = base + 2 * n_t; q < pos; ++q) {
                    kv_wait(q);
                    if (ptx::elect_one()) ptx::mbar_arrive(bar_kv_empty(t, slot_of(q)));
                    __syncwarp();
                }
            }
        }
    } else {
        // ============================ softmax + epilogue groups ===========================
        setmaxnreg_inc<208>();
        const int t = warp >> 2;                   // tile of this group (0 or 1)
        const int row = tid - t * BM;              // query row inside the tile == TMEM lane
        const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t tS = tmem + t * 128 + lane_off;        // score buffers of tile t, P_t in place
        const uint32_t tO = tmem + 256 + t * 128 + lane_off;  // O_t
        const int wq = warp & 3;                              // rows 32 wq .. 32 wq + 31 of the tile
        const float sc = p.scale_log2;
        uint32_t ph_s = 0, ph_f = 0;
        // l_run: the row sum of the un-rounded P (what the logsumexp needs).  l_fix: the rounding
        // residual bf16(p) - p of each step's LARGEST p.  O accumulates the bf16-rounded P, so its
        // normaliser should be the sum of the rounded values; summing those would cost three more
        // instructions per element pair, while correcting the step's top element is six per step
        // and removes the whole error exactly where it matters: a nearly one-hot row (sharp
        // softmax), where O = bf16(p_top) V / p_top was off by up to 2^-9 |V| -- with the running
        // max moved lazily p_top is anything in [1, 2^8], not 1.
        float m_used = 0.f, l_run = 0.f, l_fix = 0.f;
        int thr = 0;  // of the masked step in progress

        // One step: 64 scores of this row (buffer b) -> running max -> P (bf16, in place) -> row sum.
        //   kMask 0: no key masked   1: keys c > thr masked (thr = last key this row sees, relative
        //   to the step's first key)   2: every key masked (warp-uniform)
        // (Every call site is a copy of ~500 unrolled instructions and the instruction cache is
        //  small: the steady state gets one copy per buffer with b a constant, the two steps of
        //  the diagonal tile share one masked copy with b a run-time value.)
        auto step = [&](auto mask_kind, const int b, const bool first) {
            constexpr int kMask = decltype(mask_kind)::value;
            const uint32_t tSb = tS + b * BS;
            ptx::mbar_wait(bar(kBarSFull, 2 * t + b), ph_s);
            ptx::tc_fence_after();
            if constexpr (kMask == 2) {
                // rows 0-63 against keys 64-127 of the diagonal tile: P = 0
                uint32_t z[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) z[i] = 0u;
                ptx::tmem_st16(tSb, z);
                ptx::tmem_st16(tSb + 16, z);
            } else {
                // ---- A2: scores of this row, running max ---------------------------------------
                float s[BS];
#pragma unroll
                for (int c = 0; c < BS / 32; ++c)
                    ptx::tmem_ld32(tSb + c * 32, *reinterpret_cast<uint32_t(*)[32]>(&s[c * 32]));
                ptx::tmem_wait_ld();
                // kMask 1: thr does not decrease with the lane; when even the warp's last row sees
                // none of the step's second 32 keys their exponentials are skipped (P = 0)
                bool skip1 = false;
                if constexpr (kMask == 1) {
                    skip1 = __shfl_sync(0xffffffffu, thr, 31) < 32;
                    const int thr_lo = __shfl_sync(0xffffffffu, thr, 0);
                    if (thr_lo < 31) {  // (else every row of the warp sees the first 32 keys)
#pragma unroll
                        for (int c = 0; c < 32; ++c)
                            if (c > thr) s[c] = -INFINITY;
                    }
                    if (thr_lo < 63) {
#pragma unroll
                        for (int c = 32; c < BS; ++c)
                            if (c > thr) s[c] = -INFINITY;
                    }
                }
                float mx0 = s[0], mx1 = s[1], mx2 = s[2], mx3 = s[3];
#pragma unroll
                for (int c = 4; c < BS; c += 4) {
                    mx0 = fmaxf(mx0, s[c]);
                    mx1 = fmaxf(mx1, s[c + 1]);
                    mx2 = fmaxf(mx2, s[c + 2]);
                    mx3 = fmaxf(mx3, s[c + 3]);
                }
                const float mx = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3));
                const float m_new = mx * sc;
                if (first) {
                    // (a row that sees no key at all -- only against the contract, Lk < Lq -- keeps
                    //  a finite max, so that its masked scores give exp2(-inf) = 0, not NaN)
                    m_used = kMask == 1 ? fmaxf(m_new, -1e30f) : m_new;
                } else {
                    // move the max (and rescale l, O) only when it grew by more than 2^8
                    const bool need = m_new > m_used + kRescaleThreshold;
                    if (__any_sync(0xffffffffu, need)) {
                        // O_t must hold every PV up to the previous step (this one has not been
                        // issued: it needs the P written below).  The barrier has completed the
                        // phase before that one for certain (S of this step was issued behind it),
                        // so the parity of the previous step's phase is unambiguous: it is b ^ 1.
                        ptx::mbar_wait(bar(kBarPvDone, t), (uint32_t)(b ^ 1));
                        ptx::tc_fence_after();
                        const float alpha = need ? ex2_approx(m_used - m_new) : 1.f;
                        if (need) m_used = m_new;
                        l_run *= alpha;
                        l_fix *= alpha;
#pragma unroll 1  // rare: keep it small (instruction cache)
                        for (int c = 0; c < D / 16; ++c) {
                            uint32_t r[16];
                            ptx::tmem_ld16(tO + c * 16, r);
                            ptx::tmem_wait_ld();
#pragma unroll
                            for (int i = 0; i < 16; ++i)
                                r[i] = __float_as_uint(__uint_as_float(r[i]) * alpha);
                            ptx::tmem_st16(tO + c * 16, r);
                        }
                    }
                }
                // ---- P = exp2(s * scale_log2 - m), row sum, bf16 pairs into the score columns ----
                // Two elements at a time (packed fp32 FMA / ADD).  Of every four pairs, kPolyPairs
                // are exponentiated on the FMA pipe (exp2_poly2) and the rest on the MUFU unit
                // (16 results per clock per SM; DESIGN.md says why kPolyPairs is 0).
#ifndef MOSAIC_NO_TOP_FIX
                {   // the step's top element, by the same FMA and ex2 as in the loop below
                    float e_top = ex2_approx(fmaf(mx, sc, -m_used));
                    if constexpr (kMask == 1) e_top = mx == -INFINITY ? 0.f : e_top;
                    l_fix += __bfloat162float(__float2bfloat16_rn(e_top)) - e_top;
                }
#endif
                float2 la = make_float2(0.f, 0.f), lb = make_float2(0.f, 0.f);
                const float2 sc2 = make_float2(sc, sc), nm2 = make_float2(-m_used, -m_used);
#pragma unroll
                for (int c = 0; c < BS / 32; ++c) {
                    uint32_t pk[16];
                    if (kMask == 1 && c == 1 && skip1) {  // no row of the warp sees these 32 keys
#pragma unroll
                        for (int i = 0; i < 16; ++i) pk[i] = 0u;
                        ptx::tmem_st16(tSb + c * 16, pk);
                        continue;
                    }
#pragma unroll
                    for (int i = 0; i < 32; i += 2) {
                        const float x0 = s[c * 32 + i], x1 = s[c * 32 + i + 1];
                        float2 e;
                        {
                            // (a masked key is -inf and scale_log2 > 0 -- the host keeps it above
                            //  2^-100 even for softmax_scale = 0 -- so it gives exp2(-inf) = 0)
                            const float2 a = __ffma2_rn(make_float2(x0, x1), sc2, nm2);
                            if (((i >> 1) & 3) < kPolyPairs)
                                e = exp2_poly2(a);
                            else
                                e = make_float2(ex2_approx(a.x), ex2_approx(a.y));
                        }
                        if ((i >> 1) & 1)
                            lb = __fadd2_rn(lb, e);
                        else
                            la = __fadd2_rn(la, e);
                        __nv_bfloat162 h = __floats2bfloat162_rn(e.x, e.y);
                        pk[i / 2] = *reinterpret_cast<uint32_t*>(&h);
                    }
                    ptx::tmem_st16(tSb + c * 16, pk);
                }
                l_run += (la.x + la.y) + (lb.x + lb.y);
            }
            // P_t[b] is in tensor memory: hand it to the MMA issuer
            ptx::tmem_wait_st();
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar(kBarPFull, 2 * t + b));
        };
        using M0 = std::integral_constant<int, 0>;
        using M1 = std::integral_constant<int, 1>;
        using M2 = std::integral_constant<int, 2>;

        uint32_t n_units = 0;
        for (Work k; next_unit(n_units, k);) {
            const int n_t = k.n(t);
            if (n_t == 0) continue;  // this tile has no rows in this block
            m_used = 0.f;
            l_run = 0.f;
            l_fix = 0.f;
            // Row r of the sequence sees keys j <= r + off.  Steps whose 64 keys every row of the tile
            // sees run unmasked, in pairs (one copy per buffer); from the first step that some row of
            // the tile does not see in full, a warp's 32 rows x 64 keys are either masked altogether
            // or go through the masked copy with thr = r + off - 64 u (which masks nothing when
            // thr >= 63).  With off = 0 these are the two steps of the diagonal tile: untouched for
            // rows 64-127 at b = 0, masked altogether for rows 0-63 at b = 1, partly masked otherwise.
            const int tile_row0 = k.row0 + k.tile_of(t) * BM;  // first row of the tile in the sequence
            const int u_masked = ((min(tile_row0 + k.off, k.lk - 1) + 1) >> 6) & ~1;
            const int U = 2 * n_t;
            // (shared prefix: the two steps of its last tile hold prefix_pad - prefix_len padding
            //  keys, masked for every row; they lie before u_masked because every row sees the
            //  whole prefix)
            const int u_hole = p.prefix_len < p.prefix_pad ? 2 * (p.prefix_pad / BN - 1) : -1;
            for (int u = 0; u < u_masked; u += 2) {
                if (u == u_hole) {
                    thr = p.prefix_len - 1 - u * BS;  // >= 0: the tile holds at least one prefix key
                    step(M1{}, 0, u == 0);
                    thr -= BS;
                    if (thr < 0)
                        step(M2{}, 1, false);
                    else
                        step(M1{}, 1, false);
                } else {
                    step(M0{}, 0, u == 0);
                    step(M0{}, 1, false);
                }
                ph_s ^= 1;
            }
            for (int u = u_masked; u < U; ++u) {
                const int b = u & 1;
                thr = min(tile_row0 + row + k.off, k.lk - 1) - u * BS;
                if (min(tile_row0 + wq * 32 + 31 + k.off, k.lk - 1) - u * BS < 0)
                    step(M2{}, b, false);
                else
                    step(M1{}, b, u == 0);
                ph_s ^= (uint32_t)b;
            }
            // ---- hand the row's (logsumexp, 1 / normaliser) to the epilogue warps and go on to the next item -----------
            // (first make sure the epilogue has read the previous item's pair -- it releases O_t
            //  after that; an item of a single KV tile gets here without PV_t(0) having waited)
            ptx::mbar_wait(bar(kBarOFree, t), ph_f ^ 1);
            ph_f ^= 1;
            reinterpret_cast<float2*>(smem + SL::kStat)[t * BM + row] =
                make_float2((m_used + log2f(l_run)) * kLn2, 1.f / (l_run + l_fix));
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar(kBarStat, t));
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == kWarpMma1) ptx::tmem_dealloc<kTmemCols>(tmem);
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
                            const CUtensorMap& tkp, const CUtensorMap& tvp, const AttnParams& p, int negate_q, int grid, cudaStream_t s) {
    using SL = SmemLayout<D>;
    static bool configured = false;
    if (!configured) {
        MOSAIC_CUDA_TRY(cudaFuncSetAttribute(attn_fwd<D>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             SL::kDynamic));
        configured = true;
    }
    attn_fwd<D><<<grid, kThreadsAttn, SL::kDynamic, s>>>(tq, tk, tv, tkp, tvp, p, negate_q);
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

namespace mosaic {
// q rows and keys may be packed separately (cu_seqlens / total_tokens for q, O and LSE;
// cu_seqlens_k / total_k_tokens for K and V); the plain prefill passes the same for both.  With
// `desc` (device array of n_seqs views) the two cu arrays are not read.
mosaic_status_t attn_impl(const void* q, const void* k, const void* v, const int64_t* cu_seqlens,
                          const int64_t* cu_seqlens_k, const SeqDesc* desc, int32_t n_seqs,
                          int64_t total_tokens,
                          int64_t total_k_tokens, int32_t max_seqlen, int32_t Hq, int32_t Hkv,
                          int32_t D, float softmax_scale, int causal, void* o, float* lse,
                          void* workspace, size_t workspace_bytes, void* cuda_stream,
                          const void* k_prefix, const void* v_prefix, int32_t prefix_len) {
    if (prefix_len < 0 || (prefix_len > 0 && (!causal || !k_prefix || !v_prefix)))
        return MOSAIC_ERR_INVALID_ARG;
    if (n_seqs < 0 || total_tokens < 0 || total_tokens >= (1ll << 31) || total_k_tokens < 0 ||
        total_k_tokens >= (1ll << 31) || max_seqlen < 0 || Hq < 1 || Hkv < 1 || Hq % Hkv != 0 ||
        !isfinite(softmax_scale))
        return MOSAIC_ERR_INVALID_ARG;
    if (D != 64 && D != 128) return MOSAIC_ERR_UNSUPPORTED;
    if (n_seqs == 0 || total_tokens == 0) return MOSAIC_OK;
    if (!q || !k || !v || !o || !lse || (!desc && (!cu_seqlens || !cu_seqlens_k)) || !workspace ||
        !aligned16(q) ||
        !aligned16(k) || !aligned16(v) || !aligned16(o) || !aligned16(workspace))
        return MOSAIC_ERR_INVALID_ARG;
    Workspace w = carve(workspace, n_seqs, total_tokens);
    if (workspace_bytes < w.total_bytes) return MOSAIC_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);

    CUtensorMap tq, tk, tv;
    if (!make_tensor_map(&tq, q, total_tokens, Hq, D, BM) ||
        !make_tensor_map(&tk, k, total_k_tokens, Hkv, D, BN) ||
        !make_tensor_map(&tv, v, total_k_tokens, Hkv, D, BN))
        return MOSAIC_ERR_CUDA;
    CUtensorMap tkp = tk, tvp = tv;  // (never dereferenced without a prefix)
    if (prefix_len > 0 && (!make_tensor_map(&tkp, k_prefix, prefix_len, Hkv, D, BN) ||
                           !make_tensor_map(&tvp, v_prefix, prefix_len, Hkv, D, BN)))
        return MOSAIC_ERR_CUDA;

    const int levels = (int)(total_tokens / BQ) + 2;
    MOSAIC_CUDA_TRY(cudaMemsetAsync(workspace, 0, w.zero_bytes, s));
    schedule_kernel<<<1, 1024, 0, s>>>(cu_seqlens, cu_seqlens_k, desc, n_seqs, levels, w.header, w.cnt,
                                       w.start, w.cursor, w.rank, w.first, w.items, w.items_lk);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());

    AttnParams p{};
    p.cu_seqlens = cu_seqlens;
    p.items = w.items;
    p.items_lk = w.items_lk;
    p.header = w.header;
    p.o = static_cast<__nv_bfloat16*>(o);
    p.lse = lse;
    p.T = total_tokens;
    p.Hq = Hq;
    p.Hkv = Hkv;
    // (kept positive: a masked score is -inf and must stay -inf under the scale -- 0 x -inf is NaN;
    //  at 2^-100 every real score still scales to 0 to all fp32 digits, i.e. softmax_scale = 0)
    p.scale_log2 = fmaxf(fabsf(softmax_scale) * kLog2e, 7.8886091e-31f);
    p.inv_group = 1.0f / (float)(Hq / Hkv);
    p.group = Hq / Hkv;
    p.causal = causal ? 1 : 0;
    p.prefix_len = prefix_len;
    p.prefix_pad = (prefix_len + BN - 1) / BN * BN;
    p.o_align32 = (reinterpret_cast<uintptr_t>(o) & 31u) == 0 ? 1 : 0;
    const int negate_q = softmax_scale < 0.f ? 1 : 0;
    const int64_t max_work = (total_tokens / BQ + n_seqs) * (int64_t)Hq;
    if (max_work >= (1ll << 31)) return MOSAIC_ERR_UNSUPPORTED;
    const int grid = (int)(max_work < num_sms() ? max_work : num_sms());
    return D == 64 ? launch_attn<64>(tq, tk, tv, tkp, tvp, p, negate_q, grid, s)
                   : launch_attn<128>(tq, tk, tv, tkp, tvp, p, negate_q, grid, s);
}
}  // namespace mosaic

extern "C" mosaic_status_t mosaic_agg_prefill_attn(const void* q, const void* k, const void* v,
                                                   const int64_t* cu_seqlens, int32_t n_seqs,
                                                   int64_t total_tokens, int32_t max_seqlen,
                                                   int32_t Hq, int32_t Hkv, int32_t D,
                                                   float softmax_scale, void* o, float* lse,
                                                   void* workspace, size_t workspace_bytes,
                                                   void* cuda_stream) {
    return attn_impl(q, k, v, cu_seqlens, cu_seqlens, nullptr, n_seqs, total_tokens, total_tokens, max_seqlen,
                     Hq, Hkv, D, softmax_scale, 1, o, lse, workspace, workspace_bytes, cuda_stream);
}

extern "C" mosaic_status_t mosaic_agg_prefill_attn_kv(
    const void* q, const void* k, const void* v, const int64_t* cu_seqlens_q,
    const int64_t* cu_seqlens_k, int32_t n_seqs, int64_t total_q_tokens, int64_t total_k_tokens,
    int32_t max_seqlen_q, int32_t Hq, int32_t Hkv, int32_t D, float softmax_scale, int32_t causal,
    void* o, float* lse, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    return attn_impl(q, k, v, cu_seqlens_q, cu_seqlens_k, nullptr, n_seqs, total_q_tokens, total_k_tokens,
                     max_seqlen_q, Hq, Hkv, D, softmax_scale, causal, o, lse, workspace,
                     workspace_bytes, cuda_stream);
}
