// gate.cu -- step 1 of the confidence-gated aggregator stage (Sec. 4.2 P:L170-188,
// Alg. 1): per-question plurality vote, confidence, threshold, and the stream
// compaction of the surviving questions into a ragged batch with cu_seqlens.
//
// One kernel template serves the three C-ABI calls:
//   mosaic_gate          DO_GATE            -- thread per question, no ordering between blocks
//   mosaic_compact       DO_COMPACT         -- single-pass scan (decoupled look-back)
//   mosaic_gate_compact  DO_GATE|DO_COMPACT -- both in one pass over HBM
//
// HBM-bound.  A tile is kThreads x items questions in a striped
// arrangement (question = tile_base + item * kThreads + thread) so that a warp's loads and its
// compacted stores are both contiguous.  `items` is chosen on the host so that the whole grid is
// ONE wave of co-resident blocks (2 per SM) whenever Q allows: every block streams its rows
// (16- or 32-byte loads, several rows in flight per thread), keeps only (survived, ctx_len) per
// question in registers, and the scan costs one look-back round at the end of the block instead
// of one per small tile.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "common.cuh"

namespace mosaic {
namespace {

#ifndef MOSAIC_GATE_THREADS
#define MOSAIC_GATE_THREADS 256
#endif
constexpr int kThreads = MOSAIC_GATE_THREADS;
constexpr int kWarps = kThreads / 32;
constexpr int kMaxItems = 16;     // questions per thread, specialised E (<= 8)
constexpr int kMaxItemsWide = 4;  // ... generic E (<= 32): rows live in 2 x 32 registers
constexpr int kBlocksPerSM = 512 / kThreads;

using u64 = unsigned long long;

// Scan state of one tile, 16 bytes, written and read with single 128-bit accesses:
//   lo = status(2) | max ctx_len of survivors (31) | survivor count (31)
//   hi = status(2) | survivors' context tokens (62)
// status 0 = not written, 1 = this tile's aggregate, 2 = inclusive prefix over tiles 0..this.
// A reader accepts a pair only when both words carry the same non-zero status.
struct alignas(16) TileState {
    u64 lo, hi;
};
constexpr u64 kAggregate = 1ull << 62;
constexpr u64 kPrefix = 2ull << 62;
constexpr u64 kMask62 = (1ull << 62) - 1;
constexpr u64 kMask31 = (1ull << 31) - 1;

struct alignas(16) ScanHeader {
    unsigned int ticket;  // next tile id (tiles are handed out in start order)
    unsigned int pad[3];
};

struct Partial {  // the three scanned quantities
    u64 count, tokens;
    int max_len;
};

__device__ __forceinline__ u64 pack_lo(u64 status, const Partial& p) {
    return status | ((u64)(uint32_t)p.max_len << 31) | p.count;
}
__device__ __forceinline__ void ld_state(const TileState* s, u64& lo, u64& hi) {
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(lo), "=l"(hi) : "l"(s) : "memory");
}
__device__ __forceinline__ void st_state(TileState* s, u64 lo, u64 hi) {
    asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(s), "l"(lo), "l"(hi) : "memory");
}

// Programmatic dependent launch: the kernel that zeroes the scan workspace is launched just before
// this one and the two overlap; every thread that touches the workspace first waits here for the
// zeroing grid to have completed (and its writes to be visible).
__device__ __forceinline__ void wait_for_workspace() {
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

__global__ void __launch_bounds__(256) zero_workspace_kernel(uint4* p, size_t n16) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n16) p[i] = make_uint4(0u, 0u, 0u, 0u);
}

// Row loads.  Rows start 16-byte aligned when E % 4 == 0 (32-byte when E % 8 == 0) because the
// base pointer is; 32-byte rows use one 256-bit load, streamed past L1.
template <int E_T, int EM, typename T>
__device__ __forceinline__ void load_row(const T* __restrict__ base, int64_t q, int E, T (&r)[EM]) {
    static_assert(sizeof(T) == 4, "");
    if constexpr (E_T != 0 && E_T % 8 == 0) {
#pragma unroll
        for (int i = 0; i < E_T / 8; ++i) {
            uint32_t v[8];
            asm volatile("ld.global.nc.L1::no_allocate.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                         : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]),
                           "=r"(v[6]), "=r"(v[7])
                         : "l"(base + q * E_T + 8 * i));
#pragma unroll
            for (int j = 0; j < 8; ++j) r[8 * i + j] = reinterpret_cast<T&>(v[j]);
        }
    } else if constexpr (E_T != 0 && E_T % 4 == 0) {
        const int4* p = reinterpret_cast<const int4*>(base + q * E_T);
#pragma unroll
        for (int i = 0; i < E_T / 4; ++i) {
            int4 v = __ldg(p + i);
            r[4 * i + 0] = reinterpret_cast<T&>(v.x);
            r[4 * i + 1] = reinterpret_cast<T&>(v.y);
            r[4 * i + 2] = reinterpret_cast<T&>(v.z);
            r[4 * i + 3] = reinterpret_cast<T&>(v.w);
        }
    } else if constexpr (E_T != 0 && E_T % 2 == 0) {
        const int2* p = reinterpret_cast<const int2*>(base + q * E_T);
#pragma unroll
        for (int i = 0; i < E_T / 2; ++i) {
            int2 v = __ldg(p + i);
            r[2 * i + 0] = reinterpret_cast<T&>(v.x);
            r[2 * i + 1] = reinterpret_cast<T&>(v.y);
        }
    } else {
        const T* p = base + q * (int64_t)E;
#pragma unroll
        for (int i = 0; i < EM; ++i)
            if (i < E) r[i] = __ldg(p + i);
    }
}

// Sorting networks with the optimal comparator counts (1, 3, 5, 9, 12, 16, 19) for 2..8 labels.
__device__ __forceinline__ void cmp_swap(int32_t& x, int32_t& y) {
    const int32_t lo = min(x, y), hi = max(x, y);
    x = lo;
    y = hi;
}
template <int N>
__device__ __forceinline__ void sort_labels(int32_t (&s)[N]) {
    static_assert(N >= 1 && N <= 8, "");
    if constexpr (N == 2) {
        cmp_swap(s[0], s[1]);
    }
    if constexpr (N == 3) {
        cmp_swap(s[0], s[2]); cmp_swap(s[0], s[1]); cmp_swap(s[1], s[2]);
    }
    if constexpr (N == 4) {
        cmp_swap(s[0], s[2]); cmp_swap(s[1], s[3]); cmp_swap(s[0], s[1]); cmp_swap(s[2], s[3]);
        cmp_swap(s[1], s[2]);
    }
    if constexpr (N == 5) {
        cmp_swap(s[0], s[3]); cmp_swap(s[1], s[4]); cmp_swap(s[0], s[2]); cmp_swap(s[1], s[3]);
        cmp_swap(s[0], s[1]); cmp_swap(s[2], s[4]); cmp_swap(s[1], s[2]); cmp_swap(s[3], s[4]);
        cmp_swap(s[2], s[3]);
    }
    if constexpr (N == 6) {
        cmp_swap(s[0], s[5]); cmp_swap(s[1], s[3]); cmp_swap(s[2], s[4]); cmp_swap(s[1], s[2]);
        cmp_swap(s[3], s[4]); cmp_swap(s[0], s[3]); cmp_swap(s[2], s[5]); cmp_swap(s[0], s[1]);
        cmp_swap(s[2], s[3]); cmp_swap(s[4], s[5]); cmp_swap(s[1], s[2]); cmp_swap(s[3], s[4]);
    }
    if constexpr (N == 7) {
        cmp_swap(s[0], s[6]); cmp_swap(s[2], s[3]); cmp_swap(s[4], s[5]); cmp_swap(s[0], s[2]);
        cmp_swap(s[1], s[4]); cmp_swap(s[3], s[6]); cmp_swap(s[0], s[1]); cmp_swap(s[2], s[5]);
        cmp_swap(s[3], s[4]); cmp_swap(s[1], s[2]); cmp_swap(s[4], s[6]); cmp_swap(s[2], s[3]);
        cmp_swap(s[4], s[5]); cmp_swap(s[1], s[2]); cmp_swap(s[3], s[4]); cmp_swap(s[5], s[6]);
    }
    if constexpr (N == 8) {
        cmp_swap(s[0], s[2]); cmp_swap(s[1], s[3]); cmp_swap(s[4], s[6]); cmp_swap(s[5], s[7]);
        cmp_swap(s[0], s[4]); cmp_swap(s[1], s[5]); cmp_swap(s[2], s[6]); cmp_swap(s[3], s[7]);
        cmp_swap(s[0], s[1]); cmp_swap(s[2], s[3]); cmp_swap(s[4], s[5]); cmp_swap(s[6], s[7]);
        cmp_swap(s[2], s[4]); cmp_swap(s[3], s[5]); cmp_swap(s[1], s[4]); cmp_swap(s[3], s[6]);
        cmp_swap(s[1], s[2]); cmp_swap(s[3], s[4]); cmp_swap(s[5], s[6]);
    }
}

// Alg. 1 lines 2-4 for one question.  Same decisions, in the same precision, as
// the definition: c* = the largest number of equal labels, mode = smallest label among those
// reaching c* (reading G-2), agree = fl32(c*)/fl32(E) (one IEEE division, reading G-4), weighted
// share in binary64 in expert order (reading G-10), bypass = conf >= tau in fp32 (">=").
// SORTED (E known at compile time, <= 8): the labels go through a sorting network and the
// plurality is the longest run, first (= smallest label) run winning ties; otherwise every label
// is counted against every other.
template <int EM, int CONF, bool SORTED>
__device__ __forceinline__ void gate_row(const int32_t (&a)[EM], const float (&w)[EM], int E,
                                         float tau, int32_t& mode, int32_t& count, float& agree,
                                         float& conf, bool& bypass,
                                         const float* agree_lut = nullptr) {
    int32_t c_star = 0, md = 0;
    if constexpr (SORTED) {
        int32_t s[EM];
#pragma unroll
        for (int i = 0; i < EM; ++i) s[i] = a[i];
        sort_labels<EM>(s);
        int32_t run = 1;
        c_star = 1;
        md = s[0];
#pragma unroll
        for (int i = 1; i < EM; ++i) {
            run = (s[i] == s[i - 1]) ? run + 1 : 1;
            if (run > c_star) {
                c_star = run;
                md = s[i];
            }
        }
    } else {
#pragma unroll
        for (int i = 0; i < EM; ++i) {
            if (i < E) {
                int32_t n = 0;
#pragma unroll
                for (int j = 0; j < EM; ++j)
                    if (j < E) n += (a[j] == a[i]) ? 1 : 0;
                if (n > c_star || (n == c_star && a[i] < md)) {
                    c_star = n;
                    md = a[i];
                }
            }
        }
    }
    // agree_lut[c] holds the same IEEE division, done once per block
    agree = agree_lut ? agree_lut[c_star] : __fdiv_rn((float)c_star, (float)E);
    conf = agree;
    if constexpr (CONF == MOSAIC_CONF_WEIGHTED) {
        double sm = 0.0, st = 0.0;
#pragma unroll
        for (int i = 0; i < EM; ++i) {
            if (i < E) {
                const double wi = (double)w[i];
                st = __dadd_rn(st, wi);
                if (a[i] == md) sm = __dadd_rn(sm, wi);
            }
        }
        if (st > 0.0) conf = __double2float_rn(__ddiv_rn(sm, st));
    }
    mode = md;
    count = c_star;
    bypass = conf >= tau;
}

struct GateArgs {
    const int32_t* answers;
    const float* expert_conf;
    const uint8_t* bypass_in;  // compact-only
    const int32_t* ctx_len;
    int64_t Q;
    int32_t E;
    float tau;
    const float* tau_q;  // a threshold per question, else NULL: tau for all
    int32_t* mode_out;
    int32_t* count_out;
    float* agree_out;
    float* conf_out;
    uint8_t* bypass_out;
    int32_t* survivor_idx;
    int64_t* cu_seqlens;
    int32_t* n_survivors;
    int64_t* total_tokens;
    int32_t* max_seqlen;
    ScanHeader* header;
    TileState* tiles;
    int use_ticket;   // tiles numbered by an atomic ticket (grids of more than one wave), else by blockIdx
    int tile_stride;  // tile t lives at tiles[t * tile_stride]: one state per 128-byte line when the
                      // workspace allows, so the look-back loads of ~300 tiles spread over the L2 slices
    unsigned int num_tiles;
    int items;  // questions per thread in this launch
};

// Combined (count, tokens, max) of the tiles before `tile` (decoupled look-back).  Warp 0 walks
// the predecessors 256 at a time, 8 per lane, nearest first: each lane adds its entries up to and
// including its first inclusive prefix; lanes before the first lane that met a prefix count in
// full, that lane counts its partial sum, later lanes do not count.  With the grid a single wave
// of <= 296 tiles this is one round of loads.  Whole warp calls; result in every lane.
__device__ __forceinline__ Partial look_back(const TileState* tiles, int stride, int tile, int lane) {
    constexpr int W = 8;
    Partial acc{0, 0, 0};
    bool done = false;
    for (int base = tile - 1; !done; base -= 32 * W) {
        u64 lo[W], hi[W];
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const int idx = base - (lane * W + j);
            lo[j] = hi[j] = idx >= 0 ? 0ull : kPrefix;  // "tile -1": prefix of nothing
        }
        // (re)load every entry that is not published yet, all of them in flight together: one
        // L2 round trip per pass, however many entries were late
        bool pending;
        do {
#pragma unroll
            for (int j = 0; j < W; ++j) {
                const int idx = base - (lane * W + j);
                const bool ready = (lo[j] >> 62) != 0 && (lo[j] >> 62) == (hi[j] >> 62);
                if (!ready) ld_state(tiles + (size_t)idx * stride, lo[j], hi[j]);
            }
            pending = false;
#pragma unroll
            for (int j = 0; j < W; ++j)
                pending |= (lo[j] >> 62) == 0 || (lo[j] >> 62) != (hi[j] >> 62);
        } while (__any_sync(0xffffffffu, pending));
        Partial mine{0, 0, 0};
        bool met = false;
#pragma unroll
        for (int j = 0; j < W; ++j) {
            if (!met) {
                mine.count += lo[j] & kMask31;
                mine.tokens += hi[j] & kMask62;
                mine.max_len = max(mine.max_len, (int)((lo[j] >> 31) & kMask31));
                met = (lo[j] >> 62) == 2;
            }
        }
        __syncwarp();
        const unsigned pm = __ballot_sync(0xffffffffu, met);
        const int first = pm ? (__ffs(pm) - 1) : 31;
        if (lane > first) mine = Partial{0, 0, 0};
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            mine.count += __shfl_xor_sync(0xffffffffu, mine.count, o);
            mine.tokens += __shfl_xor_sync(0xffffffffu, mine.tokens, o);
            mine.max_len = max(mine.max_len, __shfl_xor_sync(0xffffffffu, mine.max_len, o));
        }
        acc.count += mine.count;
        acc.tokens += mine.tokens;
        acc.max_len = max(acc.max_len, mine.max_len);
        done = pm != 0;
    }
    return acc;
}

// Shared memory of one block: per-question (survived ? ctx_len : -1) in striped order, and the
// per-(item, warp) partials of the scan.
template <int MAXI>
struct GateSmem {
    int len[MAXI * kThreads];
    unsigned int part_count[MAXI * kWarps];  // survivors of (item, warp)  -> exclusive offsets
    u64 part_tokens[MAXI * kWarps];          // their context tokens       -> exclusive offsets
    u64 base_count, base_tokens;             // the tile's exclusive prefix
    int warp_max[kWarps];
    unsigned int tile;
};

// G4-G5 for one tile, after every thread has recorded (survived ? ctx_len : -1) for its questions
// in sm.len (striped: question = q0 + item * kThreads + thread) and the per-(item, warp) partials:
// block scan, one look-back round for the tile's exclusive prefix, stable scatter of the survivors.
template <int MAXI>
__device__ __forceinline__ void compact_tile(const GateArgs& p, GateSmem<MAXI>& sm, unsigned int tile,
                                             int64_t q0, int items, int my_max) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // ---- G4-G5: stable compaction and cu_seqlens -------------------------------------------
    // Scan order inside the tile is (item, thread): exactly ascending question index.
    my_max = __reduce_max_sync(0xffffffffu, my_max);
    if (lane == 0) sm.warp_max[warp] = my_max;
    __syncthreads();

    // (the last warp: the warp scheduler favours the highest warp id, and this warp is what the
    //  whole tile -- and every later tile -- waits for)
    if (warp == kWarps - 1) {
        // exclusive scan of the items * kWarps (<= 128) partials, 4 consecutive per lane
        constexpr int PER = (MAXI * kWarps + 31) / 32;
        const int n_part = items * kWarps;
        unsigned int c[PER];
        u64 t[PER];
        unsigned int csum = 0;
        u64 tsum = 0;
#pragma unroll
        for (int j = 0; j < PER; ++j) {
            const int e = lane * PER + j;
            c[j] = e < n_part ? sm.part_count[e] : 0u;
            t[j] = e < n_part ? sm.part_tokens[e] : 0ull;
            csum += c[j];
            tsum += t[j];
        }
        unsigned int ci = csum;
        u64 ti = tsum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned int cc = __shfl_up_sync(0xffffffffu, ci, o);
            const u64 tt = __shfl_up_sync(0xffffffffu, ti, o);
            if (lane >= o) {
                ci += cc;
                ti += tt;
            }
        }
        unsigned int cx = ci - csum;
        u64 tx = ti - tsum;
#pragma unroll
        for (int j = 0; j < PER; ++j) {
            const int e = lane * PER + j;
            if (e < n_part) {
                sm.part_count[e] = cx;
                sm.part_tokens[e] = tx;
            }
            cx += c[j];
            tx += t[j];
        }
        Partial mine;
        mine.count = __shfl_sync(0xffffffffu, ci, 31);
        mine.tokens = __shfl_sync(0xffffffffu, ti, 31);
        mine.max_len = __reduce_max_sync(0xffffffffu, lane < kWarps ? sm.warp_max[lane] : 0);

        wait_for_workspace();  // (returns at once when the zeroing grid is already complete)
        TileState* me = p.tiles + (size_t)tile * p.tile_stride;
        Partial before{0, 0, 0};
        if (tile != 0) {
            if (lane == 0) st_state(me, pack_lo(kAggregate, mine), kAggregate | mine.tokens);
            before = look_back(p.tiles, p.tile_stride, (int)tile, lane);
        }
        Partial incl{before.count + mine.count, before.tokens + mine.tokens,
                     max(before.max_len, mine.max_len)};
        if (lane == 0) {
            st_state(me, pack_lo(kPrefix, incl), kPrefix | incl.tokens);
            sm.base_count = before.count;
            sm.base_tokens = before.tokens;
            if (tile == 0) p.cu_seqlens[0] = 0;
            if (tile == p.num_tiles - 1) {
                *p.n_survivors = (int32_t)incl.count;
                *p.total_tokens = (int64_t)incl.tokens;
                *p.max_seqlen = incl.max_len;
            }
        }
    }
    __syncthreads();

    // Four items at a time so that their (independent) warp scans overlap.
    const u64 base_c = sm.base_count, base_t = sm.base_tokens;
    constexpr int U = 4;
    for (int k0 = 0; k0 < items; k0 += U) {
        int v[U];
        unsigned ballot[U];
        uint32_t x[U];
        uint32_t mx = 0;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            v[u] = (k0 + u < items) ? sm.len[(k0 + u) * kThreads + tid] : -1;
            ballot[u] = __ballot_sync(0xffffffffu, v[u] >= 0);
            x[u] = v[u] >= 0 ? (uint32_t)v[u] : 0u;
            mx = max(mx, x[u]);
        }
        const bool small = __reduce_max_sync(0xffffffffu, mx) < (1u << 26);  // 32 lanes cannot overflow
        u64 incl[U];
        if (small) {
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const uint32_t y = __shfl_up_sync(0xffffffffu, x[u], o);
                    if (lane >= o) x[u] += y;
                }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) incl[u] = x[u];
        } else {
#pragma unroll
            for (int u = 0; u < U; ++u) {
                u64 z = x[u];
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const u64 y = __shfl_up_sync(0xffffffffu, z, o);
                    if (lane >= o) z += y;
                }
                incl[u] = z;
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (v[u] >= 0) {
                const int k = k0 + u;
                const unsigned rank = __popc(ballot[u] & ((1u << lane) - 1u));
                const u64 r = base_c + sm.part_count[k * kWarps + warp] + rank;
                p.survivor_idx[r] = (int32_t)(q0 + (int64_t)k * kThreads + tid);
                p.cu_seqlens[r + 1] = (int64_t)(base_t + sm.part_tokens[k * kWarps + warp] + incl[u]);
            }
        }
    }
}

template <int E_T, int CONF, bool DO_GATE, bool DO_COMPACT, int MAXI, int BATCH>
__global__ void __launch_bounds__(kThreads, kBlocksPerSM) gate_compact_kernel(const GateArgs p) {
    constexpr int EM = DO_GATE ? (E_T ? E_T : MOSAIC_MAX_EXPERTS) : 1;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int E = E_T ? E_T : p.E;
    const int items = p.items;

    __shared__ GateSmem<DO_COMPACT ? MAXI : 1> sm;

    unsigned int tile = blockIdx.x;
    if constexpr (DO_COMPACT) {
        if (tid == 0) {
            if (p.use_ticket) {
                wait_for_workspace();
                sm.tile = atomicAdd(&p.header->ticket, 1u);
            } else {
                sm.tile = blockIdx.x;
            }
        }
        __syncthreads();
        tile = sm.tile;
    }
    const int64_t q0 = (int64_t)tile * kThreads * items;
    int my_max = 0;

    // ---- G1-G3 (vote, confidence, threshold), BATCH questions per thread in flight ---------------
    for (int it0 = 0; it0 < items; it0 += BATCH) {
        bool valid[BATCH], surv[BATCH];
        int32_t len[BATCH];
        if constexpr (DO_GATE) {
            int32_t a[BATCH][EM];
            float w[BATCH][EM];
#pragma unroll
            for (int k = 0; k < BATCH; ++k) {
                const int64_t q = q0 + (int64_t)(it0 + k) * kThreads + tid;
                valid[k] = (it0 + k < items) && (q < p.Q);
                if (valid[k]) {
                    load_row<E_T, EM>(p.answers, q, E, a[k]);
                    if constexpr (CONF == MOSAIC_CONF_WEIGHTED)
                        load_row<E_T, EM>(p.expert_conf, q, E, w[k]);
                    if constexpr (DO_COMPACT) len[k] = __ldg(p.ctx_len + q);
                }
            }
#pragma unroll
            for (int k = 0; k < BATCH; ++k) {
                const int64_t q = q0 + (int64_t)(it0 + k) * kThreads + tid;
                surv[k] = false;
                if (valid[k]) {
                    int32_t mode, count;
                    float agree, conf;
                    bool bypass;
                    gate_row<EM, CONF, (E_T != 0)>(a[k], w[k], E, p.tau_q ? __ldg(p.tau_q + q) : p.tau, mode,
                                                   count, agree, conf, bypass);
                    if (p.mode_out) __stcs(p.mode_out + q, mode);
                    if (p.count_out) __stcs(p.count_out + q, count);
                    if (p.agree_out) __stcs(p.agree_out + q, agree);
                    if (p.conf_out) __stcs(p.conf_out + q, conf);
                    if (p.bypass_out) p.bypass_out[q] = bypass ? 1 : 0;
                    surv[k] = !bypass;
                }
            }
        } else {
#pragma unroll
            for (int k = 0; k < BATCH; ++k) {
                const int64_t q = q0 + (int64_t)(it0 + k) * kThreads + tid;
                valid[k] = (it0 + k < items) && (q < p.Q);
                surv[k] = valid[k] ? (__ldg(p.bypass_in + q) == 0) : false;
                len[k] = valid[k] ? __ldg(p.ctx_len + q) : 0;
            }
        }
        if constexpr (DO_COMPACT) {
            // per-(item, warp) partials: survivors, their tokens (two 16-bit-half reductions so the
            // 32-lane sums cannot overflow 32 bits), max length
#pragma unroll
            for (int k = 0; k < BATCH; ++k) {
                if (it0 + k < items) {
                    const uint32_t v = surv[k] ? (uint32_t)len[k] : 0u;
                    sm.len[(it0 + k) * kThreads + tid] = surv[k] ? len[k] : -1;
                    const unsigned ballot = __ballot_sync(0xffffffffu, surv[k]);
                    const uint32_t lo = __reduce_add_sync(0xffffffffu, v & 0xffffu);
                    const uint32_t hi = __reduce_add_sync(0xffffffffu, v >> 16);
                    my_max = max(my_max, (int)v);
                    if (lane == 0) {
                        sm.part_count[(it0 + k) * kWarps + warp] = __popc(ballot);
                        sm.part_tokens[(it0 + k) * kWarps + warp] = (u64)lo + ((u64)hi << 16);
                    }
                }
            }
        }
    }

    if constexpr (DO_COMPACT) compact_tile<MAXI>(p, sm, tile, q0, items, my_max);
}

// Questions per thread: as many as needed for the grid to be one co-resident wave
// (kBlocksPerSM blocks per SM), capped by what a block keeps in shared memory.
inline int choose_items(int64_t Q, int max_items) {
    const int64_t wave = (int64_t)num_sms() * kBlocksPerSM * kThreads;
    int64_t items = (Q + wave - 1) / wave;
    if (items < 1) items = 1;
    if (items > max_items) items = max_items;
    return (int)items;
}

template <int E_T, int CONF, bool DO_GATE, bool DO_COMPACT, int MAXI, int BATCH>
mosaic_status_t launch(GateArgs& a, size_t ws_bytes, void* workspace, cudaStream_t stream) {
    a.items = choose_items(a.Q, MAXI);
    const int64_t tile = (int64_t)kThreads * a.items;
    const unsigned int tiles = (unsigned int)((a.Q + tile - 1) / tile);
    a.num_tiles = tiles;
    if constexpr (DO_COMPACT) {
        int stride = 8;  // 128-byte lines if the workspace holds them, else denser
        while (stride > 1 && sizeof(ScanHeader) + (size_t)tiles * stride * sizeof(TileState) > ws_bytes)
            stride >>= 1;
        a.tile_stride = stride;
        const size_t need = sizeof(ScanHeader) + (size_t)tiles * stride * sizeof(TileState);
        if (ws_bytes < need) return MOSAIC_ERR_WORKSPACE_TOO_SMALL;
        a.header = static_cast<ScanHeader*>(workspace);
        a.tiles = reinterpret_cast<TileState*>(static_cast<char*>(workspace) + sizeof(ScanHeader));
        // One co-resident wave: tile = blockIdx (blocks are dispatched in index order, so a tile
        // only ever waits for tiles that are already running) and the workspace is first touched
        // after the streaming phase, which therefore overlaps its zeroing.  Larger grids take a
        // ticket at block start instead, and wait for the zeroing there.
        a.use_ticket = tiles > (unsigned)(num_sms() * kBlocksPerSM) ? 1 : 0;
        const size_t n16 = (need + 15) / 16;
        zero_workspace_kernel<<<(unsigned)((n16 + 255) / 256), 256, 0, stream>>>(
            static_cast<uint4*>(workspace), n16);
        count_launch();
        MOSAIC_CUDA_TRY(cudaGetLastError());
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(tiles);
        cfg.blockDim = dim3(kThreads);
        cfg.dynamicSmemBytes = 0;
        cfg.stream = stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        MOSAIC_CUDA_TRY(cudaLaunchKernelEx(
            &cfg, gate_compact_kernel<E_T, CONF, DO_GATE, DO_COMPACT, MAXI, BATCH>, a));
        count_launch();
        return MOSAIC_OK;
    }
    gate_compact_kernel<E_T, CONF, DO_GATE, DO_COMPACT, MAXI, BATCH>
        <<<tiles, kThreads, 0, stream>>>(a);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());
    return MOSAIC_OK;
}

template <int CONF, bool DO_COMPACT>
mosaic_status_t dispatch_gate(GateArgs& a, size_t ws_bytes, void* ws, cudaStream_t s) {
    constexpr int M = kMaxItems;
    switch (a.E) {
        case 1: return launch<1, CONF, true, DO_COMPACT, M, 4>(a, ws_bytes, ws, s);
        case 2: return launch<2, CONF, true, DO_COMPACT, M, 4>(a, ws_bytes, ws, s);
        case 3: return launch<3, CONF, true, DO_COMPACT, M, 4>(a, ws_bytes, ws, s);
        case 4: return launch<4, CONF, true, DO_COMPACT, M, 4>(a, ws_bytes, ws, s);
        case 5: return launch<5, CONF, true, DO_COMPACT, M, 4>(a, ws_bytes, ws, s);
        case 6: return launch<6, CONF, true, DO_COMPACT, M, 4>(a, ws_bytes, ws, s);
        case 7: return launch<7, CONF, true, DO_COMPACT, M, 4>(a, ws_bytes, ws, s);
        case 8: return launch<8, CONF, true, DO_COMPACT, M, 4>(a, ws_bytes, ws, s);
        default: return launch<0, CONF, true, DO_COMPACT, kMaxItemsWide, 1>(a, ws_bytes, ws, s);
    }
}

mosaic_status_t check_gate_args(const int32_t* answers, const float* expert_conf, int64_t Q,
                                int32_t E, float tau, int32_t conf_mode) {
    if (Q < 0 || Q >= (1ll << 31) || E < 1 || E > MOSAIC_MAX_EXPERTS || isnan(tau))
        return MOSAIC_ERR_INVALID_ARG;
    if (conf_mode != MOSAIC_CONF_VOTE && conf_mode != MOSAIC_CONF_WEIGHTED)
        return MOSAIC_ERR_INVALID_ARG;
    if (Q > 0) {
        if (!answers || !aligned16(answers)) return MOSAIC_ERR_INVALID_ARG;
        if (conf_mode == MOSAIC_CONF_WEIGHTED && (!expert_conf || !aligned16(expert_conf)))
            return MOSAIC_ERR_INVALID_ARG;
        // 32-byte rows are read with 256-bit loads
        if (E % 8 == 0 && E <= 8 &&
            ((reinterpret_cast<uintptr_t>(answers) & 31u) ||
             (conf_mode == MOSAIC_CONF_WEIGHTED && (reinterpret_cast<uintptr_t>(expert_conf) & 31u))))
            return MOSAIC_ERR_INVALID_ARG;
    }
    return MOSAIC_OK;
}

mosaic_status_t write_empty_batch(int64_t* cu_seqlens, int32_t* n_survivors, int64_t* total_tokens,
                                  int32_t* max_seqlen, cudaStream_t s) {
    MOSAIC_CUDA_TRY(cudaMemsetAsync(cu_seqlens, 0, sizeof(int64_t), s));
    MOSAIC_CUDA_TRY(cudaMemsetAsync(n_survivors, 0, sizeof(int32_t), s));
    MOSAIC_CUDA_TRY(cudaMemsetAsync(total_tokens, 0, sizeof(int64_t), s));
    MOSAIC_CUDA_TRY(cudaMemsetAsync(max_seqlen, 0, sizeof(int32_t), s));
    return MOSAIC_OK;
}

}  // namespace
}  // namespace mosaic

using namespace mosaic;

extern "C" mosaic_status_t mosaic_gate(const int32_t* answers, const float* expert_conf, int64_t Q,
                                       int32_t E, float tau, int32_t conf_mode, int32_t* mode_out,
                                       int32_t* count_out, float* agree_out, float* conf_out,
                                       uint8_t* bypass_out, void* cuda_stream) {
    mosaic_status_t st = check_gate_args(answers, expert_conf, Q, E, tau, conf_mode);
    if (st != MOSAIC_OK) return st;
    if (Q == 0) return MOSAIC_OK;
    if (!bypass_out) return MOSAIC_ERR_INVALID_ARG;
    GateArgs a{};
    a.answers = answers;
    a.expert_conf = expert_conf;
    a.Q = Q;
    a.E = E;
    a.tau = tau;
    a.mode_out = mode_out;
    a.count_out = count_out;
    a.agree_out = agree_out;
    a.conf_out = conf_out;
    a.bypass_out = bypass_out;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    return conf_mode == MOSAIC_CONF_WEIGHTED
               ? dispatch_gate<MOSAIC_CONF_WEIGHTED, false>(a, 0, nullptr, s)
               : dispatch_gate<MOSAIC_CONF_VOTE, false>(a, 0, nullptr, s);
}

extern "C" size_t mosaic_compact_workspace_bytes(int64_t Q) {
    if (Q < 0) return 0;
    // worst case: one question per thread (small Q) -> Q / kThreads tiles
    const size_t tiles = (size_t)((Q + kThreads - 1) / kThreads);
    return sizeof(ScanHeader) + (tiles + 1) * sizeof(TileState);
}

extern "C" mosaic_status_t mosaic_compact(const uint8_t* bypass, const int32_t* ctx_len, int64_t Q,
                                          int32_t* survivor_idx, int64_t* cu_seqlens,
                                          int32_t* n_survivors, int64_t* total_tokens,
                                          int32_t* max_seqlen, void* workspace,
                                          size_t workspace_bytes, void* cuda_stream) {
    if (Q < 0 || Q >= (1ll << 31) || !cu_seqlens || !n_survivors || !total_tokens || !max_seqlen)
        return MOSAIC_ERR_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    if (Q == 0) return write_empty_batch(cu_seqlens, n_survivors, total_tokens, max_seqlen, s);
    if (!bypass || !ctx_len || !survivor_idx || !workspace || !aligned16(workspace))
        return MOSAIC_ERR_INVALID_ARG;
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
    return launch<1, MOSAIC_CONF_VOTE, false, true, kMaxItems, 4>(a, workspace_bytes, workspace, s);
}

extern "C" mosaic_status_t mosaic_gate_compact(
    const int32_t* answers, const float* expert_conf, const int32_t* ctx_len, int64_t Q, int32_t E,
    float tau, int32_t conf_mode, int32_t* mode_out, int32_t* count_out, float* agree_out,
    float* conf_out, uint8_t* bypass_out, int32_t* survivor_idx, int64_t* cu_seqlens,
    int32_t* n_survivors, int64_t* total_tokens, int32_t* max_seqlen, void* workspace,
    size_t workspace_bytes, void* cuda_stream) {
    mosaic_status_t st = check_gate_args(answers, expert_conf, Q, E, tau, conf_mode);
    if (st != MOSAIC_OK) return st;
    if (!cu_seqlens || !n_survivors || !total_tokens || !max_seqlen) return MOSAIC_ERR_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    if (Q == 0) return write_empty_batch(cu_seqlens, n_survivors, total_tokens, max_seqlen, s);
    if (!ctx_len || !survivor_idx || !workspace || !aligned16(workspace))
        return MOSAIC_ERR_INVALID_ARG;
    GateArgs a{};
    a.answers = answers;
    a.expert_conf = expert_conf;
    a.ctx_len = ctx_len;
    a.Q = Q;
    a.E = E;
    a.tau = tau;
    a.mode_out = mode_out;
    a.count_out = count_out;
    a.agree_out = agree_out;
    a.conf_out = conf_out;
    a.bypass_out = bypass_out;
    a.survivor_idx = survivor_idx;
    a.cu_seqlens = cu_seqlens;
    a.n_survivors = n_survivors;
    a.total_tokens = total_tokens;
    a.max_seqlen = max_seqlen;
    return conf_mode == MOSAIC_CONF_WEIGHTED
               ? dispatch_gate<MOSAIC_CONF_WEIGHTED, true>(a, workspace_bytes, workspace, s)
               : dispatch_gate<MOSAIC_CONF_VOTE, true>(a, workspace_bytes, workspace, s);
}

extern "C" mosaic_status_t mosaic_gate_compact_tau(
    const int32_t* answers, const float* expert_conf, const int32_t* ctx_len, int64_t Q, int32_t E,
    const float* tau_per_query, int32_t conf_mode, int32_t* mode_out, int32_t* count_out, float* agree_out,
    float* conf_out, uint8_t* bypass_out, int32_t* survivor_idx, int64_t* cu_seqlens,
    int32_t* n_survivors, int64_t* total_tokens, int32_t* max_seqlen, void* workspace,
    size_t workspace_bytes, void* cuda_stream) {
    mosaic_status_t st = check_gate_args(answers, expert_conf, Q, E, 0.5f, conf_mode);
    if (st == MOSAIC_OK && Q > 0 && !tau_per_query) st = MOSAIC_ERR_INVALID_ARG;
    if (st != MOSAIC_OK) return st;
    if (!cu_seqlens || !n_survivors || !total_tokens || !max_seqlen) return MOSAIC_ERR_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    if (Q == 0) return write_empty_batch(cu_seqlens, n_survivors, total_tokens, max_seqlen, s);
    if (!ctx_len || !survivor_idx || !workspace || !aligned16(workspace))
        return MOSAIC_ERR_INVALID_ARG;
    GateArgs a{};
    a.answers = answers;
    a.expert_conf = expert_conf;
    a.ctx_len = ctx_len;
    a.Q = Q;
    a.E = E;
    a.tau = 0.f;
    a.tau_q = tau_per_query;
    a.mode_out = mode_out;
    a.count_out = count_out;
    a.agree_out = agree_out;
    a.conf_out = conf_out;
    a.bypass_out = bypass_out;
    a.survivor_idx = survivor_idx;
    a.cu_seqlens = cu_seqlens;
    a.n_survivors = n_survivors;
    a.total_tokens = total_tokens;
    a.max_seqlen = max_seqlen;
    return conf_mode == MOSAIC_CONF_WEIGHTED
               ? dispatch_gate<MOSAIC_CONF_WEIGHTED, true>(a, workspace_bytes, workspace, s)
               : dispatch_gate<MOSAIC_CONF_VOTE, true>(a, workspace_bytes, workspace, s);
}


