// compact_kernel.cuh -- (included by compact.cu and the compact_inst_*.cu instantiation units)
// compact.cu -- the gate fused with the stream compaction of the surviving questions into a ragged
// batch with cu_seqlens (Alg. 1: line 6 sends the questions that failed the
// gate to the aggregator; BASELINE.json north_star: "stream-compacts the surviving queries into a
// ragged batch with cu_seqlens").  One kernel template serves
//   mosaic_gate_compact[_tau|_ext]  kSrcAnswers : Alg. 1 lines 2-4 + compaction in ONE pass over HBM
//   mosaic_compact                  kSrcBypass  : compaction of a mask computed earlier
//   mosaic_conf_compact             kSrcConf    : threshold on a caller-supplied C(q) + compaction
//
// HBM-bound.  The grid is persistent (a few blocks per SM); a block takes
// tiles of kVoters x T questions by atomic ticket (striped: question = tile_base + item *
// kVoters + thread, so a warp's loads and its compacted stores are contiguous).  Per tile:
// vote -> (survived, ctx_len) in shared memory and the tile's aggregate -> single-pass decoupled
// look-back for the tile's exclusive prefix -> stable scatter.  Eight "voter" warps stream, vote and
// scatter; a ninth "scanner" warp does the scan and the look-back, and the scatter of a tile lags
// its vote by one tile, so the HBM stream does not stop for the scan (the first version streamed
// everything, then scanned, then scattered: 55 % of the copy bandwidth at 2^20 questions).
//
// The scan state lives in the caller's workspace, whose contents are arbitrary: a small kernel
// zeroes it and the scan kernel overlaps that kernel through programmatic dependent launch.
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <type_traits>

#include "common.cuh"
#include "gate_row.cuh"

namespace mosaic {

// Scan state of one tile, 16 bytes, written and read with single 128-bit accesses:
//   lo = status(2) | max ctx_len of survivors (31) | survivor count (31)
//   hi = status(2) | survivors' context tokens (62)
// status 0 = not published, 1 = this tile's aggregate, 2 = inclusive prefix over tiles 0..this.
// A reader accepts a pair only when both words carry the same non-zero status.
struct alignas(16) TileState {
    u64 lo, hi;
};

struct alignas(128) ScanHeader {
    unsigned int ticket;  // next tile index (tiles are handed out in start order)
};

namespace {

#ifndef MOSAIC_GATE_VOTER_WARPS
#define MOSAIC_GATE_VOTER_WARPS 7
#endif
constexpr int kVoterWarps = MOSAIC_GATE_VOTER_WARPS;  // warps of a block that stream, vote and scatter
constexpr int kVoters = 32 * kVoterWarps;            // (one more warp scans)
#ifndef MOSAIC_GATE_WINDOW
#define MOSAIC_GATE_WINDOW 8
#endif
#ifndef MOSAIC_GATE_BACKOFF_NS
#define MOSAIC_GATE_BACKOFF_NS 200
#endif
constexpr int kMinTileQuestions = kVoters;   // the smallest tile any instantiation uses

constexpr u64 kAggregate = 1ull << 62;
constexpr u64 kPrefix = 2ull << 62;
constexpr u64 kMask62 = (1ull << 62) - 1;
constexpr u64 kMask31 = (1ull << 31) - 1;

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

// Combined (count, tokens, max) of the tiles before `tile` (decoupled look-back).  One warp walks
// the predecessors 256 at a time, 8 per lane, nearest first: each lane adds its entries up to and
// including its first inclusive prefix; lanes before the first lane that met a prefix count in
// full, that lane counts its partial sum, later lanes do not count.  Whole warp calls; result in
// every lane.  A tile only ever waits for tiles of smaller index, and all blocks are co-resident
// and take their tiles in increasing order, so the wait always ends.
__device__ __forceinline__ Partial look_back(const TileState* tiles, int stride, int tile, int lane) {
    constexpr int W = MOSAIC_GATE_WINDOW;
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
            pending = __any_sync(0xffffffffu, pending);
            // Back off before polling again: a spinning warp takes issue slots from the voters of
            // its scheduler and keeps ~300 scanners hammering the same few hundred L2 lines.
            if (pending) __nanosleep(MOSAIC_GATE_BACKOFF_NS);
        } while (pending);
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

#ifndef MOSAIC_GATE_MAXT
#define MOSAIC_GATE_MAXT 8
#endif
constexpr int kMaxT = MOSAIC_GATE_MAXT;  // items (questions per thread) of one tile, at most

// Shared memory of one block, double-buffered over the block's consecutive tiles: per-question
// (survived ? ctx_len : -1) in striped order, and the per-(item, warp) partials of the scan.
#ifndef MOSAIC_GATE_RING
#define MOSAIC_GATE_RING 2
#endif
constexpr int kRing = MOSAIC_GATE_RING;  // tiles a block may have voted and not yet scattered
struct ScanSmem {
    int len[kRing][kMaxT * kVoters];
    unsigned int part_count[kRing][kMaxT * kVoterWarps];  // survivors of (item, warp) -> exclusive offsets
    u64 part_tokens[kRing][kMaxT * kVoterWarps];          // their context tokens      -> exclusive offsets
    u64 base_count[kRing], base_tokens[kRing];           // the tile's exclusive prefix
    int warp_max[kRing][kVoterWarps];
    unsigned int tile_id[kRing];   // the tile in the slot (0xffffffff: the block has no more tiles)
    unsigned int next_tile[2];     // thread 0 -> voters: the ticket taken one tile ahead
};

// Roles of a block's warps: the first kVoterWarps warps ("voters", one question per thread and
// item) stream the rows, vote and later scatter; the last warp (the "scanner") turns a tile's
// partials into its exclusive prefix (block scan, published aggregate, look-back).  They meet only
// at named barriers, one pair per shared-memory slot: the voters ARRIVE on kBarVoted[slot] and go on
// with the next tile, and wait on kBarBased[slot] only when that next tile is voted too, to scatter
// the one before; the scanner waits on kBarVoted[slot] and arrives on kBarBased[slot].  So the
// look-back of a tile has a whole tile's streaming time to resolve, and the first rows of the next
// tile are requested before the scatter: the HBM stream does not stop for the scan.
// (7 + 1 warps: 256 threads, two blocks per SM at 128 registers -- four rows of E = 8 labels and
// weights in flight per thread without spills.  Measured on B200, 2^24 questions, E = 8, weighted:
// 8 + 1 warps x 3 blocks at 72 registers 271 us, 15 + 1 warps x 1 block 269 us, this 258 us.)
constexpr int kScanThreads = kVoters + 32;
enum : int { kBarVoted = 1, kBarBased = 1 + kRing };  // named barriers (0 is __syncthreads')
constexpr int kBarVoters = 1 + 2 * kRing;  // the voters among themselves
static_assert(2 * kRing + 1 < 16, "named barriers");
__device__ __forceinline__ void bar_arrive(int id) {
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "n"(kScanThreads) : "memory");
}
__device__ __forceinline__ void bar_sync(int id) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(kScanThreads) : "memory");
}
__device__ __forceinline__ void voter_bar() {
    asm volatile("bar.sync %0, %1;" ::"n"(kBarVoters), "n"(kVoters) : "memory");
}

// Programmatic dependent launch: the kernel that zeroes the scan workspace is launched just before
// this one and the two overlap; whoever touches the workspace first waits here for the zeroing grid
// to have completed (and its writes to be visible).
__device__ __forceinline__ void grid_barrier() {
    asm volatile("griddepcontrol.wait;" ::: "memory");
}
#ifndef MOSAIC_GATE_CHAIN
#define MOSAIC_GATE_CHAIN 1
#endif
// MOSAIC_GATE_CHAIN: both kernels of a call are launched as programmatic dependents and let THEIR
// dependents be scheduled at once (launch_dependents at entry), so that when calls follow one
// another in a stream the launch latency and the ramp of call N + 1 hide behind the tail of call
// N.  Nothing is read or written before griddepcontrol.wait, which returns only when everything
// earlier in the stream has completed and is visible -- so the order of the results is the
// stream's, as without it; a kernel launched the ordinary way after ours waits for full completion.
__device__ __forceinline__ void allow_dependents() {
#if MOSAIC_GATE_CHAIN
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
#endif
}
__global__ void __launch_bounds__(256) zero_states_kernel(uint4* p, size_t n16) {
    allow_dependents();
    grid_barrier();  // the workspace may be the one an earlier call in the stream is still using
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n16) p[i] = make_uint4(0u, 0u, 0u, 0u);
}

#ifdef MOSAIC_GATE_TRACE  // timing investigation builds only (_work/): per-block %globaltimer stamps
__device__ unsigned long long g_trace[1024 * 8];
__device__ __forceinline__ void trace(int slot) {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    if (blockIdx.x < 1024) g_trace[blockIdx.x * 8 + slot] = t;
}
#define MOSAIC_TRACE(slot, cond) do { if (cond) trace(slot); } while (0)
#else
#define MOSAIC_TRACE(slot, cond) do { } while (0)
#endif

template <int E_T, int CONF, int SRC, int BATCH, int BLOCKS, bool ABSTAIN>
__global__ void __launch_bounds__(kScanThreads, BLOCKS) gate_scan_kernel(const GateArgs p) {
    constexpr int EM = (SRC == kSrcAnswers) ? (E_T ? E_T : MOSAIC_MAX_EXPERTS) : 1;
    constexpr bool kWeighted = SRC == kSrcAnswers && CONF != MOSAIC_CONF_VOTE;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int E = E_T ? E_T : p.E;
    const int T = p.items;  // items of a tile (<= kMaxT): a tile is kVoters * T questions
    const int64_t tile_q = (int64_t)kVoters * T;

    __shared__ ScanSmem sm;
    __shared__ float agree_lut[MOSAIC_MAX_EXPERTS + 1];
    allow_dependents();
    fill_agree_lut(agree_lut, E);


    if (warp < kVoterWarps) {
        // ======================================= voters =======================================
        // Item k of round r is question (tile(r) * T + k) * kVoters + thread.  The rows are
        // taken BATCH items at a time: all the loads of a batch are issued, then its votes run.
        int32_t a[BATCH][EM];
        float w[BATCH][EM];   // (dead, and removed by the compiler, when no weights are read)
        int32_t len[BATCH];
        float thr[BATCH];     // tau of the question
        float given[BATCH];   // kSrcConf: C(q);  kSrcBypass: the mask byte
        bool valid[BATCH];
        const uint32_t Q32 = (uint32_t)p.Q;  // Q < 2^31: question indices are 32-bit
        // Items k0 .. k0 + BATCH - 1 of the tile whose item 0 is question `qt` for this thread.
        // FULL: the whole batch lies inside the tile and the tile inside Q (no per-row checks, no
        // branches between the rows: their loads and, below, their votes interleave freely).
        auto request = [&](auto full_c, uint32_t qt, int k0) {
            constexpr bool FULL = decltype(full_c)::value;
#pragma unroll
            for (int u = 0; u < BATCH; ++u) {
                const uint32_t q = qt + (uint32_t)(k0 + u) * kVoters;
                valid[u] = FULL || (k0 + u < T && q < Q32);
                if (valid[u]) {
                    if constexpr (SRC == kSrcAnswers) {
                        load_row<E_T, EM>(p.answers, q, E, a[u]);
                        if constexpr (kWeighted) load_row<E_T, EM>(p.expert_conf, q, E, w[u]);
                    } else if constexpr (SRC == kSrcBypass) {
                        given[u] = (float)__ldg(p.bypass_in + q);
                    } else {
                        given[u] = __ldg(p.conf_in + q);
                    }
                    if constexpr (SRC != kSrcBypass) thr[u] = p.tau_q ? __ldg(p.tau_q + q) : p.tau;
                    len[u] = __ldg(p.ctx_len + q);
                }
            }
        };
        int my_max = 0;
        // G1-G3 (vote, confidence, threshold) of the batch; (survived, ctx_len) and the (item, warp)
        // partials of the scan into shared-memory slot `slot`.
        auto vote = [&](auto full_c, uint32_t qt, int k0, int slot) {
            constexpr bool FULL = decltype(full_c)::value;
            bool surv[BATCH];
#pragma unroll
            for (int u = 0; u < BATCH; ++u) {
                [[maybe_unused]] const uint32_t q = qt + (uint32_t)(k0 + u) * kVoters;
                surv[u] = false;
                if (FULL || valid[u]) {
                    if constexpr (SRC == kSrcAnswers) {
                        int32_t mode, count;
                        float agree, conf;
                        bool bypass;
                        gate_row<EM, CONF, (E_T != 0), ABSTAIN>(a[u], w[u], E, thr[u], p.abstain,
                                                                agree_lut, mode, count, agree, conf,
                                                                bypass);
                        if (p.mode_out) __stcs(p.mode_out + q, mode);
                        if (p.count_out) __stcs(p.count_out + q, count);
                        if (p.agree_out) __stcs(p.agree_out + q, agree);
                        if (p.conf_out) __stcs(p.conf_out + q, conf);
                        if (p.bypass_out) p.bypass_out[q] = bypass ? 1 : 0;
                        surv[u] = !bypass;
                    } else if constexpr (SRC == kSrcBypass) {
                        surv[u] = given[u] == 0.f;
                    } else {
                        const bool bypass = given[u] >= thr[u];  // fp32; NaN never bypasses
                        if (p.bypass_out) p.bypass_out[q] = bypass ? 1 : 0;
                        surv[u] = !bypass;
                    }
                }
            }
#pragma unroll
            for (int u = 0; u < BATCH; ++u) {
                const int k = k0 + u;
                if (FULL || k < T) {
                    // survivors, their tokens (two 16-bit-half reductions so that the 32-lane sums
                    // cannot overflow 32 bits), max length
                    const uint32_t v = surv[u] ? (uint32_t)len[u] : 0u;
                    sm.len[slot][k * kVoters + tid] = surv[u] ? len[u] : -1;
                    const unsigned ballot = __ballot_sync(0xffffffffu, surv[u]);
                    const uint32_t lo = __reduce_add_sync(0xffffffffu, v & 0xffffu);
                    const uint32_t hi = __reduce_add_sync(0xffffffffu, v >> 16);
                    my_max = max(my_max, (int)v);
                    if (lane == 0) {
                        sm.part_count[slot][k * kVoterWarps + warp] = __popc(ballot);
                        sm.part_tokens[slot][k * kVoterWarps + warp] = (u64)lo + ((u64)hi << 16);
                    }
                }
            }
        };
        using Full = std::integral_constant<bool, true>;
        using Ragged = std::integral_constant<bool, false>;
        const uint32_t tile_q32 = (uint32_t)tile_q;
        // is every question of the tile inside Q?  (a tile past the last one is not)
        auto tile_full = [&](unsigned int t) {
            return t < p.num_tiles && (uint64_t)(t + 1) * tile_q32 <= (uint64_t)Q32;
        };
        // the first batch of a tile (also used to get the NEXT tile's first rows on their way)
        auto request_first = [&](unsigned int t) {
            if (t >= p.num_tiles) {
#pragma unroll
                for (int u = 0; u < BATCH; ++u) valid[u] = false;
            } else if (tile_full(t) && BATCH <= T) {
                request(Full{}, t * tile_q32 + tid, 0);
            } else {
                request(Ragged{}, t * tile_q32 + tid, 0);
            }
        };
        // G4-G5: stable scatter of a tile's survivors (scan order inside the tile is (item,
        // thread): exactly ascending question index).  Four items at a time, so that their
        // (independent) warp scans overlap.  A warp reads only its own entries of the slot.
        auto scatter = [&](unsigned int tile, int slot) {
            const int64_t q0 = (int64_t)tile * tile_q;
            const u64 base_c = sm.base_count[slot], base_t = sm.base_tokens[slot];
            constexpr int U = 4;
            for (int k0 = 0; k0 < T; k0 += U) {
                int v[U];
                unsigned ballot[U];
                uint32_t x[U];
                uint32_t mx = 0;
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    v[u] = (k0 + u < T) ? sm.len[slot][(k0 + u) * kVoters + tid] : -1;
                    ballot[u] = __ballot_sync(0xffffffffu, v[u] >= 0);
                    x[u] = v[u] >= 0 ? (uint32_t)v[u] : 0u;
                    mx = max(mx, x[u]);
                }
                const bool small = __reduce_max_sync(0xffffffffu, mx) < (1u << 26);  // no overflow
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
                        const u64 at = base_c + sm.part_count[slot][k * kVoterWarps + warp] + rank;
                        p.survivor_idx[at] = (int32_t)(q0 + (int64_t)k * kVoters + tid);
                        p.cu_seqlens[at + 1] =
                            (int64_t)(base_t + sm.part_tokens[slot][k * kVoterWarps + warp] + incl[u]);
                    }
                }
            }
        };

        // Tiles are handed out by an atomic ticket IN START ORDER: a tile only ever waits (in the
        // look-back) for tiles of smaller index, every one of which belongs to a block that is
        // already running, so the scan cannot deadlock however the blocks are scheduled; and a
        // block whose SM is slower (their streaming rates differ by up to 2x) simply takes fewer.
        // Thread 0 takes the ticket of the NEXT tile at the top of a tile (the atomic's round trip
        // hides behind the votes); the voters' own barrier publishes it.
        MOSAIC_TRACE(0, tid == 0);
#if MOSAIC_GATE_CHAIN
        // A hint only (no result depends on it): while this block waits for the zeroing grid -- and
        // through it for whatever runs before in the stream -- pull the rows of "its" first tile
        // towards L2; with tickets handed out in start order that is very likely the tile it gets.
        if (blockIdx.x < p.num_tiles && (lane & 3) == 0) {
            for (int k = 0; k < T; ++k) {
                const uint32_t q = (blockIdx.x * (uint32_t)T + k) * kVoters + tid;
                if (q < (uint32_t)p.Q) {
                    if constexpr (SRC == kSrcAnswers) {
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(p.answers + (size_t)q * E));
                        if constexpr (kWeighted)
                            asm volatile("prefetch.global.L2 [%0];" ::"l"(p.expert_conf + (size_t)q * E));
                    }
                }
            }
        }
#endif
        if (tid == 0) {
            grid_barrier();  // the zeroing grid is complete: ticket = 0, every state "not published"
            sm.next_tile[0] = atomicAdd(&p.header->ticket, 1u);
        }
        voter_bar();
        unsigned int tile = sm.next_tile[0];
        request_first(tile);
        MOSAIC_TRACE(1, tid == 0);
        int r = 0;
        for (; tile < p.num_tiles; ++r) {
            const int slot = r % kRing;
            const uint32_t qt = tile * tile_q32 + tid;
            if (tid == 0) {
                sm.tile_id[slot] = tile;
                sm.next_tile[(r + 1) & 1] = atomicAdd(&p.header->ticket, 1u);
            }
            if (tile_full(tile)) {
                int k0 = 0;
                for (; k0 + BATCH <= T; k0 += BATCH) {
                    if (k0 > 0) request(Full{}, qt, k0);
                    vote(Full{}, qt, k0, slot);
                }
                if (k0 < T) {  // T is not a multiple of BATCH: the last, partial batch
                    if (k0 > 0) request(Ragged{}, qt, k0);
                    vote(Ragged{}, qt, k0, slot);
                }
            } else {
                for (int k0 = 0; k0 < T; k0 += BATCH) {
                    if (k0 > 0) request(Ragged{}, qt, k0);
                    vote(Ragged{}, qt, k0, slot);
                }
            }
            // the tile is voted: hand it to the scanner; get the next tile's first rows on their
            // way; scatter the oldest tile of the ring, whose look-back has had the time since
            my_max = __reduce_max_sync(0xffffffffu, my_max);
            if (lane == 0) sm.warp_max[slot][warp] = my_max;
            my_max = 0;
            const int old = (r + 1) % kRing;  // == (r - (kRing - 1)) % kRing: the oldest slot
            const unsigned int old_tile = sm.tile_id[old];  // (read before thread 0 can reuse it)
            MOSAIC_TRACE(2 + (r > 0 ? 1 : 0), tid == 0);   // tile 0 voted / last tile voted
            voter_bar();
            bar_arrive(kBarVoted + slot);
            const unsigned int next = sm.next_tile[(r + 1) & 1];
            request_first(next);
            if (r >= kRing - 1) {
                bar_sync(kBarBased + old);
                scatter(old_tile, old);
            }
            tile = next;
        }
        // no more tiles: tell the scanner (a sentinel in the next slot, whose tile is scattered),
        // then drain the ring
        MOSAIC_TRACE(4, tid == 0);
        unsigned int left[kRing];
#pragma unroll
        for (int j = 0; j < kRing; ++j) left[j] = sm.tile_id[j];
        voter_bar();
        if (tid == 0) sm.tile_id[r % kRing] = 0xffffffffu;
        bar_arrive(kBarVoted + r % kRing);
        for (int rr = (r - (kRing - 1) > 0 ? r - (kRing - 1) : 0); rr < r; ++rr) {
            bar_sync(kBarBased + rr % kRing);
            MOSAIC_TRACE(5, tid == 0);   // last base known
#pragma unroll
            for (int j = 0; j < kRing; ++j)
                if (j == rr % kRing) scatter(left[j], j);
        }
        MOSAIC_TRACE(6, tid == 0);   // done
    } else {
        // ======================================= scanner ======================================
        grid_barrier();
        for (int r = 0;; ++r) {
            const int slot = r % kRing;
            bar_sync(kBarVoted + slot);
            const unsigned int tile = sm.tile_id[slot];
            if (tile == 0xffffffffu) break;
            // exclusive scan of the T * kVoterWarps partials, PER consecutive ones per lane
            constexpr int PER = (kMaxT * kVoterWarps + 31) / 32;
            const int n_part = T * kVoterWarps;
            unsigned int c[PER];
            u64 t[PER];
            unsigned int csum = 0;
            u64 tsum = 0;
#pragma unroll
            for (int j = 0; j < PER; ++j) {
                const int e = lane * PER + j;
                c[j] = e < n_part ? sm.part_count[slot][e] : 0u;
                t[j] = e < n_part ? sm.part_tokens[slot][e] : 0ull;
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
                    sm.part_count[slot][e] = cx;
                    sm.part_tokens[slot][e] = tx;
                }
                cx += c[j];
                tx += t[j];
            }
            Partial mine;
            mine.count = __shfl_sync(0xffffffffu, ci, 31);
            mine.tokens = __shfl_sync(0xffffffffu, ti, 31);
            mine.max_len =
                __reduce_max_sync(0xffffffffu, lane < kVoterWarps ? sm.warp_max[slot][lane] : 0);

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
                sm.base_count[slot] = before.count;
                sm.base_tokens[slot] = before.tokens;
                if (tile == 0) p.cu_seqlens[0] = 0;
                if (tile == p.num_tiles - 1) {
                    *p.n_survivors = (int32_t)incl.count;
                    *p.total_tokens = (int64_t)incl.tokens;
                    *p.max_seqlen = incl.max_len;
                }
            }
            __syncwarp();
            bar_arrive(kBarBased + slot);
        }
    }
}

// Blocks of this instantiation that fit one SM (asked of the runtime once per process).
template <int E_T, int CONF, int SRC, int BATCH, int BLOCKS, bool ABSTAIN>
int resident_blocks_per_sm() {
    static int cached = 0;
    if (cached == 0) {
        int n = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(
                &n, gate_scan_kernel<E_T, CONF, SRC, BATCH, BLOCKS, ABSTAIN>, kScanThreads, 0) != cudaSuccess ||
            n < 1)
            return 0;
        cached = n < BLOCKS ? n : BLOCKS;
    }
    return cached;
}

template <int E_T, int CONF, int SRC, int BATCH, int BLOCKS, bool ABSTAIN = false>
mosaic_status_t launch(GateArgs& a, size_t ws_bytes, void* workspace, cudaStream_t stream) {
    const int per_sm = resident_blocks_per_sm<E_T, CONF, SRC, BATCH, BLOCKS, ABSTAIN>();
    if (per_sm < 1) return cuda_fail(cudaErrorLaunchOutOfResources);
    const int64_t resident = (int64_t)num_sms() * per_sm;
    // A tile is kVoters * T questions and goes to whichever block asks next (ticket).  The
    // blocks finish together only if the tiles fill whole waves of the resident grid: T is the
    // whole multiple of BATCH (a partial batch takes the per-row checked path: 308 against 257 us
    // at 2^24 questions with T = 6 against 8) up to kMaxT with the shortest makespan (waves x T
    // items per thread); a shorter tile must win by 15 % (more tiles: more barriers and look-backs).
    const int64_t per_thread = (a.Q + resident * kVoters - 1) / (resident * kVoters);
    auto span_of = [&](int t) {
        const int64_t tiles_t = (a.Q + (int64_t)kVoters * t - 1) / ((int64_t)kVoters * t);
        return (tiles_t + resident - 1) / resident * t;
    };
    constexpr int kStep = BATCH < kMaxT ? BATCH : 1;
    if (per_thread <= kMaxT) {
        a.items = (int)per_thread;  // one wave: one tile per block
    } else {
        a.items = kMaxT / kStep * kStep;
        for (int t = a.items - kStep; t >= kStep; t -= kStep)
            if (span_of(t) * 115 < span_of(a.items) * 100) a.items = t;
    }
    const int64_t tile = (int64_t)kVoters * a.items;
    const unsigned int tiles = (unsigned int)((a.Q + tile - 1) / tile);
    a.num_tiles = tiles;
    if (ws_bytes < sizeof(ScanHeader)) return MOSAIC_ERR_WORKSPACE_TOO_SMALL;
    const size_t for_tiles = ws_bytes - sizeof(ScanHeader);
    int stride = 8;  // 128-byte lines if the workspace holds them, else denser
    while (stride > 1 && (size_t)tiles * stride * sizeof(TileState) > for_tiles) stride >>= 1;
    a.tile_stride = stride;
    if (for_tiles < (size_t)tiles * stride * sizeof(TileState)) return MOSAIC_ERR_WORKSPACE_TOO_SMALL;
    a.header = static_cast<ScanHeader*>(workspace);
    a.tiles = reinterpret_cast<TileState*>(static_cast<char*>(workspace) + sizeof(ScanHeader));
    // The workspace's contents are arbitrary: a small kernel zeroes the ticket and the tile states,
    // and the scan kernel, launched as its programmatic dependent, overlaps it (its first touch of
    // the workspace waits for it).
    const size_t n16 = sizeof(ScanHeader) / 16 + (size_t)tiles * stride;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t zcfg{};
    zcfg.gridDim = dim3((unsigned)((n16 + 255) / 256));
    zcfg.blockDim = dim3(256);
    zcfg.stream = stream;
    zcfg.attrs = attr;
    zcfg.numAttrs = MOSAIC_GATE_CHAIN ? 1 : 0;
    MOSAIC_CUDA_TRY(cudaLaunchKernelEx(&zcfg, zero_states_kernel, static_cast<uint4*>(workspace), n16));
    count_launch();
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned int)(tiles < resident ? tiles : resident));
    cfg.blockDim = dim3(kScanThreads);
    cfg.stream = stream;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    MOSAIC_CUDA_TRY(
        cudaLaunchKernelEx(&cfg, gate_scan_kernel<E_T, CONF, SRC, BATCH, BLOCKS, ABSTAIN>, a));
    count_launch();
    return MOSAIC_OK;
}


}  // namespace
}  // namespace mosaic
