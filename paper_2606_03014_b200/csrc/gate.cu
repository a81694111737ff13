// gate.cu -- step 1 of the confidence-gated aggregator stage (Sec. 4.2 P:L170-188,
// Alg. 1): per-question plurality vote, confidence, threshold, and the stream
// compaction of the surviving questions into a ragged batch with cu_seqlens.
//
// One kernel template serves the three C-ABI calls:
//   mosaic_gate          DO_GATE            -- thread per question, no ordering between blocks
//   mosaic_compact       DO_COMPACT         -- single-pass scan (decoupled look-back)
//   mosaic_gate_compact  DO_GATE|DO_COMPACT -- both in one pass over HBM
//
// HBM-bound: every input byte is read once with 16-byte loads where the
// row width allows, outputs are written once, coalesced.  A tile is THREADS x ITEMS questions in
// a striped arrangement (question = tile_base + item * THREADS + thread) so a warp's loads and
// its compacted stores are both contiguous.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "common.cuh"

namespace mosaic {
namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kMinTile = kThreads;  // smallest tile any instantiation uses (ITEMS == 1)

using u64 = unsigned long long;

// Scan state of one tile: two independent words, each carrying its own 2-bit status in bits
// 62..63 (0 = not written, 1 = tile aggregate, 2 = inclusive prefix) so that a relaxed 64-bit
// load always sees a value together with its status.
struct alignas(16) TileState {
    u64 count;   // survivors
    u64 tokens;  // context tokens of the survivors
};
constexpr u64 kValueMask = (1ull << 62) - 1;
constexpr u64 kAggregate = 1ull << 62;
constexpr u64 kPrefix = 2ull << 62;

struct alignas(16) ScanHeader {
    unsigned int ticket;    // next tile id (tiles are handed out in start order)
    unsigned int finished;  // tiles done
    int max_len;            // running max of the survivors' ctx_len
    int pad;
};

__device__ __forceinline__ u64 ld_relaxed(const u64* p) {
    u64 v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed(u64* p, u64 v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

__device__ __forceinline__ u64 warp_sum(u64 v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Row loads: 16-byte vectors when the row width allows (rows start 16-byte aligned when
// E % 4 == 0 because the base pointer is), 8-byte for E % 2 == 0, scalar otherwise.
template <int E_T, int EM, typename T>
__device__ __forceinline__ void load_row(const T* __restrict__ base, int64_t q, int E, T (&r)[EM]) {
    static_assert(sizeof(T) == 4, "");
    if constexpr (E_T != 0 && E_T % 4 == 0) {
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

// Alg. 1 lines 2-4 for one question.  Same decisions, in the same precision, as
// the definition: c* by counting, mode = smallest label among those reaching c* (reading G-2),
// agree = fl32(c*)/fl32(E) (one IEEE division, reading G-4), weighted share in binary64 in
// expert order (reading G-10), bypass = conf >= tau in fp32 (">=").
template <int EM, int CONF>
__device__ __forceinline__ void gate_row(const int32_t (&a)[EM], const float (&w)[EM], int E,
                                         float tau, int32_t& mode, int32_t& count, float& agree,
                                         float& conf, bool& bypass) {
    int32_t c_star = 0, md = 0;
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
    agree = __fdiv_rn((float)c_star, (float)E);
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
    unsigned int num_tiles;
};

// Sum, over the tiles before `tile`, of both scanned quantities (decoupled look-back: walk the
// predecessors 32 at a time, adding aggregates until an inclusive prefix is met).  The two words
// are walked in lockstep but finish independently.  Whole warp calls; result in every lane.
__device__ __forceinline__ void look_back(const TileState* tiles, int tile, int lane, u64& count,
                                          u64& tokens) {
    u64 acc_c = 0, acc_t = 0;
    bool done_c = false, done_t = false;
    for (int base = tile - 1; !(done_c && done_t); base -= 32) {
        const int idx = base - lane;
        u64 wc = kPrefix, wt = kPrefix;  // "tile -1": prefix 0
        if (idx >= 0) {
            const u64* pc = &tiles[idx].count;
            const u64* pt = &tiles[idx].tokens;
            for (;;) {
                wc = ld_relaxed(pc);
                wt = ld_relaxed(pt);
                if ((wc >> 62) != 0 && (wt >> 62) != 0) break;
                __nanosleep(20);
            }
        }
        __syncwarp();
        if (!done_c) {
            const unsigned pm = __ballot_sync(0xffffffffu, (wc >> 62) == 2);
            const int first = pm ? (__ffs(pm) - 1) : 31;
            acc_c += warp_sum(lane <= first ? (wc & kValueMask) : 0ull);
            done_c = pm != 0;
        }
        if (!done_t) {
            const unsigned pm = __ballot_sync(0xffffffffu, (wt >> 62) == 2);
            const int first = pm ? (__ffs(pm) - 1) : 31;
            acc_t += warp_sum(lane <= first ? (wt & kValueMask) : 0ull);
            done_t = pm != 0;
        }
    }
    count = acc_c;
    tokens = acc_t;
}

template <int E_T, int CONF, bool DO_GATE, bool DO_COMPACT, int ITEMS>
__global__ void __launch_bounds__(kThreads) gate_compact_kernel(const GateArgs p) {
    constexpr int EM = DO_GATE ? (E_T ? E_T : MOSAIC_MAX_EXPERTS) : 1;
    constexpr int TILE = kThreads * ITEMS;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int E = E_T ? E_T : p.E;

    __shared__ unsigned int s_tile;
    __shared__ u64 s_wcount[ITEMS * kWarps];  // per (item, warp) survivor counts -> exclusive offsets
    __shared__ u64 s_wtok[ITEMS * kWarps];    // per (item, warp) token sums      -> exclusive offsets
    __shared__ u64 s_base[2];                 // the tile's exclusive prefix (count, tokens)
    __shared__ int s_max;

    unsigned int tile = blockIdx.x;
    if constexpr (DO_COMPACT) {
        if (tid == 0) {
            s_tile = atomicAdd(&p.header->ticket, 1u);
            s_max = 0;
        }
        __syncthreads();
        tile = s_tile;
    }
    const int64_t q0 = (int64_t)tile * TILE;

    bool surv[ITEMS];
    int32_t len[ITEMS];

    // ---- G1-G3: vote, confidence, threshold ---------------------------------------------------
    if constexpr (DO_GATE) {
        int32_t a[ITEMS][EM];
        float w[ITEMS][EM];
#pragma unroll
        for (int k = 0; k < ITEMS; ++k) {
            const int64_t q = q0 + k * kThreads + tid;
            if (q < p.Q) {
                load_row<E_T, EM>(p.answers, q, E, a[k]);
                if constexpr (CONF == MOSAIC_CONF_WEIGHTED)
                    load_row<E_T, EM>(p.expert_conf, q, E, w[k]);
            }
        }
        if constexpr (DO_COMPACT) {
#pragma unroll
            for (int k = 0; k < ITEMS; ++k) {
                const int64_t q = q0 + k * kThreads + tid;
                len[k] = (q < p.Q) ? __ldg(p.ctx_len + q) : 0;
            }
        }
#pragma unroll
        for (int k = 0; k < ITEMS; ++k) {
            const int64_t q = q0 + k * kThreads + tid;
            surv[k] = false;
            if (q < p.Q) {
                int32_t mode, count;
                float agree, conf;
                bool bypass;
                gate_row<EM, CONF>(a[k], w[k], E, p.tau, mode, count, agree, conf, bypass);
                if (p.mode_out) p.mode_out[q] = mode;
                if (p.count_out) p.count_out[q] = count;
                if (p.agree_out) p.agree_out[q] = agree;
                if (p.conf_out) p.conf_out[q] = conf;
                if (p.bypass_out) p.bypass_out[q] = bypass ? 1 : 0;
                surv[k] = !bypass;
            }
        }
    } else {
#pragma unroll
        for (int k = 0; k < ITEMS; ++k) {
            const int64_t q = q0 + k * kThreads + tid;
            surv[k] = (q < p.Q) ? (__ldg(p.bypass_in + q) == 0) : false;
            len[k] = (q < p.Q) ? __ldg(p.ctx_len + q) : 0;
        }
    }
    if constexpr (DO_COMPACT) {
    // ---- G4-G5: stable compaction and cu_seqlens -------------------------------------------------
    // Scan order inside the tile is (item, thread): exactly ascending question index.
    unsigned rank_in_warp[ITEMS];
    u64 tok_incl[ITEMS];
    int my_max = 0;
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        const unsigned ballot = __ballot_sync(0xffffffffu, surv[k]);
        rank_in_warp[k] = __popc(ballot & ((1u << lane) - 1u));
        u64 v = surv[k] ? (u64)(uint32_t)len[k] : 0ull;
        if (surv[k]) my_max = max(my_max, len[k]);
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u64 t = __shfl_up_sync(0xffffffffu, v, o);
            if (lane >= o) v += t;
        }
        tok_incl[k] = v;
        if (lane == 31) {
            s_wcount[k * kWarps + warp] = (u64)__popc(ballot);
            s_wtok[k * kWarps + warp] = v;
        }
    }
    my_max = __reduce_max_sync(0xffffffffu, my_max);
    if (lane == 0 && my_max > 0) atomicMax(&s_max, my_max);
    __syncthreads();

    if (warp == 0) {
        // exclusive scan of the ITEMS*kWarps (<= 32) partials, then the tile's global prefix
        static_assert(ITEMS * kWarps <= 32, "partials must fit one warp");
        const bool has = lane < ITEMS * kWarps;
        const u64 c = has ? s_wcount[lane] : 0ull, t = has ? s_wtok[lane] : 0ull;
        u64 ci = c, ti = t;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u64 cc = __shfl_up_sync(0xffffffffu, ci, o);
            const u64 tt = __shfl_up_sync(0xffffffffu, ti, o);
            if (lane >= o) {
                ci += cc;
                ti += tt;
            }
        }
        if (has) {
            s_wcount[lane] = ci - c;
            s_wtok[lane] = ti - t;
        }
        const u64 tile_c = __shfl_sync(0xffffffffu, ci, 31), tile_t = __shfl_sync(0xffffffffu, ti, 31);
        TileState* me = p.tiles + tile;
        if (tile == 0) {
            if (lane == 0) {
                st_relaxed(&me->count, kPrefix | tile_c);
                st_relaxed(&me->tokens, kPrefix | tile_t);
                s_base[0] = 0;
                s_base[1] = 0;
                p.cu_seqlens[0] = 0;
            }
        } else {
            if (lane == 0) {
                st_relaxed(&me->count, kAggregate | tile_c);
                st_relaxed(&me->tokens, kAggregate | tile_t);
            }
            u64 pc, pt;
            look_back(p.tiles, (int)tile, lane, pc, pt);
            if (lane == 0) {
                st_relaxed(&me->count, kPrefix | (pc + tile_c));
                st_relaxed(&me->tokens, kPrefix | (pt + tile_t));
                s_base[0] = pc;
                s_base[1] = pt;
            }
        }
        if (lane == 0 && tile == p.num_tiles - 1) {
            *p.n_survivors = (int32_t)(s_base[0] + tile_c);
            *p.total_tokens = (int64_t)(s_base[1] + tile_t);
        }
    }
    __syncthreads();

    const u64 base_c = s_base[0], base_t = s_base[1];
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        if (surv[k]) {
            const u64 r = base_c + s_wcount[k * kWarps + warp] + rank_in_warp[k];
            p.survivor_idx[r] = (int32_t)(q0 + k * kThreads + tid);
            p.cu_seqlens[r + 1] = (int64_t)(base_t + s_wtok[k * kWarps + warp] + tok_incl[k]);
        }
    }

    if (tid == 0) {
        if (s_max > 0) atomicMax(&p.header->max_len, s_max);
        __threadfence();
        const unsigned done = atomicAdd(&p.header->finished, 1u);
        if (done == p.num_tiles - 1) {
            __threadfence();
            *p.max_seqlen = *reinterpret_cast<volatile int*>(&p.header->max_len);
        }
    }
    }  // DO_COMPACT
}

template <int E_T, int CONF, bool DO_GATE, bool DO_COMPACT, int ITEMS>
mosaic_status_t launch(GateArgs& a, size_t ws_bytes, void* workspace, cudaStream_t stream) {
    constexpr int TILE = kThreads * ITEMS;
    const unsigned int tiles = (unsigned int)((a.Q + TILE - 1) / TILE);
    a.num_tiles = tiles;
    if constexpr (DO_COMPACT) {
        const size_t need = sizeof(ScanHeader) + (size_t)tiles * sizeof(TileState);
        if (ws_bytes < need) return MOSAIC_ERR_WORKSPACE_TOO_SMALL;
        a.header = static_cast<ScanHeader*>(workspace);
        a.tiles = reinterpret_cast<TileState*>(static_cast<char*>(workspace) + sizeof(ScanHeader));
        MOSAIC_CUDA_TRY(cudaMemsetAsync(workspace, 0, need, stream));
    }
    gate_compact_kernel<E_T, CONF, DO_GATE, DO_COMPACT, ITEMS><<<tiles, kThreads, 0, stream>>>(a);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());
    return MOSAIC_OK;
}

template <int CONF, bool DO_COMPACT>
mosaic_status_t dispatch_gate(GateArgs& a, size_t ws_bytes, void* ws, cudaStream_t s) {
    switch (a.E) {
        case 1: return launch<1, CONF, true, DO_COMPACT, 4>(a, ws_bytes, ws, s);
        case 2: return launch<2, CONF, true, DO_COMPACT, 4>(a, ws_bytes, ws, s);
        case 3: return launch<3, CONF, true, DO_COMPACT, 4>(a, ws_bytes, ws, s);
        case 4: return launch<4, CONF, true, DO_COMPACT, 4>(a, ws_bytes, ws, s);
        case 5: return launch<5, CONF, true, DO_COMPACT, 4>(a, ws_bytes, ws, s);
        case 6: return launch<6, CONF, true, DO_COMPACT, 4>(a, ws_bytes, ws, s);
        case 7: return launch<7, CONF, true, DO_COMPACT, 4>(a, ws_bytes, ws, s);
        case 8: return launch<8, CONF, true, DO_COMPACT, 4>(a, ws_bytes, ws, s);
        default: return launch<0, CONF, true, DO_COMPACT, 1>(a, ws_bytes, ws, s);
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
    const size_t tiles = (size_t)((Q + kMinTile - 1) / kMinTile);
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
    return launch<1, MOSAIC_CONF_VOTE, false, true, 4>(a, workspace_bytes, workspace, s);
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
