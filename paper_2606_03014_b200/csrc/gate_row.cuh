// gate_row.cuh -- Alg. 1 lines 2-4 for ONE question, shared by the gate-only
// kernel (gate.cu) and the fused gate + compaction kernel (compact.cu): row loads, the sorting
// networks, the vote / confidence / threshold arithmetic and the argument block of both kernels.
// Device code of the product path; nothing here comes from oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "common.cuh"

namespace mosaic {

using u64 = unsigned long long;

constexpr int kGateThreads = 256;
constexpr int kGateWarps = kGateThreads / 32;

// Where a question's bypass decision comes from.
enum : int {
    kSrcAnswers = 0,  // Alg. 1 lines 2-4 on the E answers (mosaic_gate*, the paper's gate)
    kSrcBypass = 1,   // a bypass mask computed earlier (mosaic_compact)
    kSrcConf = 2      // a confidence C(q) supplied by the caller (mosaic_conf_compact)
};

// Failed Extract (reading N3-2): an expert whose label equals `label` abstains.
struct Abstain {
    int on;      // 0: every label is an answer (reading G-6)
    int label;   // the sentinel
    int shrink;  // 0: C divides by the k experts recruited (P:L182 literally); 1: by those that answered
};

struct ScanHeader;  // compact.cu
struct TileState;

struct GateArgs {
    const int32_t* answers;
    const float* expert_conf;
    const uint8_t* bypass_in;  // kSrcBypass
    const float* conf_in;      // kSrcConf
    const int32_t* ctx_len;
    int64_t Q;
    int32_t E;
    float tau;
    const float* tau_q;  // a threshold per question, else NULL: tau for all
    Abstain abstain;
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
    int tile_stride;  // tile t lives at tiles[t * tile_stride]: one state per 128-byte line when the
                      // workspace allows, so the look-back loads of ~300 tiles spread over the L2 slices
    unsigned int num_tiles;
    int items;  // gate-only kernel: questions per thread
};

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

// Alg. 1 lines 2-4 for one question.  Same decisions, in the same precision, as the
// definition: c* = the largest number of equal labels, mode = smallest label among those reaching
// c* (reading G-2), agree = fl32(c*) / fl32(k) (one IEEE division, reading G-4), bypass =
// conf >= tau in fp32 (">=").  conf is
//   MOSAIC_CONF_VOTE             agree                                   (the paper's C_vote)
//   MOSAIC_CONF_WEIGHTED         fl32(sum_{a_i = mode} w_i / sum_i w_i)   (reading G-10)
//   MOSAIC_CONF_WEIGHTED_ARGMAX  the same share, with mode = the label of the LARGEST weight sum
//                                (ties -> smallest label; reading N3-3), count = its votes
// with binary64 sums in expert order, and the vote rule whenever sum_i w_i is not > 0.
// An abstaining expert (reading N3-2) is left out of every tally; k stays E unless `shrink`.
// SORTED (E known at compile time, <= 8, count plurality): the labels go through a sorting network
// and the plurality is the longest run, first (= smallest label) run winning ties; otherwise every
// label is counted against every other.
// ABSTAIN is the compile-time copy of ab.on (the common no-sentinel call pays nothing for it);
// agree_lut[c] = fl32(c) / fl32(E), the same IEEE division done once per block (shared memory).
template <int EM, int CONF, bool SORTED, bool ABSTAIN>
__device__ __forceinline__ void gate_row(const int32_t (&a)[EM], const float (&w)[EM], int E,
                                         float tau, Abstain ab, const float* agree_lut,
                                         int32_t& mode, int32_t& count, float& agree, float& conf,
                                         bool& bypass) {
    ab.on = ABSTAIN ? 1 : 0;
    auto vote_fraction = [&](int32_t c, int32_t k) -> float {
        if (!(ABSTAIN && ab.shrink)) return agree_lut[c];  // k == E
        return k > 0 ? __fdiv_rn((float)c, (float)k) : 0.f;
    };
    int32_t c_star = 0, md = ab.label;  // (all experts abstaining: no answer, C = 0)
    int32_t n_real = E;
    if (ab.on) {
        n_real = 0;
#pragma unroll
        for (int i = 0; i < EM; ++i)
            if (i < E) n_real += (a[i] != ab.label) ? 1 : 0;
    }
    double s_best = 0.0;  // weighted argmax: the weight sum of `md`
    if constexpr (SORTED && CONF != MOSAIC_CONF_WEIGHTED_ARGMAX) {
        int32_t s[EM];
#pragma unroll
        for (int i = 0; i < EM; ++i) s[i] = a[i];
        sort_labels<EM>(s);
        int32_t run = 1;
        md = s[0];
        c_star = (ab.on && s[0] == ab.label) ? 0 : 1;
#pragma unroll
        for (int i = 1; i < EM; ++i) {
            run = (s[i] == s[i - 1]) ? run + 1 : 1;
            const bool real = !(ab.on && s[i] == ab.label);
            if (real && run > c_star) {
                c_star = run;
                md = s[i];
            }
        }
    } else {
        // all pairs: n_i votes (and, for the weighted argmax, s_i weight) of expert i's label
        int32_t c_w = 0, md_w = ab.label;
        bool any_w = false;
#pragma unroll
        for (int i = 0; i < EM; ++i) {
            if (i < E && !(ab.on && a[i] == ab.label)) {
                int32_t n = 0;
                double s = 0.0;
#pragma unroll
                for (int j = 0; j < EM; ++j) {
                    if (j < E && a[j] == a[i]) {
                        n += 1;
                        if constexpr (CONF == MOSAIC_CONF_WEIGHTED_ARGMAX)
                            s = __dadd_rn(s, (double)w[j]);
                    }
                }
                if (n > c_star || (n == c_star && a[i] < md)) {
                    c_star = n;
                    md = a[i];
                }
                if constexpr (CONF == MOSAIC_CONF_WEIGHTED_ARGMAX) {
                    if (!any_w || s > s_best || (s == s_best && a[i] < md_w)) {
                        any_w = true;
                        s_best = s;
                        md_w = a[i];
                        c_w = n;
                    }
                }
            }
        }
        if constexpr (CONF == MOSAIC_CONF_WEIGHTED_ARGMAX) {
            // the denominator decides below whether the weights are usable at all
            double st = 0.0;
#pragma unroll
            for (int i = 0; i < EM; ++i)
                if (i < E && !(ab.on && ab.shrink && a[i] == ab.label))
                    st = __dadd_rn(st, (double)w[i]);
            if (st > 0.0 && any_w) {
                md = md_w;
                c_star = c_w;
                const int32_t k = (ab.on && ab.shrink) ? n_real : E;
                agree = vote_fraction(c_star, k);
                conf = __double2float_rn(__ddiv_rn(s_best, st));
                mode = md;
                count = c_star;
                bypass = conf >= tau;
                return;
            }
        }
    }
    const int32_t k = (ab.on && ab.shrink) ? n_real : E;
    agree = vote_fraction(c_star, k);
    conf = agree;
    if constexpr (CONF == MOSAIC_CONF_WEIGHTED) {
        double sm = 0.0, st = 0.0;
#pragma unroll
        for (int i = 0; i < EM; ++i) {
            if (i < E) {
                const double wi = (double)w[i];
                const bool real = !(ab.on && a[i] == ab.label);
                if (real || !(ab.on && ab.shrink)) st = __dadd_rn(st, wi);
                if constexpr (ABSTAIN) {
                    if (real && a[i] == md) sm = __dadd_rn(sm, wi);
                } else {
                    // one compare and one PREDICATED add (the compiler's version adds and then
                    // selects both halves: four instructions per expert instead of two)
                    asm("{\n\t.reg .pred p;\n\tsetp.eq.s32 p, %1, %2;\n\t@p add.rn.f64 %0, %0, %3;\n\t}"
                        : "+d"(sm)
                        : "r"(a[i]), "r"(md), "d"(wi));
                }
            }
        }
        if (st > 0.0) conf = __double2float_rn(__ddiv_rn(sm, st));
    }
    mode = md;
    count = c_star;
    bypass = conf >= tau;
}

// Whole block calls, once, before any gate_row (ends in a block-wide barrier).
__device__ __forceinline__ void fill_agree_lut(float* lut /* [MOSAIC_MAX_EXPERTS + 1] shared */, int E) {
    if ((int)threadIdx.x <= E) lut[threadIdx.x] = __fdiv_rn((float)threadIdx.x, (float)E);
    __syncthreads();
}

mosaic_status_t check_gate_args(const int32_t* answers, const float* expert_conf, int64_t Q,
                                int32_t E, float tau, int32_t conf_mode);

}  // namespace mosaic
