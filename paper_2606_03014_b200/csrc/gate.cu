// gate.cu -- mosaic_gate: Alg. 1 lines 2-4 (Sec. 4.2, Alg. 1) for Q
// questions without the compaction: per-question plurality vote, confidence, threshold.
// (The fused gate + stream compaction, which is what the stage runs, is compact.cu.)
//
// HBM-bound, no ordering between blocks: a thread owns whole questions in a striped arrangement
// (question = block_base + item * kGateThreads + thread, so a warp's loads are contiguous), BATCH
// rows in flight per thread, streaming stores for the outputs.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "common.cuh"
#include "gate_row.cuh"

namespace mosaic {

mosaic_status_t check_gate_args(const int32_t* answers, const float* expert_conf, int64_t Q,
                                int32_t E, float tau, int32_t conf_mode) {
    if (Q < 0 || Q >= (1ll << 31) || E < 1 || E > MOSAIC_MAX_EXPERTS || isnan(tau))
        return MOSAIC_ERR_INVALID_ARG;
    if (conf_mode != MOSAIC_CONF_VOTE && conf_mode != MOSAIC_CONF_WEIGHTED &&
        conf_mode != MOSAIC_CONF_WEIGHTED_ARGMAX)
        return MOSAIC_ERR_INVALID_ARG;
    const bool weighted = conf_mode != MOSAIC_CONF_VOTE;
    if (Q > 0) {
        if (!answers || !aligned16(answers)) return MOSAIC_ERR_INVALID_ARG;
        if (weighted && (!expert_conf || !aligned16(expert_conf))) return MOSAIC_ERR_INVALID_ARG;
        // 32-byte rows are read with 256-bit loads
        if (E % 8 == 0 && E <= 8 &&
            ((reinterpret_cast<uintptr_t>(answers) & 31u) ||
             (weighted && (reinterpret_cast<uintptr_t>(expert_conf) & 31u))))
            return MOSAIC_ERR_INVALID_ARG;
    }
    return MOSAIC_OK;
}

namespace {

constexpr int kMaxItems = 16;     // questions per thread, specialised E (<= 8)
constexpr int kMaxItemsWide = 4;  // ... generic E (<= 32): rows live in 2 x 32 registers
constexpr int kBlocksPerSM = 512 / kGateThreads;

template <int E_T, int CONF, int BATCH>
__global__ void __launch_bounds__(kGateThreads, kBlocksPerSM) gate_kernel(const GateArgs p) {
    constexpr int EM = E_T ? E_T : MOSAIC_MAX_EXPERTS;
    const int tid = threadIdx.x;
    const int E = E_T ? E_T : p.E;
    const int items = p.items;
    const int64_t q0 = (int64_t)blockIdx.x * kGateThreads * items;
    __shared__ float agree_lut[MOSAIC_MAX_EXPERTS + 1];
    fill_agree_lut(agree_lut, E);
    for (int it0 = 0; it0 < items; it0 += BATCH) {
        bool valid[BATCH];
        int32_t a[BATCH][EM];
        float w[BATCH][EM];
#pragma unroll
        for (int k = 0; k < BATCH; ++k) {
            const int64_t q = q0 + (int64_t)(it0 + k) * kGateThreads + tid;
            valid[k] = (it0 + k < items) && (q < p.Q);
            if (valid[k]) {
                load_row<E_T, EM>(p.answers, q, E, a[k]);
                if constexpr (CONF != MOSAIC_CONF_VOTE) load_row<E_T, EM>(p.expert_conf, q, E, w[k]);
            }
        }
#pragma unroll
        for (int k = 0; k < BATCH; ++k) {
            const int64_t q = q0 + (int64_t)(it0 + k) * kGateThreads + tid;
            if (valid[k]) {
                int32_t mode, count;
                float agree, conf;
                bool bypass;
                gate_row<EM, CONF, (E_T != 0), false>(a[k], w[k], E,
                                                      p.tau_q ? __ldg(p.tau_q + q) : p.tau, p.abstain,
                                                      agree_lut, mode, count, agree, conf, bypass);
                if (p.mode_out) __stcs(p.mode_out + q, mode);
                if (p.count_out) __stcs(p.count_out + q, count);
                if (p.agree_out) __stcs(p.agree_out + q, agree);
                if (p.conf_out) __stcs(p.conf_out + q, conf);
                p.bypass_out[q] = bypass ? 1 : 0;
            }
        }
    }
}

template <int E_T, int CONF, int MAXI, int BATCH>
mosaic_status_t launch(GateArgs& a, cudaStream_t stream) {
    // as many questions per thread as one co-resident wave of blocks needs, capped
    const int64_t wave = (int64_t)num_sms() * kBlocksPerSM * kGateThreads;
    int64_t items = (a.Q + wave - 1) / wave;
    a.items = (int)(items < 1 ? 1 : (items > MAXI ? MAXI : items));
    const int64_t tile = (int64_t)kGateThreads * a.items;
    gate_kernel<E_T, CONF, BATCH><<<(unsigned)((a.Q + tile - 1) / tile), kGateThreads, 0, stream>>>(a);
    count_launch();
    MOSAIC_CUDA_TRY(cudaGetLastError());
    return MOSAIC_OK;
}

template <int CONF>
mosaic_status_t dispatch(GateArgs& a, cudaStream_t s) {
    constexpr int M = kMaxItems;
    switch (a.E) {
        case 1: return launch<1, CONF, M, 4>(a, s);
        case 2: return launch<2, CONF, M, 4>(a, s);
        case 3: return launch<3, CONF, M, 4>(a, s);
        case 4: return launch<4, CONF, M, 4>(a, s);
        case 5: return launch<5, CONF, M, 4>(a, s);
        case 6: return launch<6, CONF, M, 4>(a, s);
        case 7: return launch<7, CONF, M, 4>(a, s);
        case 8: return launch<8, CONF, M, 4>(a, s);
        default: return launch<0, CONF, kMaxItemsWide, 1>(a, s);
    }
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
    switch (conf_mode) {
        case MOSAIC_CONF_WEIGHTED: return dispatch<MOSAIC_CONF_WEIGHTED>(a, s);
        case MOSAIC_CONF_WEIGHTED_ARGMAX: return dispatch<MOSAIC_CONF_WEIGHTED_ARGMAX>(a, s);
        default: return dispatch<MOSAIC_CONF_VOTE>(a, s);
    }
}
