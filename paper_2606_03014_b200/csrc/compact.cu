// compact.cu -- the gate fused with the stream compaction of the surviving questions into a ragged
// batch with cu_seqlens (Alg. 1: line 6 sends the questions that failed the
// gate to the aggregator; BASELINE.json north_star: "stream-compacts the surviving queries into a
// ragged batch with cu_seqlens").  One kernel template serves
//   mosaic_gate_compact[_tau|_ext]  kSrcAnswers : Alg. 1 lines 2-4 + compaction in ONE pass over HBM
//   mosaic_compact                  kSrcBypass  : compaction of a mask computed earlier
//   mosaic_conf_compact             kSrcConf    : threshold on a caller-supplied C(q) + compaction
//
// The kernel is compact_kernel.cuh; its instantiations for the answer-vote source live in the
// compact_inst_c?a?.cu units, this file holds the entry points and the two light sources.
#include "compact_kernel.cuh"

namespace mosaic {
// The instantiation units (compact_inst_c?a?.cu): one per (confidence estimator, abstention) pair.
mosaic_status_t dispatch_gate_c0a0(GateArgs& a, size_t ws_bytes, void* ws, cudaStream_t s);
mosaic_status_t dispatch_gate_c0a1(GateArgs& a, size_t ws_bytes, void* ws, cudaStream_t s);
mosaic_status_t dispatch_gate_c1a0(GateArgs& a, size_t ws_bytes, void* ws, cudaStream_t s);
mosaic_status_t dispatch_gate_c1a1(GateArgs& a, size_t ws_bytes, void* ws, cudaStream_t s);
mosaic_status_t dispatch_gate_c2a0(GateArgs& a, size_t ws_bytes, void* ws, cudaStream_t s);
mosaic_status_t dispatch_gate_c2a1(GateArgs& a, size_t ws_bytes, void* ws, cudaStream_t s);

namespace {

// resident blocks per SM the two light sources (a mask, a confidence) are built for
constexpr int kLightBlocks = kVoterWarps > 8 ? 2 : 3;

mosaic_status_t dispatch_gate(int conf_mode, GateArgs& a, size_t ws_bytes, void* ws, cudaStream_t s) {
    const bool ab = a.abstain.on != 0;
    switch (conf_mode) {
        case MOSAIC_CONF_WEIGHTED:
            return ab ? dispatch_gate_c1a1(a, ws_bytes, ws, s) : dispatch_gate_c1a0(a, ws_bytes, ws, s);
        case MOSAIC_CONF_WEIGHTED_ARGMAX:
            return ab ? dispatch_gate_c2a1(a, ws_bytes, ws, s) : dispatch_gate_c2a0(a, ws_bytes, ws, s);
        default:
            return ab ? dispatch_gate_c0a1(a, ws_bytes, ws, s) : dispatch_gate_c0a0(a, ws_bytes, ws, s);
    }
}

mosaic_status_t write_empty_batch(int64_t* cu_seqlens, int32_t* n_survivors, int64_t* total_tokens,
                                  int32_t* max_seqlen, cudaStream_t s) {
    MOSAIC_CUDA_TRY(cudaMemsetAsync(cu_seqlens, 0, sizeof(int64_t), s));
    MOSAIC_CUDA_TRY(cudaMemsetAsync(n_survivors, 0, sizeof(int32_t), s));
    MOSAIC_CUDA_TRY(cudaMemsetAsync(total_tokens, 0, sizeof(int64_t), s));
    MOSAIC_CUDA_TRY(cudaMemsetAsync(max_seqlen, 0, sizeof(int32_t), s));
    return MOSAIC_OK;
}

// The fused gate + compaction behind mosaic_gate_compact, _tau and _ext.
mosaic_status_t gate_compact_impl(const int32_t* answers, const float* expert_conf,
                                  const int32_t* ctx_len, int64_t Q, int32_t E, float tau,
                                  const float* tau_q, int32_t conf_mode, Abstain abstain,
                                  int32_t* mode_out, int32_t* count_out, float* agree_out,
                                  float* conf_out, uint8_t* bypass_out, int32_t* survivor_idx,
                                  int64_t* cu_seqlens, int32_t* n_survivors, int64_t* total_tokens,
                                  int32_t* max_seqlen, void* workspace, size_t workspace_bytes,
                                  void* cuda_stream) {
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
    a.tau_q = tau_q;
    a.abstain = abstain;
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
    return dispatch_gate(conf_mode, a, workspace_bytes, workspace, s);
}

}  // namespace
}  // namespace mosaic

using namespace mosaic;

extern "C" size_t mosaic_compact_workspace_bytes(int64_t Q) {
    if (Q < 0) return 0;
    // One 16-byte scan state per tile; the smallest tile is kMinTileQuestions questions.  One state
    // per 128-byte line up to 8 MB (the look-back loads then spread over the L2 slices), denser
    // beyond that.
    const size_t tiles = (size_t)((Q + kMinTileQuestions - 1) / kMinTileQuestions) + 1;
    const size_t dense = tiles * sizeof(TileState), wide = tiles * 128;
    const size_t cap = (size_t)8 << 20;
    return sizeof(ScanHeader) + (wide <= cap ? wide : (dense > cap ? dense : cap));
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
    return launch<1, MOSAIC_CONF_VOTE, kSrcBypass, 4, kLightBlocks>(a, workspace_bytes, workspace, s);
}

extern "C" mosaic_status_t mosaic_conf_compact(const float* conf, const int32_t* ctx_len, int64_t Q,
                                               float tau, const float* tau_per_query,
                                               uint8_t* bypass_out, int32_t* survivor_idx,
                                               int64_t* cu_seqlens, int32_t* n_survivors,
                                               int64_t* total_tokens, int32_t* max_seqlen,
                                               void* workspace, size_t workspace_bytes,
                                               void* cuda_stream) {
    if (Q < 0 || Q >= (1ll << 31) || !cu_seqlens || !n_survivors || !total_tokens || !max_seqlen ||
        (!tau_per_query && isnan(tau)))
        return MOSAIC_ERR_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    if (Q == 0) return write_empty_batch(cu_seqlens, n_survivors, total_tokens, max_seqlen, s);
    if (!conf || !ctx_len || !survivor_idx || !workspace || !aligned16(workspace))
        return MOSAIC_ERR_INVALID_ARG;
    GateArgs a{};
    a.conf_in = conf;
    a.ctx_len = ctx_len;
    a.Q = Q;
    a.E = 1;
    a.tau = tau;
    a.tau_q = tau_per_query;
    a.bypass_out = bypass_out;
    a.survivor_idx = survivor_idx;
    a.cu_seqlens = cu_seqlens;
    a.n_survivors = n_survivors;
    a.total_tokens = total_tokens;
    a.max_seqlen = max_seqlen;
    return launch<1, MOSAIC_CONF_VOTE, kSrcConf, 4, kLightBlocks>(a, workspace_bytes, workspace, s);
}

extern "C" mosaic_status_t mosaic_gate_compact(
    const int32_t* answers, const float* expert_conf, const int32_t* ctx_len, int64_t Q, int32_t E,
    float tau, int32_t conf_mode, int32_t* mode_out, int32_t* count_out, float* agree_out,
    float* conf_out, uint8_t* bypass_out, int32_t* survivor_idx, int64_t* cu_seqlens,
    int32_t* n_survivors, int64_t* total_tokens, int32_t* max_seqlen, void* workspace,
    size_t workspace_bytes, void* cuda_stream) {
    return gate_compact_impl(answers, expert_conf, ctx_len, Q, E, tau, nullptr, conf_mode,
                             Abstain{0, 0, 0}, mode_out, count_out, agree_out, conf_out, bypass_out,
                             survivor_idx, cu_seqlens, n_survivors, total_tokens, max_seqlen,
                             workspace, workspace_bytes, cuda_stream);
}

extern "C" mosaic_status_t mosaic_gate_compact_tau(
    const int32_t* answers, const float* expert_conf, const int32_t* ctx_len, int64_t Q, int32_t E,
    const float* tau_per_query, int32_t conf_mode, int32_t* mode_out, int32_t* count_out,
    float* agree_out, float* conf_out, uint8_t* bypass_out, int32_t* survivor_idx,
    int64_t* cu_seqlens, int32_t* n_survivors, int64_t* total_tokens, int32_t* max_seqlen,
    void* workspace, size_t workspace_bytes, void* cuda_stream) {
    if (Q > 0 && !tau_per_query) return MOSAIC_ERR_INVALID_ARG;
    return gate_compact_impl(answers, expert_conf, ctx_len, Q, E, 0.f, tau_per_query, conf_mode,
                             Abstain{0, 0, 0}, mode_out, count_out, agree_out, conf_out, bypass_out,
                             survivor_idx, cu_seqlens, n_survivors, total_tokens, max_seqlen,
                             workspace, workspace_bytes, cuda_stream);
}

extern "C" mosaic_status_t mosaic_gate_compact_ext(
    const int32_t* answers, const float* expert_conf, const int32_t* ctx_len, int64_t Q, int32_t E,
    float tau, const float* tau_per_query, int32_t conf_mode, int32_t abstain_policy,
    int32_t abstain_label, int32_t* mode_out, int32_t* count_out, float* agree_out, float* conf_out,
    uint8_t* bypass_out, int32_t* survivor_idx, int64_t* cu_seqlens, int32_t* n_survivors,
    int64_t* total_tokens, int32_t* max_seqlen, void* workspace, size_t workspace_bytes,
    void* cuda_stream) {
    if (abstain_policy != MOSAIC_ABSTAIN_NONE && abstain_policy != MOSAIC_ABSTAIN_KEEP_K &&
        abstain_policy != MOSAIC_ABSTAIN_SHRINK_K)
        return MOSAIC_ERR_INVALID_ARG;
    const Abstain ab{abstain_policy != MOSAIC_ABSTAIN_NONE ? 1 : 0, abstain_label,
                     abstain_policy == MOSAIC_ABSTAIN_SHRINK_K ? 1 : 0};
    return gate_compact_impl(answers, expert_conf, ctx_len, Q, E, tau_per_query ? 0.f : tau,
                             tau_per_query, conf_mode, ab, mode_out, count_out, agree_out, conf_out,
                             bypass_out, survivor_idx, cu_seqlens, n_survivors, total_tokens,
                             max_seqlen, workspace, workspace_bytes, cuda_stream);
}

#ifdef MOSAIC_GATE_TRACE
extern "C" int mosaic_debug_gate_trace(unsigned long long* out_host, int n) {
    return (int)cudaMemcpyFromSymbol(out_host, mosaic::g_trace, sizeof(unsigned long long) * n);
}
#endif
