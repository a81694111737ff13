// stage.cu -- mosaic_stage_host: the whole confidence-gated aggregator stage (Alg. 1)
// from HOST buffers: H2D copies, gate + compaction, survivors' prefill attention, D2H copies.
// Only marshalling lives here; every step of the path runs in the kernels of gate.cu / attn.cu.
// The survivors go through in chunks of ~8 k tokens (cut anywhere): chunk c+1 is on its way to the device
// and the results of chunk c-1 on their way back while chunk c is in the attention kernel (PCIe
// is full duplex, and at 2.6 GB per C2 step the copies are 94 % of the call).
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>
#include <vector>

#include "common.cuh"

namespace mosaic {
namespace {

#ifndef MOSAIC_STAGE_CHUNK_TOKENS
#define MOSAIC_STAGE_CHUNK_TOKENS 8192
#endif
#ifndef MOSAIC_STAGE_MAX_CHUNKS
#define MOSAIC_STAGE_MAX_CHUNKS 64
#endif
constexpr int kMaxChunks = MOSAIC_STAGE_MAX_CHUNKS;

struct Arena {
    int32_t* answers;
    float* expert_conf;
    int32_t* ctx_len;
    int32_t* mode;
    float* conf;
    uint8_t* bypass;
    int32_t* survivor_idx;
    int64_t* cu_seqlens;
    int32_t* n_survivors;   // 3 scalars share one 32-byte slot
    int64_t* total_tokens;
    int32_t* max_seqlen;
    void* compact_ws;
    size_t compact_ws_bytes;
    void *q, *k, *v, *o;
    float* lse;
    void* attn_ws;
    size_t attn_ws_bytes;
    SeqDesc* views;  // one (q rows, key range) view per (chunk, sequence) overlap
    size_t total;
};

Arena carve_arena(void* base, int64_t Q, int32_t E, int64_t T_cap, int32_t Hq, int32_t Hkv,
                  int32_t D) {
    Arena a{};
    char* p = static_cast<char*>(base);
    size_t off = 0;
    auto take = [&](size_t bytes) {
        char* r = p + off;
        off += (bytes + 255) & ~size_t(255);
        return r;
    };
    a.answers = reinterpret_cast<int32_t*>(take((size_t)Q * E * 4));
    a.expert_conf = reinterpret_cast<float*>(take((size_t)Q * E * 4));
    a.ctx_len = reinterpret_cast<int32_t*>(take((size_t)Q * 4));
    a.mode = reinterpret_cast<int32_t*>(take((size_t)Q * 4));
    a.conf = reinterpret_cast<float*>(take((size_t)Q * 4));
    a.bypass = reinterpret_cast<uint8_t*>(take((size_t)Q));
    a.survivor_idx = reinterpret_cast<int32_t*>(take((size_t)Q * 4));
    a.cu_seqlens = reinterpret_cast<int64_t*>(take((size_t)(Q + 1) * 8));
    char* sc = take(32);
    a.total_tokens = reinterpret_cast<int64_t*>(sc);
    a.n_survivors = reinterpret_cast<int32_t*>(sc + 8);
    a.max_seqlen = reinterpret_cast<int32_t*>(sc + 12);
    a.compact_ws_bytes = mosaic_compact_workspace_bytes(Q);
    a.compact_ws = take(a.compact_ws_bytes);
    a.q = take((size_t)T_cap * Hq * D * 2);
    a.k = take((size_t)T_cap * Hkv * D * 2);
    a.v = take((size_t)T_cap * Hkv * D * 2);
    a.o = take((size_t)T_cap * Hq * D * 2);
    a.lse = reinterpret_cast<float*>(take((size_t)T_cap * Hq * 4));
    const int64_t max_seqs = Q < T_cap ? Q : T_cap;
    a.attn_ws_bytes = mosaic_agg_prefill_attn_workspace_bytes((int32_t)max_seqs, T_cap, Hq, Hkv, D);
    a.attn_ws = take(a.attn_ws_bytes);
    a.views = reinterpret_cast<SeqDesc*>(take((size_t)(max_seqs + kMaxChunks + 1) * sizeof(SeqDesc)));
    a.total = off;
    return a;
}

// Copy streams and events of the chunk pipeline (one set per process; the call is synchronous,
// so one call uses them at a time -- concurrent calls serialise on the mutex).
struct Pipe {
    cudaStream_t in = nullptr, out = nullptr;
    cudaEvent_t ev_in[kMaxChunks], ev_out[kMaxChunks], ev_ready;
    int device = -1;
    bool ok = false;
    std::mutex mu;
};
Pipe& pipe() {
    static Pipe p;
    return p;
}
bool pipe_init(Pipe& p) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return false;
    if (p.ok && p.device == dev) return true;
    if (p.ok) return false;  // one device per process (one process per GPU)
    if (cudaStreamCreateWithFlags(&p.in, cudaStreamNonBlocking) != cudaSuccess) return false;
    if (cudaStreamCreateWithFlags(&p.out, cudaStreamNonBlocking) != cudaSuccess) return false;
    for (int i = 0; i < kMaxChunks; ++i) {
        if (cudaEventCreateWithFlags(&p.ev_in[i], cudaEventDisableTiming) != cudaSuccess) return false;
        if (cudaEventCreateWithFlags(&p.ev_out[i], cudaEventDisableTiming) != cudaSuccess) return false;
    }
    if (cudaEventCreateWithFlags(&p.ev_ready, cudaEventDisableTiming) != cudaSuccess) return false;
    p.device = dev;
    p.ok = true;
    return true;
}

}  // namespace
}  // namespace mosaic

using namespace mosaic;

extern "C" size_t mosaic_stage_host_arena_bytes(int64_t Q, int32_t E, int64_t T_cap, int32_t Hq,
                                                int32_t Hkv, int32_t D) {
    if (Q < 0 || E < 1 || T_cap < 0 || Hq < 1 || Hkv < 1 || D < 1) return 0;
    return carve_arena(nullptr, Q, E, T_cap, Hq, Hkv, D).total;
}

extern "C" mosaic_status_t mosaic_stage_host(
    const int32_t* answers_h, const float* expert_conf_h, const int32_t* ctx_len_h, int64_t Q,
    int32_t E, float tau, int32_t conf_mode, int32_t* mode_h, float* conf_h, uint8_t* bypass_h,
    int32_t* survivor_idx_h, int64_t* cu_seqlens_h, int32_t* n_survivors_h,
    int64_t* total_tokens_h, int32_t* max_seqlen_h, int32_t max_attn_seqs, const void* q_h,
    const void* k_h, const void* v_h, int64_t T_cap, int32_t Hq, int32_t Hkv, int32_t D,
    float softmax_scale, void* o_h, float* lse_h, void* arena, size_t arena_bytes,
    void* cuda_stream) {
    if (Q < 0 || Q >= (1ll << 31) || E < 1 || E > MOSAIC_MAX_EXPERTS || T_cap < 0 || Hq < 1 ||
        Hkv < 1 || Hq % Hkv != 0)
        return MOSAIC_ERR_INVALID_ARG;
    if (D != 64 && D != 128) return MOSAIC_ERR_UNSUPPORTED;
    if (!bypass_h || !survivor_idx_h || !cu_seqlens_h || !n_survivors_h || !total_tokens_h ||
        !max_seqlen_h || !arena || !aligned16(arena))
        return MOSAIC_ERR_INVALID_ARG;
    if (Q > 0 && (!answers_h || !ctx_len_h)) return MOSAIC_ERR_INVALID_ARG;
    if (conf_mode == MOSAIC_CONF_WEIGHTED && Q > 0 && !expert_conf_h) return MOSAIC_ERR_INVALID_ARG;
    Arena a = carve_arena(arena, Q, E, T_cap, Hq, Hkv, D);
    if (arena_bytes < a.total) return MOSAIC_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const cudaMemcpyKind H2D = cudaMemcpyHostToDevice, D2H = cudaMemcpyDeviceToHost;

    if (Q > 0) {
        MOSAIC_CUDA_TRY(cudaMemcpyAsync(a.answers, answers_h, (size_t)Q * E * 4, H2D, s));
        if (conf_mode == MOSAIC_CONF_WEIGHTED)
            MOSAIC_CUDA_TRY(cudaMemcpyAsync(a.expert_conf, expert_conf_h, (size_t)Q * E * 4, H2D, s));
        MOSAIC_CUDA_TRY(cudaMemcpyAsync(a.ctx_len, ctx_len_h, (size_t)Q * 4, H2D, s));
    }
    mosaic_status_t st = mosaic_gate_compact(
        a.answers, conf_mode == MOSAIC_CONF_WEIGHTED ? a.expert_conf : nullptr, a.ctx_len, Q, E, tau,
        conf_mode, a.mode, nullptr, nullptr, a.conf, a.bypass, a.survivor_idx, a.cu_seqlens,
        a.n_survivors, a.total_tokens, a.max_seqlen, a.compact_ws, a.compact_ws_bytes, s);
    if (st != MOSAIC_OK) return st;

    struct {
        int64_t total;
        int32_t S;
        int32_t max_len;
    } sc;
    MOSAIC_CUDA_TRY(cudaMemcpyAsync(&sc, a.total_tokens, 16, D2H, s));
    if (Q > 0) {
        if (mode_h) MOSAIC_CUDA_TRY(cudaMemcpyAsync(mode_h, a.mode, (size_t)Q * 4, D2H, s));
        if (conf_h) MOSAIC_CUDA_TRY(cudaMemcpyAsync(conf_h, a.conf, (size_t)Q * 4, D2H, s));
        MOSAIC_CUDA_TRY(cudaMemcpyAsync(bypass_h, a.bypass, (size_t)Q, D2H, s));
    }
    MOSAIC_CUDA_TRY(cudaStreamSynchronize(s));
    *n_survivors_h = sc.S;
    *total_tokens_h = sc.total;
    *max_seqlen_h = sc.max_len;
    const int64_t S = sc.S;
    if (S > 0) MOSAIC_CUDA_TRY(cudaMemcpyAsync(survivor_idx_h, a.survivor_idx, (size_t)S * 4, D2H, s));
    MOSAIC_CUDA_TRY(cudaMemcpyAsync(cu_seqlens_h, a.cu_seqlens, (size_t)(S + 1) * 8, D2H, s));
    MOSAIC_CUDA_TRY(cudaStreamSynchronize(s));

    const int64_t n_att = (max_attn_seqs < 0 || max_attn_seqs > S) ? S : max_attn_seqs;
    if (n_att == 0) return MOSAIC_OK;
    const int64_t T = cu_seqlens_h[n_att];
    if (T == 0) return MOSAIC_OK;
    if (T > T_cap) return MOSAIC_ERR_WORKSPACE_TOO_SMALL;
    if (!q_h || !k_h || !v_h || !o_h || !lse_h) return MOSAIC_ERR_INVALID_ARG;
    // Chunks of about T / n_chunks TOKENS each, cut anywhere -- also inside a sequence (at least
    // ~8 k tokens a chunk: smaller ones would make the attention launches and the copies latency-
    // bound).  The packed order is the upload order, so when chunk c has arrived every key its q
    // rows may see has: the rows of sequence i inside the chunk, [r0, r1), attend that sequence's
    // keys [0, r1) (bottom-right alignment, reading N2-1) -- one view per (chunk,
    // sequence) overlap.  Cutting by tokens keeps the chunks equal (the first upload and the last
    // attention + download are what the pipeline cannot hide) whatever the sequence lengths are.
    Pipe& pp = pipe();
    std::lock_guard<std::mutex> lock(pp.mu);
    if (!pipe_init(pp)) return MOSAIC_ERR_CUDA;
    int n_chunks = (int)(T / MOSAIC_STAGE_CHUNK_TOKENS);
    n_chunks = n_chunks < 1 ? 1 : (n_chunks > kMaxChunks ? kMaxChunks : n_chunks);
    std::vector<SeqDesc> views;
    int first_view[kMaxChunks + 1];
    int64_t bound[kMaxChunks + 1];
    {
        int64_t seq = 0;
        for (int c = 0; c <= n_chunks; ++c) bound[c] = T * c / n_chunks;
        for (int c = 0; c < n_chunks; ++c) {
            first_view[c] = (int)views.size();
            const int64_t ta = bound[c], tb = bound[c + 1];
            while (seq < n_att && cu_seqlens_h[seq + 1] <= ta) ++seq;
            for (int64_t i = seq; i < n_att && cu_seqlens_h[i] < tb; ++i) {
                const int64_t b0 = cu_seqlens_h[i], b1 = cu_seqlens_h[i + 1];
                const int64_t r0 = ta > b0 ? ta : b0, r1 = tb < b1 ? tb : b1;
                if (r1 > r0) views.push_back(SeqDesc{r0, b0, (int32_t)(r1 - r0), (int32_t)(r1 - b0)});
            }
        }
        first_view[n_chunks] = (int)views.size();
    }
    if (views.size() > (size_t)(n_att + kMaxChunks)) return MOSAIC_ERR_WORKSPACE_TOO_SMALL;
    MOSAIC_CUDA_TRY(cudaMemcpyAsync(a.views, views.data(), views.size() * sizeof(SeqDesc), H2D, s));
    // the copy streams start after everything this call has enqueued on s so far
    MOSAIC_CUDA_TRY(cudaEventRecord(pp.ev_ready, s));
    MOSAIC_CUDA_TRY(cudaStreamWaitEvent(pp.in, pp.ev_ready, 0));
    MOSAIC_CUDA_TRY(cudaStreamWaitEvent(pp.out, pp.ev_ready, 0));
    const size_t q_row = (size_t)Hq * D * 2, kv_row = (size_t)Hkv * D * 2;
    for (int c = 0; c < n_chunks; ++c) {
        const int64_t t0 = bound[c], t1 = bound[c + 1];
        const int n_views = first_view[c + 1] - first_view[c];
        if (t1 == t0 || n_views == 0) continue;
        const size_t rows = (size_t)(t1 - t0);
        auto at = [](const void* base, size_t off) { return static_cast<const char*>(base) + off; };
        auto at_w = [](void* base, size_t off) { return static_cast<char*>(base) + off; };
        MOSAIC_CUDA_TRY(cudaMemcpyAsync(at_w(a.q, t0 * q_row), at(q_h, t0 * q_row), rows * q_row, H2D, pp.in));
        MOSAIC_CUDA_TRY(cudaMemcpyAsync(at_w(a.k, t0 * kv_row), at(k_h, t0 * kv_row), rows * kv_row, H2D, pp.in));
        MOSAIC_CUDA_TRY(cudaMemcpyAsync(at_w(a.v, t0 * kv_row), at(v_h, t0 * kv_row), rows * kv_row, H2D, pp.in));
        MOSAIC_CUDA_TRY(cudaEventRecord(pp.ev_in[c], pp.in));
        MOSAIC_CUDA_TRY(cudaStreamWaitEvent(s, pp.ev_in[c], 0));
        // K and V are declared only as far as this chunk's last token (total_k_tokens = t1): the
        // last 128-row K / V box of the chunk reaches past it into rows whose copy (chunk c + 1)
        // may still be in flight -- those rows are masked, but a masked P = 0 times a stale NaN
        // pattern in V would still be NaN -- and rows past the tensor map's extent are zero-filled
        // by the TMA unit instead of being read.
        st = attn_impl(a.q, a.k, a.v, nullptr, nullptr, a.views + first_view[c], n_views, T, t1,
                       sc.max_len, Hq, Hkv, D, softmax_scale, /*causal=*/1, a.o, a.lse, a.attn_ws,
                       a.attn_ws_bytes, s);
        if (st != MOSAIC_OK) {
            cudaStreamSynchronize(pp.in);
            cudaStreamSynchronize(s);
            cudaStreamSynchronize(pp.out);
            return st;
        }
        MOSAIC_CUDA_TRY(cudaEventRecord(pp.ev_out[c], s));
        MOSAIC_CUDA_TRY(cudaStreamWaitEvent(pp.out, pp.ev_out[c], 0));
        MOSAIC_CUDA_TRY(cudaMemcpyAsync(at_w(o_h, t0 * q_row), at(a.o, t0 * q_row), rows * q_row, D2H, pp.out));
        // LSE is [Hq, T]: the chunk's columns of every head
        MOSAIC_CUDA_TRY(cudaMemcpy2DAsync(lse_h + t0, (size_t)T * 4, a.lse + t0, (size_t)T * 4,
                                          rows * 4, (size_t)Hq, D2H, pp.out));
    }
    MOSAIC_CUDA_TRY(cudaStreamSynchronize(pp.in));
    MOSAIC_CUDA_TRY(cudaStreamSynchronize(s));
    MOSAIC_CUDA_TRY(cudaStreamSynchronize(pp.out));
    return MOSAIC_OK;
}
