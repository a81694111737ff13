/*
 * mosaic.h -- C ABI of the confidence-gated aggregator stage of MOSAIC
 * (arxiv/paper_2606_03014, "PAPER.md" cited as P:Lnn) for one NVIDIA B200 (sm_100a).
 *
 * The stage (Sec. 4.2 "adaptive aggregation"; Alg. 1):
 *
 *     for every question q with extracted expert answers a_1..a_k:
 *         C(q) = max_a |{i : a_i = a}| / k                    (C_vote)
 *         if C(q) >= tau:  y(q) = majority({a_i})             (aggregator skipped)
 *         else:            y(q) = Aggregator(q, {a_i})        (the survivors)
 *
 * and the aggregator's prefill attention over each survivor's concatenated context (question
 * prompt + all expert traces), which BASELINE.json's north_star fixes as variable-length
 * causal grouped-query attention producing bf16 O and fp32 row logsumexp.
 *
 * Conventions (all entry points)
 *   - Pointers marked [dev] are CUDA device pointers, 16-byte aligned, owned by the caller.
 *     Pointers marked [host] are ordinary host pointers.  The library allocates no device
 *     memory; scratch comes from caller workspaces sized by the *_workspace_bytes helpers, whose
 *     contents may be arbitrary on entry.  No call depends on an earlier one: what the library
 *     keeps per process is caches only (kernel attributes, occupancy figures, the tensor-map
 *     encoder entry point) and, for mosaic_stage_host alone, two copy streams and their events,
 *     created on first use and kept until the process exits.
 *   - cuda_stream is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls
 *     marked "async" only enqueue work on that stream and never synchronise.
 *   - Errors are return codes; nothing is thrown or printed.  Host-visible arguments are
 *     validated (MOSAIC_ERR_INVALID_ARG / MOSAIC_ERR_UNSUPPORTED / MOSAIC_ERR_WORKSPACE_TOO_SMALL);
 *     device-side contents (monotone cu_seqlens, non-negative ctx_len) are trusted.
 *     MOSAIC_ERR_CUDA reports a failed CUDA call (mosaic_last_cuda_error() gives its code).
 *   - There is no CPU fallback: without a CUDA device every compute call returns MOSAIC_ERR_CUDA.
 */
#ifndef MOSAIC_H_
#define MOSAIC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    MOSAIC_OK = 0,
    MOSAIC_ERR_INVALID_ARG = 1,
    MOSAIC_ERR_UNSUPPORTED = 2,
    MOSAIC_ERR_WORKSPACE_TOO_SMALL = 3,
    MOSAIC_ERR_CUDA = 4
} mosaic_status_t;

/* Confidence estimator C(q) used by the gate (the gate "is agnostic to the choice of
 * confidence estimator"). */
enum {
    MOSAIC_CONF_VOTE = 0,     /* C_vote = plurality fraction, the paper's instantiation */
    MOSAIC_CONF_WEIGHTED = 1, /* extension (reading G-10): weight share of the modal answer */
    MOSAIC_CONF_WEIGHTED_ARGMAX = 2 /* extension (reading N3-3): the answer is the label with the
                                       LARGEST weight sum (ties -> smallest label), C its share */
};

/* What a failed Extract (Alg. 1 line 1) does to the vote (reading N3-2): an
 * expert whose label equals the caller's sentinel abstains and is left out of every tally. */
enum {
    MOSAIC_ABSTAIN_NONE = 0,     /* no sentinel: every label is an answer (reading G-6)               */
    MOSAIC_ABSTAIN_KEEP_K = 1,   /* C still divides by the k experts recruited (P:L182 literally)     */
    MOSAIC_ABSTAIN_SHRINK_K = 2  /* C divides by the experts that answered                            */
};

#define MOSAIC_MAX_EXPERTS 32

/* ---------------------------------------------------------------------------------------------
 * mosaic_gate -- Alg. 1 lines 2-4 for Q questions, async.
 *
 *   answers     [dev] int32 [Q, E] row-major (question-major): a_i = Extract(E_i(q)).
 *                     Any int32 is a label; only equality matters.
 *   expert_conf [dev] fp32 [Q, E] per-response weights w; required iff conf_mode != VOTE, else
 *                     may be NULL.
 *   Q, E              0 <= Q < 2^31, 1 <= E <= MOSAIC_MAX_EXPERTS (the paper's k; k = 3 at P:L331).
 *   tau               threshold, compared in fp32 (reading G-4); NaN -> INVALID_ARG.
 *   mode_out    [dev] int32 [Q]  majority({a_i}); ties -> smallest label (reading G-2). May be NULL.
 *   count_out   [dev] int32 [Q]  c* = max_a |{i: a_i = a}|.                        May be NULL.
 *   agree_out   [dev] fp32  [Q]  C_vote = fl32(c*) / fl32(E), one IEEE division.    May be NULL.
 *   conf_out    [dev] fp32  [Q]  the C(q) the gate compared: agree (VOTE) or
 *                                fl32(sum_{i: a_i = mode} w_i / sum_i w_i) with binary64 sums in
 *                                expert order, agree when sum_i w_i <= 0 (WEIGHTED).  May be NULL.
 *                                WEIGHTED_ARGMAX: the same share with mode = the label whose
 *                                weight sum is largest (ties -> smallest label); count_out is
 *                                then that label's votes and agree_out = count / E; when
 *                                sum_i w_i <= 0 the call falls back to VOTE for the question.
 *   bypass_out  [dev] uint8 [Q]  1 iff C(q) >= tau (aggregator skipped, answer = mode). Required.
 *
 * Q == 0 is a successful no-op.
 * ------------------------------------------------------------------------------------------- */
mosaic_status_t mosaic_gate(const int32_t* answers, const float* expert_conf, int64_t Q, int32_t E,
                            float tau, int32_t conf_mode, int32_t* mode_out, int32_t* count_out,
                            float* agree_out, float* conf_out, uint8_t* bypass_out,
                            void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_compact -- Alg. 1 line 6: the questions that failed the gate become the
 * aggregator's ragged batch (north_star: "stream-compacts the surviving queries into a ragged
 * batch with cu_seqlens"), async.  Stable: ascending question index (reading G-11).
 *
 *   bypass       [dev] uint8 [Q]   from mosaic_gate (0 = survivor).
 *   ctx_len      [dev] int32 [Q]   tokens in question q's aggregator context (prompt + all expert
 *                                  traces, reading G-12), >= 0.
 *   survivor_idx [dev] int32 [Q]   capacity Q; first S entries written.
 *   cu_seqlens   [dev] int64 [Q+1] capacity Q+1; first S+1 entries written: cu[0] = 0,
 *                                  cu[j+1] = cu[j] + ctx_len[survivor_idx[j]].
 *   n_survivors  [dev] int32 [1]   S.
 *   total_tokens [dev] int64 [1]   cu[S].
 *   max_seqlen   [dev] int32 [1]   max_j ctx_len[survivor_idx[j]] (0 if S == 0).
 *   workspace    [dev] >= mosaic_compact_workspace_bytes(Q) bytes, contents arbitrary.
 *
 * Q == 0 writes S = 0, cu[0] = 0, total_tokens = 0, max_seqlen = 0.
 * ------------------------------------------------------------------------------------------- */
size_t mosaic_compact_workspace_bytes(int64_t Q);
mosaic_status_t mosaic_compact(const uint8_t* bypass, const int32_t* ctx_len, int64_t Q,
                               int32_t* survivor_idx, int64_t* cu_seqlens, int32_t* n_survivors,
                               int64_t* total_tokens, int32_t* max_seqlen, void* workspace,
                               size_t workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_compact_static -- mosaic_compact (Alg. 1 line 6; same arguments, same results
 * bit for bit) WITHOUT a caller workspace, for callers that cannot allocate device memory (code
 * under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  The scan
 * state lives in a 1 MiB device array inside the library, which every GPU that loads the library
 * holds until the process exits; the call allocates nothing (no cudaMalloc / cudaFree / allocating
 * library routine) and zeroes the part of the array it uses on the stream before it scans.
 *
 *   Q > MOSAIC_COMPACT_STATIC_MAX_Q returns MOSAIC_ERR_WORKSPACE_TOO_SMALL (the array holds the
 *   scan state of at most that many questions); use mosaic_compact with a workspace there.
 *   Every call on a device shares the one array: calls that overlap on the GPU (different
 *   streams, several host threads) RACE and give undefined results -- keep them on one stream or
 *   order them with events.  Calls on different devices are independent.
 *   The first call on a device asks the runtime for the array's address (cudaGetSymbolAddress, which
 *   may load the module): make that call outside a stream capture; later calls only launch kernels.
 * ------------------------------------------------------------------------------------------- */
#define MOSAIC_COMPACT_STATIC_MAX_Q (1 << 22)
mosaic_status_t mosaic_compact_static(const uint8_t* bypass, const int32_t* ctx_len, int64_t Q,
                                      int32_t* survivor_idx, int64_t* cu_seqlens,
                                      int32_t* n_survivors, int64_t* total_tokens,
                                      int32_t* max_seqlen, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_gate_compact -- mosaic_gate followed by mosaic_compact in ONE kernel launch (the
 * bypass mask never makes a round trip through HBM before the scan), async.  Same arguments,
 * same results bit for bit; bypass_out may be NULL here.  Workspace: mosaic_compact's.
 * ------------------------------------------------------------------------------------------- */
mosaic_status_t mosaic_gate_compact(const int32_t* answers, const float* expert_conf,
                                    const int32_t* ctx_len, int64_t Q, int32_t E, float tau,
                                    int32_t conf_mode, int32_t* mode_out, int32_t* count_out,
                                    float* agree_out, float* conf_out, uint8_t* bypass_out,
                                    int32_t* survivor_idx, int64_t* cu_seqlens,
                                    int32_t* n_survivors, int64_t* total_tokens,
                                    int32_t* max_seqlen, void* workspace, size_t workspace_bytes,
                                    void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_agg_prefill_attn -- the aggregator's prefill attention over the survivors' packed
 * contexts (math fixed by north_star), async.  For sequence s with tokens
 * t0 = cu_seqlens[s] .. t0 + L - 1, q head h, kv head g = h / (Hq / Hkv), row i:
 *
 *     x_j = softmax_scale * sum_d Q[t0+i,h,d] K[t0+j,g,d],   j = 0..i  (causal, sequence-local)
 *     LSE = ln sum_j exp(x_j)                    O_d = sum_j exp(x_j - LSE) V[t0+j,g,d]
 *
 *   q            [dev] bf16 [T, Hq, D]   packed, D fastest, no padding between sequences.
 *   k, v         [dev] bf16 [T, Hkv, D]
 *   cu_seqlens   [dev] int64 [n_seqs+1]  cu[0] = 0, non-decreasing, cu[n_seqs] = total_tokens.
 *   n_seqs, total_tokens, max_seqlen     HOST values; max_seqlen >= every sequence length (only
 *                                        its sign is checked today: the work list is built on
 *                                        the device from cu_seqlens).  0 <= total_tokens < 2^31.
 *   Hq, Hkv, D                           Hq % Hkv == 0; D in {64, 128} (else UNSUPPORTED).
 *   softmax_scale                        finite fp32 (the configs use 1/sqrt(D)).
 *   o            [dev] bf16 [T, Hq, D]   fp32 accumulator rounded to nearest-even.
 *   lse          [dev] fp32 [Hq, T]      natural log, of the scaled scores.
 *   workspace    [dev] >= mosaic_agg_prefill_attn_workspace_bytes(...) bytes, contents arbitrary.
 *
 * n_seqs == 0 or total_tokens == 0 is a successful no-op; zero-length sequences contribute no rows.
 * ------------------------------------------------------------------------------------------- */
size_t mosaic_agg_prefill_attn_workspace_bytes(int32_t n_seqs, int64_t total_tokens, int32_t Hq,
                                               int32_t Hkv, int32_t D);
mosaic_status_t mosaic_agg_prefill_attn(const void* q, const void* k, const void* v,
                                        const int64_t* cu_seqlens, int32_t n_seqs,
                                        int64_t total_tokens, int32_t max_seqlen, int32_t Hq,
                                        int32_t Hkv, int32_t D, float softmax_scale, void* o,
                                        float* lse, void* workspace, size_t workspace_bytes,
                                        void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_gate_compact_tau -- SURVEY.md section 8(f) N3 (a "next" row): mosaic_gate_compact with a
 * threshold PER QUESTION.  The paper fixes one skip criterion per task in advance and names that
 * as a limitation (P:L188 invites other criteria); with tau_per_query[q] = table[task(q)]
 * a mixed batch of tasks is gated in one call.  Alg. 1 line 4 becomes
 *     bypass[q] = conf[q] >= tau_per_query[q]      (fp32 compare; a NaN threshold never bypasses);
 * vote, mode and confidence are mosaic_gate's.
 *   tau_per_query [dev] fp32 [Q]; every other argument as mosaic_gate_compact.
 * ------------------------------------------------------------------------------------------- */
mosaic_status_t mosaic_gate_compact_tau(const int32_t* answers, const float* expert_conf,
                                        const int32_t* ctx_len, int64_t Q, int32_t E,
                                        const float* tau_per_query, int32_t conf_mode,
                                        int32_t* mode_out, int32_t* count_out, float* agree_out,
                                        float* conf_out, uint8_t* bypass_out, int32_t* survivor_idx,
                                        int64_t* cu_seqlens, int32_t* n_survivors,
                                        int64_t* total_tokens, int32_t* max_seqlen, void* workspace,
                                        size_t workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_gate_compact_ext -- SURVEY.md section 8(f) N3: mosaic_gate_compact with every optional
 * estimator setting in one call.  P:L188: the gate "is agnostic to the choice of confidence
 * estimator"; `Extract` may fail; a static tau is a stated limitation.
 *   tau_per_query  [dev] fp32 [Q] or NULL (then `tau` for every question), as mosaic_gate_compact_tau.
 *   conf_mode      MOSAIC_CONF_VOTE / _WEIGHTED / _WEIGHTED_ARGMAX.
 *   abstain_policy MOSAIC_ABSTAIN_*; abstain_label is the sentinel `Extract` returns on failure.
 *                  An abstaining expert is not counted for any label, cannot be the mode, and adds
 *                  no weight to a label; with KEEP_K the denominators stay E (votes) and
 *                  sum over ALL experts of w (weights), with SHRINK_K they run over the experts
 *                  that answered.  If every expert abstains: mode = abstain_label, count = 0,
 *                  agree = conf = 0 (the question bypasses only when tau <= 0).
 * Every other argument, the outputs and the errors as mosaic_gate_compact.
 * ------------------------------------------------------------------------------------------- */
mosaic_status_t mosaic_gate_compact_ext(const int32_t* answers, const float* expert_conf,
                                        const int32_t* ctx_len, int64_t Q, int32_t E, float tau,
                                        const float* tau_per_query, int32_t conf_mode,
                                        int32_t abstain_policy, int32_t abstain_label,
                                        int32_t* mode_out, int32_t* count_out, float* agree_out,
                                        float* conf_out, uint8_t* bypass_out, int32_t* survivor_idx,
                                        int64_t* cu_seqlens, int32_t* n_survivors,
                                        int64_t* total_tokens, int32_t* max_seqlen, void* workspace,
                                        size_t workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_conf_compact -- SURVEY.md section 8(f) N3: Alg. 1 lines 4-6 on a confidence the CALLER
 * computed ("response-level uncertainty, or context-aware features" may replace C_vote):
 *     bypass[q] = conf[q] >= tau (or tau_per_query[q]), fp32 compare, NaN never bypasses;
 * then the compaction of mosaic_compact, in the same launch.
 *   conf [dev] fp32 [Q]; tau_per_query [dev] fp32 [Q] or NULL; bypass_out [dev] uint8 [Q] or NULL;
 *   the remaining arguments as mosaic_compact.  NaN `tau` without tau_per_query -> INVALID_ARG.
 * ------------------------------------------------------------------------------------------- */
mosaic_status_t mosaic_conf_compact(const float* conf, const int32_t* ctx_len, int64_t Q, float tau,
                                    const float* tau_per_query, uint8_t* bypass_out,
                                    int32_t* survivor_idx, int64_t* cu_seqlens, int32_t* n_survivors,
                                    int64_t* total_tokens, int32_t* max_seqlen, void* workspace,
                                    size_t workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_agg_prefill_attn_kv -- SURVEY.md section 8(f) N2 (a "next" row): the same attention with
 * the q rows and the keys of a sequence packed separately, for prefix-cached prompts and chunked
 * prefill of the aggregator's long contexts (32 k-class windows): sequence s has Lq q rows
 * (cu_seqlens_q) and Lk >= Lq keys (cu_seqlens_k), the q rows being the LAST Lq positions, so
 * row i sees keys j <= i + (Lk - Lq) ("bottom-right" causal alignment, reading N2-1).
 * Lk = Lq for every sequence is mosaic_agg_prefill_attn.  Together with the exported LSE this is
 * what split-KV / chunked prefill merges are built from.
 *
 *   q [dev] bf16 [total_q_tokens, Hq, D]; k, v [dev] bf16 [total_k_tokens, Hkv, D];
 *   cu_seqlens_q, cu_seqlens_k [dev] int64 [n_seqs + 1]; max_seqlen_q >= every Lq;
 *   o [dev] bf16 [total_q_tokens, Hq, D]; lse [dev] fp32 [Hq, total_q_tokens];
 *   workspace >= mosaic_agg_prefill_attn_workspace_bytes(n_seqs, total_q_tokens, ...).
 *   causal: 1 as above; 0: every q row sees ALL Lk keys of its sequence (the partial result of a
 *   block of earlier keys in a split-KV prefill; Lk >= 1 wherever Lq >= 1) -- see mosaic_lse_merge.
 * Everything else (alignment, D, errors, asynchrony) as mosaic_agg_prefill_attn.  Lk < Lq with
 * causal = 1 is outside the contract and cannot be checked on the host (the lengths are device
 * data): the kernel then visits no key tile for the q tiles that see none and finishes, but the
 * O / LSE rows of such a sequence are unspecified.
 * ------------------------------------------------------------------------------------------- */
mosaic_status_t mosaic_agg_prefill_attn_kv(const void* q, const void* k, const void* v,
                                           const int64_t* cu_seqlens_q,
                                           const int64_t* cu_seqlens_k, int32_t n_seqs,
                                           int64_t total_q_tokens, int64_t total_k_tokens,
                                           int32_t max_seqlen_q, int32_t Hq, int32_t Hkv, int32_t D,
                                           float softmax_scale, int32_t causal, void* o, float* lse,
                                           void* workspace, size_t workspace_bytes,
                                           void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_lse_merge -- SURVEY.md section 8(f) N2: merges the partial attention results of two
 * DISJOINT key sets A, B for the same q rows (split-KV / chunked prefill):
 *     LSE = ln(e^LSE_a + e^LSE_b),   O = O_a e^(LSE_a - LSE) + O_b e^(LSE_b - LSE).
 * This is exact: a row's softmax weights over A u B are its weights over A times e^(LSE_a - LSE)
 * (north_star's LSE is exported for this).  LSE = -inf marks an empty partial (weight 0; its O
 * is not read as a number).
 *
 *   o_a, o_b [dev] bf16 [total_tokens, Hq, D] (16-byte aligned), lse_a, lse_b [dev] fp32
 *   [Hq, total_tokens];  o, lse: outputs of the same shapes (o may alias o_a or o_b, lse may alias
 *   lse_a or lse_b).  D a multiple of 8.  fp32 arithmetic, O rounded to nearest-even bf16.
 * ------------------------------------------------------------------------------------------- */
mosaic_status_t mosaic_lse_merge(const void* o_a, const float* lse_a, const void* o_b,
                                 const float* lse_b, int64_t total_tokens, int32_t Hq, int32_t D,
                                 void* o, float* lse, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_lse_merge_n -- mosaic_lse_merge for n partial results over pairwise DISJOINT key sets
 * (the blocks of a split-KV pass): LSE = ln sum_p e^LSE_p, O = sum_p O_p e^(LSE_p - LSE).
 *   o_parts [dev] bf16 [n_parts, total_tokens, Hq, D] (16-byte aligned), lse_parts [dev] fp32
 *   [n_parts, Hq, total_tokens]; o, lse: outputs as mosaic_lse_merge (must not alias the inputs).
 *   n_parts >= 1.  A row all of whose partials are empty (-inf) gets O = 0, LSE = -inf.
 * ------------------------------------------------------------------------------------------- */
mosaic_status_t mosaic_lse_merge_n(const void* o_parts, const float* lse_parts, int32_t n_parts,
                                   int64_t total_tokens, int32_t Hq, int32_t D, void* o, float* lse,
                                   void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_agg_prefill_attn_chunked -- SURVEY.md section 8(f) N2: mosaic_agg_prefill_attn with every
 * sequence taken in chunks of q_chunk query rows (chunked prefill of the aggregator's long
 * contexts: 32 k-token window at P:L194, 45 312 tokens possible in configs[2]).  Chunk c of a
 * sequence is rows [c q_chunk, min(L, (c+1) q_chunk)) against keys [0, that end): each row sees
 * exactly the keys the plain prefill shows it, so O and LSE are the plain prefill's (same
 * tolerances); all chunks of all sequences run in ONE launch of the attention kernel.
 *   q_chunk >= 1 (a multiple of 256 keeps the tiles of the plain prefill); every other argument as
 *   mosaic_agg_prefill_attn; workspace >= mosaic_agg_prefill_attn_chunked_workspace_bytes(...).
 * ------------------------------------------------------------------------------------------- */
size_t mosaic_agg_prefill_attn_chunked_workspace_bytes(int32_t n_seqs, int64_t total_tokens,
                                                       int32_t q_chunk, int32_t Hq, int32_t Hkv,
                                                       int32_t D);
mosaic_status_t mosaic_agg_prefill_attn_chunked(const void* q, const void* k, const void* v,
                                                const int64_t* cu_seqlens, int32_t n_seqs,
                                                int64_t total_tokens, int32_t max_seqlen,
                                                int32_t Hq, int32_t Hkv, int32_t D,
                                                float softmax_scale, int32_t q_chunk, void* o,
                                                float* lse, void* workspace,
                                                size_t workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_agg_prefill_attn_shared_prefix -- SURVEY.md section 8(f) N2, the shared-prefix cascade:
 * one aggregator serves all survivors with a common prompt template in front of every
 * context (`Aggregator(q, {a_i})`), so the first prefix_len keys of every sequence are the
 * SAME block.  Sequence s is  prefix ++ own tokens;  the call computes the rows of the own tokens
 * (the prefix's rows are the same for every sequence and are the caller's, once): row i of
 * sequence s sees all prefix_len prefix keys and its own keys j <= i.
 *   q, o [dev] bf16 [total_tokens, Hq, D], k, v [dev] bf16 [total_tokens, Hkv, D], cu_seqlens,
 *   lse: the sequences' OWN tokens, as mosaic_agg_prefill_attn;
 *   k_prefix, v_prefix [dev] bf16 [prefix_len, Hkv, D] (16-byte aligned); prefix_len >= 0.
 * One launch of the attention kernel: a q tile visits the shared block's K / V tiles (a few MB that
 * stay in L2: read from HBM once for the whole batch) and then its sequence's own, in one online
 * softmax -- no partial results, no merge.
 *   workspace >= mosaic_agg_prefill_attn_shared_prefix_workspace_bytes(...).  Errors, alignment
 *   and asynchrony as mosaic_agg_prefill_attn.
 * ------------------------------------------------------------------------------------------- */
size_t mosaic_agg_prefill_attn_shared_prefix_workspace_bytes(int32_t n_seqs, int64_t total_tokens,
                                                             int32_t Hq, int32_t Hkv, int32_t D);
mosaic_status_t mosaic_agg_prefill_attn_shared_prefix(
    const void* q, const void* k_prefix, const void* v_prefix, int32_t prefix_len, const void* k,
    const void* v, const int64_t* cu_seqlens, int32_t n_seqs, int64_t total_tokens,
    int32_t max_seqlen, int32_t Hq, int32_t Hkv, int32_t D, float softmax_scale, void* o, float* lse,
    void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_agg_decode_attn -- SURVEY.md section 8(f) N2: the aggregator's GQA decode attention, one
 * new q token per sequence against all Lk cached keys of that sequence (decode follows prefill in
 * the aggregator): O[s,h,:] = softmax_j(scale q_{s,h} . k_{j,g(h)}) V, LSE as north_star.
 * K and V are read once: the Hq / Hkv q heads of a KV head go through the prefill kernel together
 * as the rows of one tile, and every sequence's keys are cut into chunks whose partial results
 * are merged by their LSEs, so that a few long sequences still fill the GPU (see decode.cu).
 * A sequence without keys gets O = 0 and LSE = -inf.
 *
 *   q [dev] bf16 [n_seqs, Hq, D]; k, v [dev] bf16 [total_k_tokens, Hkv, D]; cu_seqlens_k [dev]
 *   int64 [n_seqs + 1]; o [dev] bf16 [n_seqs, Hq, D]; lse [dev] fp32 [Hq, n_seqs];
 *   workspace [dev] >= mosaic_agg_decode_attn_workspace_bytes(n_seqs, total_k_tokens, Hq, Hkv, D),
 *   16-byte aligned.
 * Hq / Hkv <= 128; D, alignment, errors and asynchrony as mosaic_agg_prefill_attn.
 * ------------------------------------------------------------------------------------------- */
size_t mosaic_agg_decode_attn_workspace_bytes(int32_t n_seqs, int64_t total_k_tokens, int32_t Hq,
                                              int32_t Hkv, int32_t D);
mosaic_status_t mosaic_agg_decode_attn(const void* q, const void* k, const void* v,
                                       const int64_t* cu_seqlens_k, int32_t n_seqs,
                                       int64_t total_k_tokens, int32_t Hq, int32_t Hkv, int32_t D,
                                       float softmax_scale, void* o, float* lse, void* workspace,
                                       size_t workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_assemble_context -- SURVEY.md section 8(f) N1 (a "next" row, between G5 and A1): the
 * survivors' aggregator contexts as one packed token batch.  The aggregator "process[es] the
 * combined output or reasoning traces of its experts" (Alg. 1
 * `Aggregator(q, {a_i})`); template and order are not given, reading N1-1 fixes
 * them: the context of survivor j (question q = survivor_idx[j]) is
 *     prompt(q) ++ trace(q, 0) ++ trace(q, 1) ++ ... ++ trace(q, E-1).
 *
 *   survivor_idx  [dev] int32 [n_survivors], cu_seqlens [dev] int64 [n_survivors + 1]: as written
 *                 by mosaic_compact (ctx_len[q] = tokens of q's context).
 *   n_survivors, max_seqlen  host values read back from mosaic_compact.
 *   prompt_tokens [dev] int32, the prompts of all Q questions packed; prompt_off [dev] int64 [Q+1].
 *   trace_tokens  [dev] int32, the traces packed in (q, e) order; trace_off [dev] int64 [Q*E + 1].
 *                 Both token buffers are read in whole 16-byte units (bulk copies): the 16-byte-
 *                 aligned closure of each must be readable, which holds for any CUDA allocation.
 *   input_ids     [dev] int32 [total_tokens]  out: the packed contexts (16-byte aligned, as is
 *                 position_ids).
 *   position_ids  [dev] int32 [total_tokens]  out: 0, 1, ... inside every sequence.
 *   n_mismatch    [dev] int32 or NULL         out: sequences whose cu_seqlens length differs from
 *                 prompt + traces; such a sequence is truncated, or padded with -1.
 * Nothing is owned or retained; asynchronous on cuda_stream.  1 <= E <= MOSAIC_MAX_EXPERTS.
 * ------------------------------------------------------------------------------------------- */
mosaic_status_t mosaic_assemble_context(const int32_t* survivor_idx, const int64_t* cu_seqlens,
                                        int32_t n_survivors, int32_t max_seqlen,
                                        const int32_t* prompt_tokens, const int64_t* prompt_off,
                                        const int32_t* trace_tokens, const int64_t* trace_off,
                                        int32_t E, int32_t* input_ids, int32_t* position_ids,
                                        int32_t* n_mismatch, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_rope_packed -- SURVEY.md section 8(f) N1, second half: rotary position embedding applied
 * IN PLACE to packed Q / K by the position_ids of mosaic_assemble_context.  The paper runs
 * Qwen-family aggregators and does not describe the embedding; reading N1-4
 * fixes those models' convention: pairs (i, i + D/2), w_i = theta^(-2i/D), a = position * w_i,
 *     out[i] = x[i] cos a - x[i+D/2] sin a,   out[i+D/2] = x[i+D/2] cos a + x[i] sin a,
 * angles and sin / cos in binary64, products in fp32, result rounded to nearest-even bf16.
 *
 *   q [dev] bf16 [total_tokens, Hq, D], k [dev] bf16 [total_tokens, Hkv, D]  in/out, 16-byte
 *   aligned (either may be NULL when its head count is 0);  position_ids [dev] int32 [total_tokens];
 *   D in {64, 128}; theta > 0 (e.g. 1e6).  Asynchronous on cuda_stream; nothing retained.
 * ------------------------------------------------------------------------------------------- */
mosaic_status_t mosaic_rope_packed(void* q, void* k, const int32_t* position_ids,
                                   int64_t total_tokens, int32_t Hq, int32_t Hkv, int32_t D,
                                   float theta, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * mosaic_stage_host -- the whole stage from HOST buffers (the end-to-end call): copies the gate
 * inputs to the device, runs mosaic_gate_compact, reads S / total_tokens / max_seqlen back,
 * copies the survivors' packed Q/K/V to the device, runs mosaic_agg_prefill_attn and copies every
 * result back.  SYNCHRONOUS: returns after the results are in the host buffers.
 * The survivors' Q/K/V go up, through the attention kernel and back in chunks of ~8 k tokens (cut
 * anywhere, also inside a sequence: a chunk's rows attend the keys uploaded so far) on
 * two internal copy streams (created on first use, one set per process), so the two PCIe
 * directions and the kernel overlap; concurrent calls from several threads serialise.
 *
 *   answers_h, expert_conf_h, ctx_len_h  [host] as mosaic_gate / mosaic_compact.
 *   mode_h, conf_h, bypass_h             [host] [Q] outputs (mode_h, conf_h may be NULL).
 *   survivor_idx_h [host] int32 [Q], cu_seqlens_h [host] int64 [Q+1] capacities as mosaic_compact.
 *   n_survivors_h, total_tokens_h, max_seqlen_h [host] scalars.
 *   max_attn_seqs   attention runs over the first min(S, max_attn_seqs) survivors (< 0: all S).
 *   q_h, k_h, v_h   [host] bf16 packed [T_cap, H, D] holding AT LEAST the tokens of those
 *                   survivors, laid out by the cu_seqlens this call will compute (the caller
 *                   knows ctx_len, hence the layout, once it knows the mask; pass buffers built
 *                   for a previous identical gate, or sized for the worst case).
 *   T_cap           rows available in q_h/k_h/v_h and o_h, lse_h row stride ([Hq, T_cap]).
 *   o_h, lse_h      [host] outputs; lse_h is [Hq, T_attn] contiguous with T_attn = tokens attended.
 *   arena           [dev] scratch of arena_bytes >= mosaic_stage_host_arena_bytes(...).
 *
 * Returns MOSAIC_ERR_WORKSPACE_TOO_SMALL if the survivors' tokens exceed T_cap or the arena.
 * ------------------------------------------------------------------------------------------- */
size_t mosaic_stage_host_arena_bytes(int64_t Q, int32_t E, int64_t T_cap, int32_t Hq, int32_t Hkv,
                                     int32_t D);
mosaic_status_t mosaic_stage_host(const int32_t* answers_h, const float* expert_conf_h,
                                  const int32_t* ctx_len_h, int64_t Q, int32_t E, float tau,
                                  int32_t conf_mode, int32_t* mode_h, float* conf_h,
                                  uint8_t* bypass_h, int32_t* survivor_idx_h,
                                  int64_t* cu_seqlens_h, int32_t* n_survivors_h,
                                  int64_t* total_tokens_h, int32_t* max_seqlen_h,
                                  int32_t max_attn_seqs, const void* q_h, const void* k_h,
                                  const void* v_h, int64_t T_cap, int32_t Hq, int32_t Hkv,
                                  int32_t D, float softmax_scale, void* o_h, float* lse_h,
                                  void* arena, size_t arena_bytes, void* cuda_stream);

/* Diagnostics. */
const char* mosaic_status_string(mosaic_status_t status);
int mosaic_version(void);            /* major*10000 + minor*100 + patch */
int mosaic_last_cuda_error(void);    /* cudaError_t of the last failed CUDA call on this thread */
/* Kernel launches this library has enqueued from this process since load (every kernel counts 1;
 * memsets and copies do not).  bench.py reports the delta over its timed region. */
int64_t mosaic_kernel_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* MOSAIC_H_ */
