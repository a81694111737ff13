/*
 * oracle/mosaic_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, obviously-correct CPU statement of what MOSAIC's confidence-gated
 * aggregator stage computes, written from /root/reference/PAPER.md (cited "P:Lnn") and
 * BASELINE.json's north_star ("BJ").  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no code, header, table or
 * helper with paper_2606_03014_b200/csrc (the CUDA path) and neither includes the other.
 *
 * Integers are exact; floating point is IEEE binary64 except where the paper's quantity is
 * itself a single fp32 operation (the vote fraction compared against an fp32 tau,
 * DESIGN.md reading G-4).  Build without -ffast-math (see oracle/__init__.py).
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`):
 *   oracle_gate     : P:L184-186 worked values (tests/golden/gate_k3_buckets.txt), unanimous /
 *                     all-distinct / permutation / tau-monotone invariants, brute force of all
 *                     10^3 triples and all 4^E tables (E<=6) against a sort+run-length
 *                     restatement, closed-form bypass rates of the seeded generator.
 *   oracle_gate (conf_mode 1, "weighted" extension G2'): NOT defined by the paper
 *                     (P:L188 only licenses a substitute estimator) -- PARITY UNPINNED by the
 *                     paper; pinned only by reductions (equal weights == vote fraction,
 *                     unanimous == 1, all-distinct == w_mode/sum w) and exact rationals.
 *   oracle_gate_ext (abstention sentinel, weighted argmax, tau per question): the
 *                     paper defines none of them (P:L188, L251, L367 only name the openings) --
 *                     PARITY UNPINNED by the paper; pinned to DESIGN.md readings N3-1..N3-3 by
 *                     hand-worked k = 3 cases under both abstention policies, reduction to
 *                     oracle_gate when no sentinel occurs, an always-abstaining extra expert that
 *                     must drop out, equal weights == count plurality, exact rationals
 *                     (tests/test_oracle_gate_ext.py).
 *   oracle_compact  : numpy.flatnonzero / numpy.cumsum special case, S = Q - sum(bypass),
 *                     all-bypass / none-bypass cases.
 *   oracle_attn_*   : L=1 returns V; identical keys give causal prefix mean and
 *                     LSE = scale*q.k + ln(i+1); scale=0; V==1; softmax rows sum to 1;
 *                     causality (future K/V do not matter); split-key LSE merge; GQA == MHA on
 *                     repeated K/V; torch fp64 scaled_dot_product_attention; dense-matrix
 *                     brute force on tiny inputs.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------------------------
 * Step 1a: the confidence gate.  P:L176-186 (Sec. 4.2, the untagged "Equation (11)" and
 * C_vote) and P:L362-380 (Alg. 1).
 *
 *   for each question q with answers a_1..a_k (k = E):
 *     n(x)  = |{ i : a_i = x }|
 *     c*    = max_x n(x)
 *     mode  = majority({a_i}) = the label with n(x) = c*;  ties -> the smallest label value
 *             (paper silent, reading G-2: must not depend on expert order)
 *     agree = C_vote(q) = c* / k, one IEEE fp32 division             (reading G-4)
 *     conf  = agree                                              (conf_mode 0, the paper's C)
 *           = fl32( sum_{i: a_i = mode} w_i / sum_i w_i ), sums in binary64 in expert order,
 *             falling back to agree when sum_i w_i is not > 0  (conf_mode 1, extension G2')
 *     bypass = (conf >= tau), an fp32 comparison                   (">=")
 * ---------------------------------------------------------------------------------------- */
void oracle_gate(const int32_t *answers, const float *expert_conf, int64_t Q, int32_t E,
                 float tau, int32_t conf_mode, int32_t *mode_out, int32_t *count_out,
                 float *agree_out, float *conf_out, uint8_t *bypass_out)
{
    for (int64_t q = 0; q < Q; ++q) {
        const int32_t *a = answers + q * (int64_t)E;
        int32_t c_star = 0, mode = 0;
        for (int32_t i = 0; i < E; ++i) {
            int32_t x = a[i], n = 0;
            for (int32_t j = 0; j < E; ++j)
                n += (a[j] == x);
            if (n > c_star || (n == c_star && x < mode)) {
                c_star = n;
                mode = x;
            }
        }
        float agree = (float)c_star / (float)E;
        float conf = agree;
        if (conf_mode == 1) {
            const float *w = expert_conf + q * (int64_t)E;
            double sm = 0.0, st = 0.0;
            for (int32_t i = 0; i < E; ++i) {
                st += (double)w[i];
                if (a[i] == mode)
                    sm += (double)w[i];
            }
            if (st > 0.0)
                conf = (float)(sm / st);
        }
        if (mode_out) mode_out[q] = mode;
        if (count_out) count_out[q] = c_star;
        if (agree_out) agree_out[q] = agree;
        if (conf_out) conf_out[q] = conf;
        bypass_out[q] = (uint8_t)(conf >= tau);
    }
}

/* ------------------------------------------------------------------------------------------
 * Step 1b: survivor batch.  Alg. 1 line 6: the questions whose gate failed go to
 * Aggregator(q, {a_i}); BJ:north_star: "stream-compacts the surviving queries into a ragged
 * batch with cu_seqlens".  Order: ascending question index (reading G-11).  A survivor's
 * context length is ctx_len[q] (prompt + all expert traces, reading G-12).
 * Returns S; writes survivor_idx[0..S), cu_seqlens[0..S], *total_tokens, *max_seqlen.
 * ---------------------------------------------------------------------------------------- */
int64_t oracle_compact(const uint8_t *bypass, const int32_t *ctx_len, int64_t Q,
                       int32_t *survivor_idx, int64_t *cu_seqlens, int64_t *total_tokens,
                       int32_t *max_seqlen)
{
    int64_t S = 0, tokens = 0;
    int32_t longest = 0;
    cu_seqlens[0] = 0;
    for (int64_t q = 0; q < Q; ++q) {
        if (bypass[q] == 0) {
            survivor_idx[S] = (int32_t)q;
            tokens += (int64_t)ctx_len[q];
            if (ctx_len[q] > longest)
                longest = ctx_len[q];
            ++S;
            cu_seqlens[S] = tokens;
        }
    }
    *total_tokens = tokens;
    *max_seqlen = longest;
    return S;
}

/* ------------------------------------------------------------------------------------------
 * Step 2: the aggregator's prefill attention over each survivor's concatenated context
 * ("process the combined output or reasoning traces of its experts"; the math is fixed
 * by BJ:north_star: variable-length causal grouped-query prefill attention, bf16 O and fp32
 * row logsumexp).  The plain definition, one output row at a time:
 *
 *   sequence s owns tokens t0 = cu_seqlens[s] .. t0+L-1;  q head h reads kv head g = h/(Hq/Hkv)
 *   x_j = scale * sum_d Q[t0+i,h,d] K[t0+j,g,d]      j = 0..i   (causal, sequence-local)
 *   M   = max_j x_j ;  Z = sum_j exp(x_j - M)
 *   LSE = M + ln Z
 *   O_d = sum_j (exp(x_j - M)/Z) V[t0+j,g,d]
 *
 * Inputs are bf16 bit patterns widened exactly to binary64; nothing is rounded afterwards.
 * Layout: q[T,Hq,D], k[T,Hkv,D], v[T,Hkv,D], D fastest (reading A-4).
 * ---------------------------------------------------------------------------------------- */
static inline double bf16_to_double(uint16_t b)
{
    uint32_t u = (uint32_t)b << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

/* One row (s, h, i).  x is caller scratch of at least i+1 doubles.  Returns sum_j p_j. */
static double attn_row(const uint16_t *q, const uint16_t *k, const uint16_t *v, int64_t t0,
                       int32_t h, int64_t i, int32_t Hq, int32_t Hkv, int32_t D, double scale,
                       double *x, double *o_out, double *lse_out)
{
    const int32_t g = h / (Hq / Hkv);
    const uint16_t *qrow = q + ((t0 + i) * Hq + h) * (int64_t)D;
    double M = -INFINITY;
    for (int64_t j = 0; j <= i; ++j) {
        const uint16_t *krow = k + ((t0 + j) * Hkv + g) * (int64_t)D;
        double dot = 0.0;
        for (int32_t d = 0; d < D; ++d)
            dot += bf16_to_double(qrow[d]) * bf16_to_double(krow[d]);
        x[j] = scale * dot;
        if (x[j] > M)
            M = x[j];
    }
    double Z = 0.0;
    for (int64_t j = 0; j <= i; ++j)
        Z += exp(x[j] - M);
    for (int32_t d = 0; d < D; ++d)
        o_out[d] = 0.0;
    double psum = 0.0;
    for (int64_t j = 0; j <= i; ++j) {
        const uint16_t *vrow = v + ((t0 + j) * Hkv + g) * (int64_t)D;
        double p = exp(x[j] - M) / Z;
        psum += p;
        for (int32_t d = 0; d < D; ++d)
            o_out[d] += p * bf16_to_double(vrow[d]);
    }
    *lse_out = M + log(Z);
    return psum;
}

/* Selected rows: row r is (row_seq[r], row_head[r], row_pos[r]); o_out[n_rows,D], lse_out[n_rows],
 * psum_out[n_rows] (may be NULL) = sum of the row's softmax weights (pin: == 1).
 * Rows are independent; OpenMP only hands different rows to different threads. */
int oracle_attn_rows(const uint16_t *q, const uint16_t *k, const uint16_t *v,
                     const int64_t *cu_seqlens, int64_t n_rows, const int32_t *row_seq,
                     const int32_t *row_head, const int64_t *row_pos, int32_t Hq, int32_t Hkv,
                     int32_t D, float softmax_scale, double *o_out, double *lse_out,
                     double *psum_out)
{
    int failed = 0;
#pragma omp parallel
    {
        double *x = NULL;
        int64_t cap = 0;
#pragma omp for schedule(dynamic, 1)
        for (int64_t r = 0; r < n_rows; ++r) {
            int64_t i = row_pos[r];
            if (i + 1 > cap) {
                free(x);
                cap = i + 1;
                x = (double *)malloc((size_t)cap * sizeof(double));
            }
            if (!x) {
                failed = 1;
                continue;
            }
            double ps = attn_row(q, k, v, cu_seqlens[row_seq[r]], row_head[r], i, Hq, Hkv, D,
                                 (double)softmax_scale, x, o_out + r * (int64_t)D, lse_out + r);
            if (psum_out)
                psum_out[r] = ps;
        }
        free(x);
    }
    return failed;
}

/* Every row of every sequence: o_out[T,Hq,D] binary64, lse_out[Hq,T] binary64 (reading A-3). */
int oracle_attn_full(const uint16_t *q, const uint16_t *k, const uint16_t *v,
                     const int64_t *cu_seqlens, int32_t n_seqs, int32_t Hq, int32_t Hkv,
                     int32_t D, float softmax_scale, double *o_out, double *lse_out)
{
    const int64_t T = cu_seqlens[n_seqs];
    int failed = 0;
    for (int32_t s = 0; s < n_seqs; ++s) {
        const int64_t t0 = cu_seqlens[s], L = cu_seqlens[s + 1] - t0;
#pragma omp parallel
        {
            double *x = (double *)malloc((size_t)(L > 0 ? L : 1) * sizeof(double));
            if (!x)
                failed = 1;
#pragma omp for collapse(2) schedule(dynamic, 4)
            for (int64_t i = 0; i < L; ++i)
                for (int32_t h = 0; h < Hq; ++h)
                    if (x)
                        attn_row(q, k, v, t0, h, i, Hq, Hkv, D, (double)softmax_scale, x,
                                 o_out + ((t0 + i) * Hq + h) * (int64_t)D,
                                 lse_out + (int64_t)h * T + t0 + i);
            free(x);
        }
    }
    return failed;
}

int oracle_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp master
        n = omp_get_num_threads();
    }
#endif
    return n;
}

/* ------------------------------------------------------------------------------------------
 * the gate with the other confidence estimators P:L188 invites ("agnostic to
 * the choice of confidence estimator"), a threshold per question (P:L251 names the static
 * threshold as a limitation) and a failed Extract (Alg. 1 line 1).  Readings
 * (DESIGN.md section 2): N3-1 tau per question; N3-2 abstention; N3-3 weighted argmax.
 *
 *   for each question q with answers a_1..a_E and (conf_mode 1, 2) weights w_1..w_E:
 *     expert i ABSTAINS iff abstain_policy != 0 and a_i == abstain_label; an abstaining expert
 *       is counted for no label and adds its weight to no label
 *     n(x) = |{ i answering : a_i = x }|,  s(x) = sum_{i answering, a_i = x} w_i  (binary64,
 *       increasing i)
 *     k  = E                          (policy 0, 1: P:L182 divides by the k experts recruited)
 *        = |{ i answering }|          (policy 2)
 *     St = sum of w_i over all i (policy 0, 1) or over the answering i (policy 2), increasing i
 *     mode:  conf_mode 0, 1, or St <= 0: the x with the largest n(x), ties -> smallest x
 *            conf_mode 2 and St > 0    : the x with the largest s(x), ties -> smallest x
 *            nobody answers            : abstain_label, with count 0
 *     count = n(mode);  agree = fl32(count) / fl32(k)  (0 when k == 0)
 *     conf  = agree                        (conf_mode 0, or St <= 0)
 *           = fl32( s(mode) / St )         (conf_mode 1, 2)
 *     bypass = conf >= (tau_q ? tau_q[q] : tau), fp32 comparison, false for a NaN threshold
 *
 * With policy 0, conf_mode 0 / 1 and tau_q == NULL this is oracle_gate.
 * ---------------------------------------------------------------------------------------- */
void oracle_gate_ext(const int32_t *answers, const float *expert_conf, int64_t Q, int32_t E,
                     float tau, const float *tau_q, int32_t conf_mode, int32_t abstain_policy,
                     int32_t abstain_label, int32_t *mode_out, int32_t *count_out,
                     float *agree_out, float *conf_out, uint8_t *bypass_out)
{
    for (int64_t q = 0; q < Q; ++q) {
        const int32_t *a = answers + q * (int64_t)E;
        const float *w = conf_mode ? expert_conf + q * (int64_t)E : NULL;
        int32_t answering = 0;
        double st = 0.0;
        for (int32_t i = 0; i < E; ++i) {
            const int abst = abstain_policy != 0 && a[i] == abstain_label;
            if (!abst)
                ++answering;
            if (w && !(abst && abstain_policy == 2))
                st += (double)w[i];
        }
        const int32_t k = abstain_policy == 2 ? answering : E;
        const int by_weight = conf_mode == 2 && st > 0.0;
        int32_t mode = abstain_label, count = 0;
        double s_mode = 0.0;
        int found = 0;
        for (int32_t i = 0; i < E; ++i) {
            if (abstain_policy != 0 && a[i] == abstain_label)
                continue;
            const int32_t x = a[i];
            int32_t n = 0;
            double s = 0.0;
            for (int32_t j = 0; j < E; ++j) {
                if (a[j] == x) { /* x is not the sentinel, so expert j answers */
                    ++n;
                    if (w)
                        s += (double)w[j];
                }
            }
            int better;
            if (!found)
                better = 1;
            else if (by_weight)
                better = s > s_mode || (s == s_mode && x < mode);
            else
                better = n > count || (n == count && x < mode);
            if (better) {
                found = 1;
                mode = x;
                count = n;
                s_mode = s;
            }
        }
        const float agree = k > 0 ? (float)count / (float)k : 0.0f;
        float conf = agree;
        if (conf_mode != 0 && st > 0.0)
            conf = (float)(s_mode / st);
        const float t = tau_q ? tau_q[q] : tau;
        if (mode_out) mode_out[q] = mode;
        if (count_out) count_out[q] = count;
        if (agree_out) agree_out[q] = agree;
        if (conf_out) conf_out[q] = conf;
        bypass_out[q] = (uint8_t)(conf >= t);
    }
}
