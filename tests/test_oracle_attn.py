"""Pins for the attention oracle (oracle/mosaic_oracle.c: oracle_attn_rows / _full) -- CPU only.

The paper gives no attention math (PAPER.md P:L21 only says the aggregator prefill over the
combined traces is long and expensive); BASELINE.json's north_star fixes the definition and the
invariants used here: single-token sequences return V, identical keys give the causal prefix
mean of V, softmax rows sum to 1, brute force on tiny inputs.  Further pins: torch's fp64
scaled_dot_product_attention (a library routine, independent code), LSE-merge of split keys,
causality, GQA == MHA on repeated K/V.
"""
import numpy as np
import pytest
import torch

import oracle


def bf16_bits(x):
    """float array -> nearest-even bf16 bit patterns (uint16)."""
    t = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).to(torch.bfloat16)
    return t.view(torch.int16).numpy().view(np.uint16).copy()


def bits_f64(b):
    return (b.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def ragged(seed, lens, Hq, Hkv, D, kscale=1.0):
    g = np.random.default_rng(seed)
    T = int(sum(lens))
    q = bf16_bits(g.standard_normal((T, Hq, D)))
    k = bf16_bits(g.standard_normal((T, Hkv, D)) * kscale)
    v = bf16_bits(g.standard_normal((T, Hkv, D)))
    cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    return q, k, v, cu


def all_rows(cu, Hq):
    rs, rh, rp = [], [], []
    for s in range(len(cu) - 1):
        for h in range(Hq):
            for i in range(int(cu[s + 1] - cu[s])):
                rs.append(s), rh.append(h), rp.append(i)
    return np.array(rs, np.int32), np.array(rh, np.int32), np.array(rp, np.int64)


def test_single_token_sequences_return_v():
    q, k, v, cu = ragged(0, [1, 1, 1, 1, 1], 6, 3, 64)
    scale = 0.125
    O, lse = oracle.attn_full(q, k, v, cu, scale)
    vf, qf, kf = bits_f64(v), bits_f64(q), bits_f64(k)
    for t in range(5):
        for h in range(6):
            assert np.array_equal(O[t, h], vf[t, h // 2])                 # exactly V
            want = scale * float(np.dot(qf[t, h], kf[t, h // 2]))
            assert abs(lse[h, t] - want) <= 1e-12 * max(1.0, abs(want))


def test_identical_keys_give_prefix_mean_and_log_count():
    lens = [37, 200, 5]
    q, k, v, cu = ragged(1, lens, 4, 2, 64)
    for s in range(3):                                    # one key per (sequence, kv head)
        k[cu[s]:cu[s + 1]] = k[cu[s]]
    scale = 1 / 8
    O, lse = oracle.attn_full(q, k, v, cu, scale)
    vf, qf, kf = bits_f64(v), bits_f64(q), bits_f64(k)
    for s in range(3):
        t0, L = int(cu[s]), lens[s]
        for h in range(4):
            g = h // 2
            pm = np.cumsum(vf[t0:t0 + L, g], axis=0) / np.arange(1, L + 1)[:, None]
            assert np.max(np.abs(O[t0:t0 + L, h] - pm)) < 1e-13
            want = scale * (qf[t0:t0 + L, h] @ kf[t0, g]) + np.log(np.arange(1, L + 1))
            assert np.max(np.abs(lse[h, t0:t0 + L] - want)) < 1e-12


def test_zero_scale_is_uniform_and_v_ones_gives_ones():
    lens = [64, 3, 129]
    q, k, v, cu = ragged(2, lens, 4, 4, 64, kscale=3.0)
    O, lse = oracle.attn_full(q, k, v, cu, 0.0)
    vf = bits_f64(v)
    for s, L in enumerate(lens):
        t0 = int(cu[s])
        for h in range(4):
            pm = np.cumsum(vf[t0:t0 + L, h], axis=0) / np.arange(1, L + 1)[:, None]
            assert np.max(np.abs(O[t0:t0 + L, h] - pm)) < 1e-13
            assert np.max(np.abs(lse[h, t0:t0 + L] - np.log(np.arange(1, L + 1)))) < 1e-13
    v1 = bf16_bits(np.ones(v.shape))
    O1, _ = oracle.attn_full(q, k, v1, cu, 0.37)
    assert np.max(np.abs(O1 - 1.0)) < 1e-13


def test_softmax_rows_sum_to_one():
    q, k, v, cu = ragged(3, [300, 17], 4, 2, 128, kscale=2.0)
    rs, rh, rp = all_rows(cu, 4)
    _, _, ps = oracle.attn_rows(q, k, v, cu, rs, rh, rp, 128 ** -0.5)
    assert np.max(np.abs(ps - 1.0)) < 1e-12


def test_future_tokens_and_other_sequences_do_not_matter():
    lens = [50, 70]
    q, k, v, cu = ragged(4, lens, 4, 2, 64)
    rs = np.array([0, 0, 1, 1], np.int32)
    rh = np.array([0, 3, 1, 2], np.int32)
    rp = np.array([10, 49, 0, 33], np.int64)
    O1, l1, _ = oracle.attn_rows(q, k, v, cu, rs, rh, rp, 0.125)
    g = np.random.default_rng(99)
    k2, v2, q2 = k.copy(), v.copy(), q.copy()
    # seq 0: everything after position 10 changes -> row (0,*,10) must not move
    k2[11:50] = bf16_bits(g.standard_normal((39, 2, 64)))
    v2[11:50] = bf16_bits(g.standard_normal((39, 2, 64)))
    O2, l2, _ = oracle.attn_rows(q, k2, v2, cu, rs[:1], rh[:1], rp[:1], 0.125)
    assert np.array_equal(O1[:1], O2) and np.array_equal(l1[:1], l2)
    # seq 1 rows ignore all of seq 0 and seq 1's positions > 33
    k3, v3 = k.copy(), v.copy()
    k3[:50] = bf16_bits(g.standard_normal((50, 2, 64)))
    v3[:50] = bf16_bits(g.standard_normal((50, 2, 64)))
    k3[50 + 34:] = 0
    v3[50 + 34:] = 0
    O3, l3, _ = oracle.attn_rows(q, k3, v3, cu, rs[2:], rh[2:], rp[2:], 0.125)
    assert np.array_equal(O1[2:], O3) and np.array_equal(l1[2:], l3)
    # and a past token does matter (the mask is not upside down)
    k4 = k.copy()
    k4[0] = bf16_bits(g.standard_normal((2, 64)))
    O4, _, _ = oracle.attn_rows(q, k4, v, cu, rs[:1], rh[:1], rp[:1], 0.125)
    assert not np.array_equal(O1[:1], O4)


def test_split_keys_merge_by_lse():
    """Attend keys [0,m) and [m,i] separately, merge with the row logsumexps: this is what LSE is
    exported for, and it pins LSE as the natural log of the sum of exp of the SCALED scores."""
    L, m, i, Hq, Hkv, D, scale = 90, 41, 77, 4, 2, 64, 0.2
    q, k, v, cu = ragged(5, [L], Hq, Hkv, D)
    h = 3
    O, lse, _ = oracle.attn_rows(q, k, v, cu, [0], [h], [i], scale)
    # left part: a sequence 0..m-1 whose last query is q_i
    qa = q[:m].copy()
    qa[m - 1] = q[i]
    Oa, la, _ = oracle.attn_rows(qa, k[:m], v[:m], np.array([0, m]), [0], [h], [m - 1], scale)
    # right part: tokens m..i re-packed as their own sequence, last query q_i
    n = i - m + 1
    Ob, lb, _ = oracle.attn_rows(q[m:i + 1], k[m:i + 1], v[m:i + 1], np.array([0, n]), [0], [h], [n - 1], scale)
    lm = np.logaddexp(la[0], lb[0])
    Om = np.exp(la[0] - lm) * Oa[0] + np.exp(lb[0] - lm) * Ob[0]
    assert abs(lm - lse[0]) < 1e-12
    assert np.max(np.abs(Om - O[0])) < 1e-13


@pytest.mark.parametrize("Hq,Hkv,D,lens", [(4, 2, 64, [64, 1, 130, 256]), (28, 4, 128, [33, 140]),
                                           (8, 8, 128, [100]), (8, 1, 64, [70, 9])])
def test_against_torch_fp64_sdpa(Hq, Hkv, D, lens):
    """Library special case: per sequence, torch's scaled_dot_product_attention(is_causal=True)
    in fp64 on K/V repeated per group (GQA == MHA with repeat_interleave)."""
    scale = float(np.float32(D ** -0.5))
    q, k, v, cu = ragged(6, lens, Hq, Hkv, D, kscale=1.5)
    O, lse = oracle.attn_full(q, k, v, cu, scale)
    G = Hq // Hkv
    for s, L in enumerate(lens):
        t0 = int(cu[s])
        qt = torch.from_numpy(bits_f64(q[t0:t0 + L])).permute(1, 0, 2)[None]
        kt = torch.from_numpy(bits_f64(k[t0:t0 + L])).permute(1, 0, 2).repeat_interleave(G, 0)[None]
        vt = torch.from_numpy(bits_f64(v[t0:t0 + L])).permute(1, 0, 2).repeat_interleave(G, 0)[None]
        ref = torch.nn.functional.scaled_dot_product_attention(qt, kt, vt, is_causal=True, scale=scale)
        ref = ref[0].permute(1, 0, 2).numpy()
        assert np.max(np.abs(O[t0:t0 + L] - ref)) < 1e-12
        sc = (qt[0] @ kt[0].transpose(1, 2)) * scale
        sc = sc.masked_fill(~torch.ones(L, L, dtype=torch.bool).tril(), float("-inf"))
        assert np.max(np.abs(lse[:, t0:t0 + L] - torch.logsumexp(sc, -1).numpy())) < 1e-12


def test_dense_matrix_brute_force_tiny():
    """L <= 8: build the whole L x L score matrix, mask, exponentiate, normalise."""
    Hq, Hkv, D, scale = 4, 2, 64, 0.11
    for L in range(1, 9):
        q, k, v, cu = ragged(10 + L, [L], Hq, Hkv, D)
        O, lse = oracle.attn_full(q, k, v, cu, scale)
        qf, kf, vf = bits_f64(q), bits_f64(k), bits_f64(v)
        for h in range(Hq):
            g = h // (Hq // Hkv)
            S = np.float64(np.float32(scale)) * np.einsum("id,jd->ij", qf[:, h], kf[:, g])
            W = np.where(np.tril(np.ones((L, L), bool)), np.exp(S), 0.0)
            P = W / W.sum(axis=1, keepdims=True)
            assert np.max(np.abs(P @ vf[:, g] - O[:, h])) < 1e-13
            assert np.max(np.abs(np.log(W.sum(axis=1)) - lse[h])) < 1e-13


def test_rows_and_full_agree_and_layouts():
    q, k, v, cu = ragged(20, [19, 0, 45], 6, 2, 64)          # a zero-length sequence in the middle
    O, lse = oracle.attn_full(q, k, v, cu, 0.125)
    assert O.shape == (64, 6, 64) and lse.shape == (6, 64)
    rs, rh, rp = all_rows(cu, 6)
    Or, lr, _ = oracle.attn_rows(q, k, v, cu, rs, rh, rp, 0.125)
    for n in range(0, len(rs), 7):
        t = int(cu[rs[n]] + rp[n])
        assert np.array_equal(Or[n], O[t, rh[n]]) and lr[n] == lse[rh[n], t]


def test_sharp_softmax_picks_the_argmax_value():
    """K x 256: the weights collapse onto the best key, O -> V[argmax]."""
    L, D = 120, 64
    q, k, v, cu = ragged(30, [L], 2, 2, D, kscale=256.0)
    O, _ = oracle.attn_full(q, k, v, cu, D ** -0.5)
    qf, kf, vf = bits_f64(q), bits_f64(k), bits_f64(v)
    hits = 0
    for i in range(L):
        s = qf[i, 0] @ kf[:i + 1, 0].T
        top2 = np.sort(s)[-2:] if i else np.array([-np.inf, s[0]])
        if (top2[1] - top2[0]) * D ** -0.5 > 40:
            hits += 1
            assert np.max(np.abs(O[i, 0] - vf[int(np.argmax(s)), 0])) < 1e-12
    assert hits > 20
