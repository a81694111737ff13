"""Pins of oracle.attn_kv_full (reading N2-1) against the already
pinned C oracle of the plain prefill and against closed forms -- not against its own formula:

* Lk = Lq must reproduce oracle.attn_full (a different implementation: C loops);
* the last Lq rows of a plain causal prefill over Lk tokens are exactly the bottom-right-aligned
  problem with the same K / V (a wrong sign or an off-by-one in the offset fails this);
* Lq = 1 with identical keys: O = mean of all Lk value rows, LSE = scale q.k + ln Lk."""
import numpy as np
import torch

import oracle


def _bits(shape, seed, scale=1.0):
    g = torch.Generator().manual_seed(seed)
    t = (torch.randn(shape, generator=g) * scale).to(torch.bfloat16)
    return t.view(torch.int16).numpy().view(np.uint16)


def _cu(lengths):
    return np.concatenate([[0], np.cumsum(np.asarray(lengths, np.int64))]).astype(np.int64)


def test_equal_lengths_reproduce_the_plain_prefill_oracle():
    cu = _cu([5, 0, 130, 77])
    T, Hq, Hkv, D = int(cu[-1]), 4, 2, 64
    q, k, v = _bits((T, Hq, D), 1), _bits((T, Hkv, D), 2), _bits((T, Hkv, D), 3)
    O0, l0 = oracle.attn_full(q, k, v, cu, 0.125)
    O1, l1 = oracle.attn_kv_full(q, k, v, cu, cu, 0.125)
    assert np.abs(O0 - O1).max() < 1e-12 and np.abs(l0 - l1).max() < 1e-12


def test_last_rows_of_a_plain_prefill():
    Lk_all, Lq_all = [200, 131, 64], [37, 131, 1]
    cu_k, cu_q = _cu(Lk_all), _cu(Lq_all)
    Hq, Hkv, D = 6, 2, 64
    qf = _bits((int(cu_k[-1]), Hq, D), 4)           # q for EVERY position; the tails are the q rows
    k, v = _bits((int(cu_k[-1]), Hkv, D), 5), _bits((int(cu_k[-1]), Hkv, D), 6)
    Of, lf = oracle.attn_full(qf, k, v, cu_k, 0.11)
    take = np.concatenate([np.arange(cu_k[s + 1] - Lq_all[s], cu_k[s + 1]) for s in range(3)])
    O, l = oracle.attn_kv_full(qf[take], k, v, cu_q, cu_k, 0.11)
    assert np.abs(O - Of[take]).max() < 1e-12 and np.abs(l - lf[:, take]).max() < 1e-12


def test_single_query_identical_keys_closed_form():
    Lk, Hq, Hkv, D = 300, 2, 1, 64
    krow = _bits((1, Hkv, D), 7)
    k = np.repeat(krow, Lk, axis=0)
    v, q = _bits((Lk, Hkv, D), 8), _bits((1, Hq, D), 9)
    O, l = oracle.attn_kv_full(q, k, v, _cu([1]), _cu([Lk]), 0.2)
    f = lambda b: (b.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    assert np.abs(O[0, 0] - f(v)[:, 0].mean(axis=0)).max() < 1e-12
    dots = np.float64(np.float32(0.2)) * (f(q)[0] * f(krow)[0, 0][None, :]).sum(-1)
    assert np.abs(l[:, 0] - (dots + np.log(Lk))).max() < 1e-12


def test_non_causal_rows_see_every_key():
    """causal = False pinned two ways: the LAST row of the causal problem sees every key, so it
    must equal the same row of the non-causal one; with identical keys every row is mean(V)."""
    Lq, Lk, Hq, Hkv, D = 5, 40, 2, 2, 64
    q, k, v = _bits((Lq, Hq, D), 11), _bits((Lk, Hkv, D), 12), _bits((Lk, Hkv, D), 13)
    Oc, lc = oracle.attn_kv_full(q, k, v, _cu([Lq]), _cu([Lk]), 0.3, causal=True)
    On, ln = oracle.attn_kv_full(q, k, v, _cu([Lq]), _cu([Lk]), 0.3, causal=False)
    assert np.abs(Oc[-1] - On[-1]).max() < 1e-12 and np.abs(lc[:, -1] - ln[:, -1]).max() < 1e-12
    assert np.abs(Oc[0] - On[0]).max() > 1e-3          # the first row does differ
    kk = np.repeat(_bits((1, Hkv, D), 14), Lk, axis=0)
    On, _ = oracle.attn_kv_full(q, kk, v, _cu([Lq]), _cu([Lk]), 0.3, causal=False)
    f = lambda b: (b.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    assert np.abs(On[:, 0] - f(v)[:, 0].mean(axis=0)[None, :]).max() < 1e-12


def test_merge_of_a_key_split_is_the_unsplit_attention():
    """oracle.lse_merge pinned to the attention oracle: keys [0, a) seen by all rows >= a, merged with
    the causal prefill over keys [a, L), must reproduce rows a.. of the plain prefill over [0, L);
    an empty partial (LSE = -inf) must leave the other unchanged."""
    L, a, Hq, Hkv, D = 150, 70, 4, 2, 64
    q, k, v = _bits((L, Hq, D), 21), _bits((L, Hkv, D), 22), _bits((L, Hkv, D), 23)
    Of, lf = oracle.attn_full(q, k, v, _cu([L]), 0.2)
    O1, l1 = oracle.attn_kv_full(q[a:], k[:a], v[:a], _cu([L - a]), _cu([a]), 0.2, causal=False)
    O2, l2 = oracle.attn_full(q[a:], k[a:], v[a:], _cu([L - a]), 0.2)
    O, l = oracle.lse_merge(O1, l1, O2, l2)
    assert np.abs(O - Of[a:]).max() < 1e-12 and np.abs(l - lf[:, a:]).max() < 1e-12
    O, l = oracle.lse_merge(np.full_like(O2, np.nan), np.full_like(l2, -np.inf), O2, l2)
    assert np.array_equal(O, O2) and np.array_equal(l, l2)
