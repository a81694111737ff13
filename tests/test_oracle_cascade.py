"""Pins of oracle.lse_merge_n and oracle.attn_shared_prefix against functions
that are themselves pinned (the C prefill oracle, attn_kv_full, the 2-way lse_merge)."""
import numpy as np
import torch

import oracle


def _bits(shape, seed, scale=1.0):
    g = torch.Generator().manual_seed(seed)
    t = (torch.randn(shape, generator=g) * scale).to(torch.bfloat16)
    return t.contiguous().view(torch.int16).numpy().view(np.uint16)


def _cu(lengths):
    return np.concatenate([[0], np.cumsum(np.asarray(lengths, np.int64))]).astype(np.int64)


def test_merge_n_of_a_three_way_key_split_is_the_unsplit_prefill():
    """Keys [0, a), [a, b) seen in full by the rows >= b (two non-causal blocks) and the causal
    prefill over [b, L): merged n-way they must give rows b.. of the plain prefill."""
    L, a, b, Hq, Hkv, D = 300, 70, 190, 4, 2, 64
    q, k, v = _bits((L, Hq, D), 1), _bits((L, Hkv, D), 2), _bits((L, Hkv, D), 3)
    O_ref, lse_ref = oracle.attn_full(q, k, v, _cu([L]), 0.125)
    n = L - b
    cq = _cu([n])
    parts = [oracle.attn_kv_full(q[b:], k[:a], v[:a], cq, _cu([a]), 0.125, causal=False),
             oracle.attn_kv_full(q[b:], k[a:b], v[a:b], cq, _cu([b - a]), 0.125, causal=False),
             oracle.attn_full(q[b:], k[b:], v[b:], cq, 0.125)]
    o, lse = oracle.lse_merge_n(np.stack([p[0] for p in parts]), np.stack([p[1] for p in parts]))
    assert np.abs(o - O_ref[b:]).max() < 1e-12 and np.abs(lse - lse_ref[:, b:]).max() < 1e-12


def test_merge_n_reduces_to_the_two_way_merge_and_handles_empty_partials():
    g = np.random.default_rng(4)
    T, Hq, D = 50, 3, 16
    op = g.standard_normal((2, T, Hq, D))
    lp = g.standard_normal((2, Hq, T)) * 3
    lp[0, 0, :5] = -np.inf
    lp[:, 1, 7] = -np.inf
    o2, l2 = oracle.lse_merge(op[0], lp[0], op[1], lp[1])
    o, lse = oracle.lse_merge_n(op, lp)
    fin = np.isfinite(l2)
    assert np.array_equal(np.isneginf(lse), np.isneginf(l2))
    assert np.abs(lse[fin] - l2[fin]).max() < 1e-12
    assert np.abs(o - np.nan_to_num(o2)).max() < 1e-12
    assert np.all(o[7, 1] == 0) and lse[1, 7] == -np.inf
    # one part: the identity; associativity: merging ((0,1),2) = merging (0,1,2)
    o1, l1 = oracle.lse_merge_n(op[:1], lp[:1])
    keep = np.isfinite(lp[0])
    assert np.abs(l1[keep] - lp[0][keep]).max() < 1e-12
    op3 = g.standard_normal((3, T, Hq, D))
    lp3 = g.standard_normal((3, Hq, T))
    oa, la = oracle.lse_merge(*oracle.lse_merge(op3[0], lp3[0], op3[1], lp3[1]), op3[2], lp3[2])
    ob, lb = oracle.lse_merge_n(op3, lp3)
    assert np.abs(oa - ob).max() < 1e-12 and np.abs(la - lb).max() < 1e-12


def test_shared_prefix_is_the_tail_of_a_plain_prefill_over_prefix_plus_own_tokens():
    """Give the prefix positions arbitrary q rows and run the C prefill oracle on the explicitly
    concatenated sequence: its last L_s rows are the shared-prefix result (and do not depend on the
    q rows invented for the prefix)."""
    P, lens, Hq, Hkv, D = 37, [5, 0, 64, 130], 4, 2, 64
    cu = _cu(lens)
    T = int(cu[-1])
    q, k, v = _bits((T, Hq, D), 11), _bits((T, Hkv, D), 12), _bits((T, Hkv, D), 13)
    kp, vp = _bits((P, Hkv, D), 14), _bits((P, Hkv, D), 15)
    O, lse = oracle.attn_shared_prefix(q, kp, vp, k, v, cu, 0.2)
    for s, L in enumerate(lens):
        if L == 0:
            continue
        a, b = int(cu[s]), int(cu[s + 1])
        qq = np.concatenate([_bits((P, Hq, D), 100 + s), q[a:b]])
        O_ref, l_ref = oracle.attn_full(qq, np.concatenate([kp, k[a:b]]), np.concatenate([vp, v[a:b]]),
                                        _cu([P + L]), 0.2)
        assert np.abs(O[a:b] - O_ref[P:]).max() < 1e-12
        assert np.abs(lse[:, a:b] - l_ref[:, P:]).max() < 1e-12
    # no shared block: the plain prefill
    z = np.zeros((0, Hkv, D), np.uint16)
    O0, l0 = oracle.attn_shared_prefix(q, z, z, k, v, cu, 0.2)
    O1, l1 = oracle.attn_full(q, k, v, cu, 0.2)
    assert np.abs(O0 - O1).max() < 1e-12 and np.abs(l0 - l1).max() < 1e-12
