"""Pins of oracle.assemble_context against things other than itself:

* tokens that ENCODE where they came from (question, segment, index): the expected value at every
  output position then follows from the definition in DESIGN.md reading N1-1 by decoding, with no
  concatenation code shared with the oracle;
* a brute-force restatement with Python lists on tiny inputs;
* closed forms: position_ids = arange(T) - repeat(cu[:-1], L); token conservation (the output is a
  permutation of the survivors' source tokens, in order inside every segment)."""
import numpy as np
import pytest

import oracle
from paper_2606_03014_b200 import workloads as wl


def _encoded_inputs(Q, E, g, max_prompt=9, max_trace=13):
    """Token = q * 2^20 + segment * 2^14 + index (segment 0 = prompt, 1 + e = trace e)."""
    p_len = g.integers(0, max_prompt + 1, size=Q)
    t_len = g.integers(0, max_trace + 1, size=(Q, E))
    t_len[g.random((Q, E)) < 0.2] = 0  # empty traces are legal
    po = np.concatenate([[0], np.cumsum(p_len)]).astype(np.int64)
    to = np.concatenate([[0], np.cumsum(t_len.reshape(-1))]).astype(np.int64)
    pt = np.concatenate([q * 2**20 + np.arange(p_len[q]) for q in range(Q)] + [np.empty(0, int)])
    tt = np.concatenate([q * 2**20 + (1 + e) * 2**14 + np.arange(t_len[q, e])
                         for q in range(Q) for e in range(E)] + [np.empty(0, int)])
    ctx = (p_len + t_len.sum(axis=1)).astype(np.int32)
    return pt.astype(np.int32), po, tt.astype(np.int32), to, ctx, p_len, t_len


@pytest.mark.parametrize("Q,E,seed", [(1, 1, 0), (7, 3, 1), (40, 8, 2), (64, 5, 3)])
def test_decoded_tokens_follow_the_definition(Q, E, seed):
    g = np.random.default_rng(seed)
    pt, po, tt, to, ctx, p_len, t_len = _encoded_inputs(Q, E, g)
    bypass = (g.random(Q) < 0.4).astype(np.uint8)
    oc = oracle.compact(bypass, ctx)
    out = oracle.assemble_context(oc["survivor_idx"], oc["cu_seqlens"], pt, po, tt, to, E)
    ids, pos, cu = out["input_ids"], out["position_ids"], oc["cu_seqlens"]
    assert out["n_mismatch"] == 0 and ids.shape == (oc["total_tokens"],)
    for j, q in enumerate(oc["survivor_idx"]):
        a, b = int(cu[j]), int(cu[j + 1])
        tok = ids[a:b].astype(np.int64)
        assert np.all(tok >> 20 == q)                       # only question q's tokens
        seg, k = (tok >> 14) & 63, tok & (2**14 - 1)
        assert np.all(np.diff(seg) >= 0)                    # prompt first, then traces 0..E-1
        lens = np.concatenate([[p_len[q]], t_len[q]])
        assert np.array_equal(np.bincount(seg, minlength=E + 1), lens)   # every token, once
        starts = np.concatenate([[0], np.cumsum(lens)])[seg]
        assert np.array_equal(k, np.arange(b - a) - starts)  # in order inside every segment
        assert np.array_equal(pos[a:b], np.arange(b - a))


def test_brute_force_lists_tiny():
    g = np.random.default_rng(7)
    Q, E = 6, 2
    pt, po, tt, to, ctx, _, _ = _encoded_inputs(Q, E, g, 4, 5)
    idx = np.array([0, 2, 3, 5], np.int32)
    cu = np.concatenate([[0], np.cumsum(ctx[idx])]).astype(np.int64)
    want_ids, want_pos = [], []
    for q in idx:
        seq = list(pt[po[q]:po[q + 1]])
        for e in range(E):
            seq += list(tt[to[q * E + e]:to[q * E + e + 1]])
        want_ids += seq
        want_pos += list(range(len(seq)))
    out = oracle.assemble_context(idx, cu, pt, po, tt, to, E)
    assert out["input_ids"].tolist() == want_ids and out["position_ids"].tolist() == want_pos


def test_closed_forms_on_the_workload_generator():
    cfg = wl.C1
    for seed in range(3):
        gi = wl.gate_inputs(cfg, seed)
        oc = oracle.compact(oracle.gate(gi.answers, gi.tau)["bypass"], gi.ctx_len)
        pt, po, tt, to = wl.context_parts(cfg, seed)
        # the generator's parts add up to the ctx_len every other step uses
        E = cfg.E
        per_q = np.diff(po) + np.diff(to).reshape(-1, E).sum(axis=1)
        assert np.array_equal(per_q, gi.ctx_len)
        out = oracle.assemble_context(oc["survivor_idx"], oc["cu_seqlens"], pt, po, tt, to, E)
        cu, L = oc["cu_seqlens"], np.diff(oc["cu_seqlens"])
        T = oc["total_tokens"]
        assert out["n_mismatch"] == 0
        assert np.array_equal(out["position_ids"], np.arange(T) - np.repeat(cu[:-1], L))
        src = np.concatenate([np.concatenate([pt[po[q]:po[q + 1]], tt[to[q * E]:to[q * E + E]]])
                              for q in oc["survivor_idx"]] + [np.empty(0, np.int32)])
        assert np.array_equal(out["input_ids"], src)  # traces of one question are adjacent in (q, e) order


def test_length_mismatch_is_counted_truncated_or_padded():
    pt = np.array([10, 11, 12], np.int32)
    po = np.array([0, 1, 3], np.int64)            # prompts: [10], [11, 12]
    tt = np.array([20, 21, 22, 23], np.int32)
    to = np.array([0, 2, 4], np.int64)            # E = 1 traces: [20, 21], [22, 23]
    idx = np.array([0, 1], np.int32)
    cu = np.array([0, 2, 8], np.int64)            # says 2 and 6 tokens; the sources have 3 and 4
    out = oracle.assemble_context(idx, cu, pt, po, tt, to, 1)
    assert out["n_mismatch"] == 2
    assert out["input_ids"].tolist() == [10, 20, 11, 12, 22, 23, -1, -1]
    assert out["position_ids"].tolist() == [0, 1, 0, 1, 2, 3, 4, 5]
