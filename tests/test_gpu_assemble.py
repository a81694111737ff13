"""GPU parity of mosaic_assemble_context against the oracle: bit-exact."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_03014_b200 import mosaic
from paper_2606_03014_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _run(idx, cu, pt, po, tt, to, E):
    d = lambda a, t: torch.from_numpy(np.ascontiguousarray(a)).to(t).cuda()
    S = len(idx)
    L = np.diff(cu)
    ids, pos, mm = mosaic.assemble_context(
        d(idx if S else np.zeros(1, np.int32), torch.int32), d(cu, torch.int64), S,
        int(L.max()) if S else 0, int(cu[-1]),
        d(pt if len(pt) else np.zeros(1, np.int32), torch.int32), d(po, torch.int64),
        d(tt if len(tt) else np.zeros(1, np.int32), torch.int32), d(to, torch.int64), E)
    torch.cuda.synchronize()
    return ids.cpu().numpy(), pos.cpu().numpy(), int(mm.item())


@pytest.mark.parametrize("cid", [1, 2, 3, 4])
def test_configs_bit_exact(cid):
    cfg = wl.CONFIGS[cid]
    gi = wl.gate_inputs(cfg, 0)
    oc = oracle.compact(oracle.gate(gi.answers, gi.tau)["bypass"], gi.ctx_len)
    pt, po, tt, to = wl.context_parts(cfg, 0)
    want = oracle.assemble_context(oc["survivor_idx"], oc["cu_seqlens"], pt, po, tt, to, cfg.E)
    ids, pos, mm = _run(oc["survivor_idx"], oc["cu_seqlens"], pt, po, tt, to, cfg.E)
    assert mm == 0 == want["n_mismatch"]
    assert np.array_equal(ids, want["input_ids"]) and np.array_equal(pos, want["position_ids"])


def test_edges_bit_exact():
    """E = 1 and E = 8, empty prompts and traces, sequences of 2048 / 2049 tokens (several 16-byte
    store groups and a ragged tail; the 8192-token block edge is test_block_edges_and_every_expert_count),
    zero-length sequences, survivors in arbitrary (non-contiguous) question order."""
    g = np.random.default_rng(5)
    for E in (1, 8):
        Q = 37
        p_len = g.integers(0, 300, size=Q)
        t_len = g.integers(0, 900, size=(Q, E))
        t_len[g.random((Q, E)) < 0.25] = 0
        p_len[:3] = 0
        t_len[0] = 0                                   # question 0: an empty context
        t_len[1] = 0
        t_len[1, E - 1] = 2048
        t_len[2, 0] = 2049
        po = np.concatenate([[0], np.cumsum(p_len)]).astype(np.int64)
        to = np.concatenate([[0], np.cumsum(t_len.reshape(-1))]).astype(np.int64)
        pt = g.integers(0, wl.VOCAB, size=int(po[-1]), dtype=np.int32)
        tt = g.integers(0, wl.VOCAB, size=int(to[-1]), dtype=np.int32)
        ctx = (p_len + t_len.sum(axis=1)).astype(np.int32)
        idx = np.array([0, 1, 2, 5, 6, 11, 30, 36], np.int32)
        cu = np.concatenate([[0], np.cumsum(ctx[idx])]).astype(np.int64)
        want = oracle.assemble_context(idx, cu, pt, po, tt, to, E)
        ids, pos, mm = _run(idx, cu, pt, po, tt, to, E)
        assert mm == 0
        assert np.array_equal(ids, want["input_ids"]) and np.array_equal(pos, want["position_ids"])


def test_mismatch_and_empty():
    pt = np.array([10, 11, 12], np.int32)
    po = np.array([0, 1, 3], np.int64)
    tt = np.array([20, 21, 22, 23], np.int32)
    to = np.array([0, 2, 4], np.int64)
    idx = np.array([0, 1], np.int32)
    cu = np.array([0, 2, 8], np.int64)
    want = oracle.assemble_context(idx, cu, pt, po, tt, to, 1)
    ids, pos, mm = _run(idx, cu, pt, po, tt, to, 1)
    assert mm == want["n_mismatch"] == 2
    assert np.array_equal(ids, want["input_ids"]) and np.array_equal(pos, want["position_ids"])
    ids, pos, mm = _run(np.zeros(0, np.int32), np.zeros(1, np.int64), pt, po, tt, to, 1)
    assert ids.size == 0 and pos.size == 0 and mm == 0


@pytest.mark.parametrize("E", [1, 3, 8, 9, 15, 16, 17, 31, 32])
def test_block_edges_and_every_expert_count(E):
    """Every expert count the ABI accepts on both sides of the 16-segment and 32-segment marks
    (E + 1 segments: prompt + E traces), with contexts of exactly 8191 / 8192 / 8193 (one block of
    the kernel and one token more or less), 16385 and 32768 tokens (several blockIdx.y), empty
    segments in between and the boundaries of the segments falling anywhere."""
    g = np.random.default_rng(900 + E)
    totals = [8191, 8192, 8193, 16385, 32768, 5, 0, 24577, 1, 12000]
    Q = len(totals)
    p_len = np.array([min(256, n // 4) for n in totals], np.int64)
    t_len = np.zeros((Q, E), np.int64)
    for q, n in enumerate(totals):
        rest = n - int(p_len[q])
        cuts = np.sort(g.integers(0, rest + 1, size=E - 1)) if E > 1 else np.zeros(0, np.int64)
        edges = np.concatenate([[0], cuts, [rest]])
        t_len[q] = np.diff(edges)
    t_len[9, : E // 2] = 0                              # leading empty traces
    t_len[9, E - 1] += 12000 - int(p_len[9]) - int(t_len[9].sum())
    assert np.all(t_len >= 0) and np.array_equal(p_len + t_len.sum(axis=1), np.array(totals))
    po = np.concatenate([[0], np.cumsum(p_len)]).astype(np.int64)
    to = np.concatenate([[0], np.cumsum(t_len.reshape(-1))]).astype(np.int64)
    pt = g.integers(0, wl.VOCAB, size=int(po[-1]), dtype=np.int32)
    tt = g.integers(0, wl.VOCAB, size=int(to[-1]), dtype=np.int32)
    idx = np.array([4, 0, 1, 2, 3, 5, 6, 7, 8, 9], np.int32)   # not in question order
    cu = np.concatenate([[0], np.cumsum(np.array(totals)[idx])]).astype(np.int64)
    want = oracle.assemble_context(idx, cu, pt, po, tt, to, E)
    ids, pos, mm = _run(idx, cu, pt, po, tt, to, E)
    assert mm == 0 == want["n_mismatch"]
    assert np.array_equal(ids, want["input_ids"]) and np.array_equal(pos, want["position_ids"])


def test_c5_shaped_slice_bit_exact():
    """The shape bench.py times: E = 8, contexts of U{8192..32768} tokens (64 survivors of the
    configs[4] gate at p = 0.6, tau = 0.75)."""
    cfg = wl.C5
    Q = 256
    gi = wl.gate_inputs(cfg, 0, Q=Q)
    oc = oracle.compact(oracle.gate(gi.answers, gi.tau)["bypass"], gi.ctx_len)
    n = min(64, oc["n_survivors"])
    idx, cu = oc["survivor_idx"][:n], oc["cu_seqlens"][:n + 1]
    pt, po, tt, to = wl.context_parts(cfg, 0, Q=Q)
    want = oracle.assemble_context(idx, cu, pt, po, tt, to, cfg.E)
    ids, pos, mm = _run(idx, cu, pt, po, tt, to, cfg.E)
    assert mm == 0 == want["n_mismatch"] and int(np.diff(cu).max()) > 3 * 8192
    assert np.array_equal(ids, want["input_ids"]) and np.array_equal(pos, want["position_ids"])
