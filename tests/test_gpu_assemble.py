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


@pytest.mark.parametrize("cid", [1, 2, 4])
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
    """E = 1 and E = 8, empty prompts and traces, sequences around the 2048-token block edge,
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
        t_len[1, E - 1] = 2048                         # exactly one block
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
