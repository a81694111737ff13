"""GPU parity of mosaic_gate_compact_tau against oracle.gate_tau_per_query +
oracle.compact: bit-exact."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_03014_b200 import mosaic
from paper_2606_03014_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cid,mode", [(1, 0), (2, 1), (4, 0), (5, 1)])
def test_task_table_thresholds_bit_exact(cid, mode):
    cfg = wl.CONFIGS[cid]
    Q = min(cfg.Q, 1 << 17)
    gi = wl.gate_inputs(cfg, 0, Q=Q) if cid == 5 else wl.gate_inputs(cfg, 0)
    Q = gi.answers.shape[0]
    rng = np.random.default_rng(cid)
    table = np.array([0.5, 2 / 3, 0.75, 1.0, np.nan, -np.inf], np.float32)   # six "tasks"
    tau_q = table[rng.integers(0, len(table), size=Q)]
    w = gi.expert_conf if mode == 1 else None
    want = oracle.gate_tau_per_query(gi.answers, tau_q, w, mode)
    oc = oracle.compact(want["bypass"], gi.ctx_len)
    d = lambda a: None if a is None else torch.from_numpy(a).cuda()
    r = mosaic.gate_compact_tau(d(gi.answers), d(gi.ctx_len), d(tau_q), d(w), mode)
    torch.cuda.synchronize()
    S = int(r["n_survivors"])
    assert np.array_equal(r["bypass"].cpu().numpy(), want["bypass"])
    assert np.array_equal(r["mode"].cpu().numpy(), want["mode"])
    assert np.array_equal(r["conf"].cpu().numpy().view(np.uint32), want["conf"].view(np.uint32))
    assert S == oc["n_survivors"] and int(r["total_tokens"]) == oc["total_tokens"]
    assert int(r["max_seqlen"]) == oc["max_seqlen"]
    assert np.array_equal(r["survivor_idx"][:S].cpu().numpy(), oc["survivor_idx"])
    assert np.array_equal(r["cu_seqlens"][:S + 1].cpu().numpy(), oc["cu_seqlens"])
