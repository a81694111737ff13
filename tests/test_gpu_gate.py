"""GPU parity, step 1: mosaic_gate / mosaic_compact / mosaic_gate_compact against the oracle,
bit-exact (BASELINE.json north_star), on the five configs x seeds {0,1,2} (the paper's seed set,
P:L350) plus the edge cases of the boundary."""
import numpy as np
import pytest
import torch

import _parity as P
import oracle
from paper_2606_03014_b200 import mosaic
from paper_2606_03014_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("seed", [0, 1, 2])
@pytest.mark.parametrize("cid", [1, 2, 3, 4])
def test_configs_bit_exact(cid, seed):
    from paper_2606_03014_b200 import mosaic  # noqa: F401  (fails loudly if the .so is missing)
    cfg = wl.CONFIGS[cid]
    gi = wl.gate_inputs(cfg, seed)
    for conf_mode in ([0, 1] if cfg.has_conf else [0]):
        want = P.oracle_gate_compact(gi, conf_mode)
        sep, fused = P.gpu_gate_compact_all(gi, conf_mode)
        P.assert_gate_equal(sep, want)
        P.assert_gate_equal(fused, want)


@pytest.mark.parametrize("p_agree,tau", wl.C5_SWEEP)
def test_c5_sweep_bit_exact(p_agree, tau):
    """2^20 questions, E = 8, both confidence modes, int64 cu_seqlens past 2^31 tokens."""
    cfg = wl.C5
    gi = wl.gate_inputs(cfg, 0, p_agree=p_agree, tau=tau)
    for conf_mode in (0, 1):
        want = P.oracle_gate_compact(gi, conf_mode)
        sep, fused = P.gpu_gate_compact_all(gi, conf_mode)
        P.assert_gate_equal(sep, want)
        P.assert_gate_equal(fused, want)
    assert want["total_tokens"] > 2 ** 31 or want["n_survivors"] < 2 ** 17


@pytest.mark.parametrize("E", [1, 2, 3, 4, 5, 6, 7, 8, 9, 13, 16, 32])
def test_every_expert_count_and_ragged_sizes(E):
    g = np.random.default_rng(100 + E)
    for Q in (1, 31, 255, 256, 257, 1023, 1025, 4097, 70001):
        a = g.integers(-3, 4, size=(Q, E), dtype=np.int32)
        w = (g.integers(0, 1 << 24, size=(Q, E)).astype(np.float64) * 2.0 ** -24).astype(np.float32)
        ctx = g.integers(0, 50000, size=Q, dtype=np.int32)
        for tau in (0.5, 2.0 / 3.0, 1.0):
            gi = wl.GateInputs(a, w, ctx, tau, E)
            for conf_mode in (0, 1):
                want = P.oracle_gate_compact(gi, conf_mode)
                sep, fused = P.gpu_gate_compact_all(gi, conf_mode)
                P.assert_gate_equal(sep, want)
                P.assert_gate_equal(fused, want)


def test_all_bypass_none_bypass_and_empty():
    from paper_2606_03014_b200 import mosaic
    Q, E = 5000, 3
    a = np.tile(np.array([[4, 4, 4]], np.int32), (Q, 1))
    ctx = np.arange(1, Q + 1, dtype=np.int32)
    for tau, S in ((1.0, 0), (1.5, Q)):
        gi = wl.GateInputs(a, None, ctx, tau, E)
        want = P.oracle_gate_compact(gi, 0)
        assert want["n_survivors"] == S
        sep, fused = P.gpu_gate_compact_all(gi, 0)
        P.assert_gate_equal(sep, want)
        P.assert_gate_equal(fused, want)
    # Q == 0: success, S = 0, cu_seqlens = [0]
    e8 = torch.empty(0, dtype=torch.uint8, device="cuda")
    e32 = torch.empty(0, dtype=torch.int32, device="cuda")
    out = dict(n_survivors=torch.full((1,), 7, dtype=torch.int32, device="cuda"),
               total_tokens=torch.full((1,), 7, dtype=torch.int64, device="cuda"),
               max_seqlen=torch.full((1,), 7, dtype=torch.int32, device="cuda"),
               cu_seqlens=torch.full((1,), 7, dtype=torch.int64, device="cuda"))
    r = mosaic.compact(e8, e32, out=out)
    torch.cuda.synchronize()
    assert (int(r["n_survivors"]), int(r["total_tokens"]), int(r["max_seqlen"]),
            int(r["cu_seqlens"][0])) == (0, 0, 0, 0)


def test_workspace_contents_do_not_matter_and_calls_repeat():
    """The scan workspace is caller scratch with arbitrary contents; repeated calls on the same
    buffers give the same answer (no state between calls)."""
    from paper_2606_03014_b200 import mosaic
    cfg = wl.C4
    gi = wl.gate_inputs(cfg, 1, Q=100000)
    want = P.oracle_gate_compact(gi, 0)
    a = torch.from_numpy(gi.answers).cuda()
    cl = torch.from_numpy(gi.ctx_len).cuda()
    ws = torch.randint(0, 255, (mosaic.compact_workspace_bytes(len(cl)),), dtype=torch.uint8,
                       device="cuda")
    for _ in range(3):
        r = mosaic.gate_compact(a, cl, gi.tau, out=dict(workspace=ws))
        torch.cuda.synchronize()
        S = int(r["n_survivors"])
        assert S == want["n_survivors"]
        assert np.array_equal(r["survivor_idx"][:S].cpu().numpy(), want["survivor_idx"])
        assert np.array_equal(r["cu_seqlens"][:S + 1].cpu().numpy(), want["cu_seqlens"])
        ws.random_(0, 255)


def test_too_small_workspace_is_an_error():
    from paper_2606_03014_b200 import mosaic
    by = torch.zeros(100000, dtype=torch.uint8, device="cuda")
    cl = torch.ones(100000, dtype=torch.int32, device="cuda")
    with pytest.raises(mosaic.MosaicError) as e:
        mosaic.compact(by, cl, out=dict(workspace=torch.empty(64, dtype=torch.uint8, device="cuda")))
    assert e.value.status == mosaic.ERR_WORKSPACE_TOO_SMALL


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_n4_paper_shaped_workload_bit_exact(seed):
    """the paper-shaped inputs bench.py's gated-stage leg runs (k = 3, MMLU-Pro bucket
    rates, trace lengths falling with agreement) through the gate and the
    compaction at the paper's two operating points (tau = 2/3 and 1) against the oracle."""
    for Q in (768, 50000):
        a, ctx, _ = wl.n4_inputs(seed, Q)
        for tau in (2.0 / 3.0, 1.0):
            gi = wl.GateInputs(a, None, ctx, tau, 3)
            want = P.oracle_gate_compact(gi, 0)
            sep, fused = P.gpu_gate_compact_all(gi, 0)
            P.assert_gate_equal(sep, want)
            P.assert_gate_equal(fused, want)
        assert 0.80 < 1.0 - P.oracle_gate_compact(wl.GateInputs(a, None, ctx, 2.0 / 3.0, 3), 0)[
            "n_survivors"] / Q < 0.89   # Table 1: 84.62 % skipped at tau = 2/3


def _wide_weights(g, Q, E):
    """fp32 weights spread over 2^+-40 with zeros and all-zero rows: the binary64 sums round (a
    kernel that accumulated in fp32, or dropped the small terms, would show in conf's bits)."""
    w = np.exp2(g.uniform(-40.0, 40.0, size=(Q, E))).astype(np.float32)
    w[g.random((Q, E)) < 0.1] = 0.0
    w[::97] = 0.0                                            # St = 0: conf falls back to agree
    return w


@pytest.mark.parametrize("E", [3, 5, 8, 13])
def test_weights_of_very_different_magnitudes(E):
    g = np.random.default_rng(500 + E)
    Q = 30011
    a = g.integers(0, 3, size=(Q, E), dtype=np.int32)
    w = _wide_weights(g, Q, E)
    ctx = g.integers(0, 50000, size=Q, dtype=np.int32)
    gi = wl.GateInputs(a, w, ctx, 0.6, E)
    want = P.oracle_gate_compact(gi, 1)
    assert 0.05 < want["bypass"].mean() < 0.95              # both outcomes occur
    sep, fused = P.gpu_gate_compact_all(gi, 1)
    P.assert_gate_equal(sep, want)
    P.assert_gate_equal(fused, want)
    # the weighted-argmax estimator: per-label sums, ties between labels included (zero rows)
    want2 = oracle.gate_ext(a, 0.6, w, 2)
    r = mosaic.gate_compact_ext(torch.from_numpy(a).cuda(), torch.from_numpy(ctx).cuda(), 0.6,
                                torch.from_numpy(w).cuda(), 2)
    torch.cuda.synchronize()
    assert np.array_equal(r["mode"].cpu().numpy(), want2["mode"])
    assert np.array_equal(r["conf"].cpu().numpy().view(np.uint32), want2["conf"].view(np.uint32))
    assert np.array_equal(r["bypass"].cpu().numpy(), want2["bypass"])


def test_sixteen_million_questions_bit_exact():
    """2^24 + 12 345 questions (E = 8, weighted): ~57 tiles per block of the persistent grid, a ragged
    last tile, token totals far beyond 2^31 -- the size of bench.py's supplementary gate point."""
    cfg = wl.C5
    Q = (1 << 24) + 12345
    gi = wl.gate_inputs(cfg, 3, Q=Q)
    want = P.oracle_gate_compact(gi, 1)
    assert want["total_tokens"] > 2 ** 37
    a = torch.from_numpy(gi.answers).cuda()
    w = torch.from_numpy(gi.expert_conf).cuda()
    cl = torch.from_numpy(gi.ctx_len).cuda()
    for _ in range(2):                                        # (the second call reuses the workspace)
        r = mosaic.gate_compact(a, cl, gi.tau, w, 1, want_count=True, want_agree=True)
        torch.cuda.synchronize()
        S = int(r["n_survivors"])
        got = dict(mode=r["mode"].cpu().numpy(), count=r["count"].cpu().numpy(),
                   agree=r["agree"].cpu().numpy(), conf=r["conf"].cpu().numpy(),
                   bypass=r["bypass"].cpu().numpy(), survivor_idx=r["survivor_idx"][:S].cpu().numpy(),
                   cu_seqlens=r["cu_seqlens"][:S + 1].cpu().numpy(), n_survivors=S,
                   total_tokens=int(r["total_tokens"]), max_seqlen=int(r["max_seqlen"]))
        P.assert_gate_equal(got, want)


def test_concurrent_calls_on_three_streams():
    """Three fused calls at a time on three streams (own workspaces and outputs): their persistent
    grids cannot all be resident, so a scan that needed every block of a call on the GPU at once
    would hang here; tiles are handed out by ticket in start order and a tile only waits for
    smaller tickets, whose blocks are running.  Results bit-exact as ever."""
    cfg = wl.C5
    Q = 1 << 20
    gis = [wl.gate_inputs(cfg, seed, Q=Q) for seed in (0, 1, 2)]
    wants = [P.oracle_gate_compact(gi, 1) for gi in gis]
    dev = []
    for gi in gis:
        a = torch.from_numpy(gi.answers).cuda()
        w = torch.from_numpy(gi.expert_conf).cuda()
        cl = torch.from_numpy(gi.ctx_len).cuda()
        dev.append((a, w, cl, mosaic.gate_compact(a, cl, gi.tau, w, 1)))
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream() for _ in gis]
    for _ in range(6):
        for (a, w, cl, out), gi, st in zip(dev, gis, streams):
            mosaic.gate_compact(a, cl, gi.tau, w, 1, out=out, stream=st)
    torch.cuda.synchronize()
    for (a, w, cl, r), want in zip(dev, wants):
        S = int(r["n_survivors"])
        assert S == want["n_survivors"] and int(r["total_tokens"]) == want["total_tokens"]
        assert int(r["max_seqlen"]) == want["max_seqlen"]
        assert np.array_equal(r["bypass"].cpu().numpy(), want["bypass"])
        assert np.array_equal(r["conf"].cpu().numpy().view(np.uint32), want["conf"].view(np.uint32))
        assert np.array_equal(r["survivor_idx"][:S].cpu().numpy(), want["survivor_idx"])
        assert np.array_equal(r["cu_seqlens"][:S + 1].cpu().numpy(), want["cu_seqlens"])
