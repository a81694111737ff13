"""GPU parity of the SURVEY.md 8(f) N3 estimators -- mosaic_gate_compact_ext (weighted argmax,
abstention sentinel with keep-k / shrink-k, optional per-question tau), mosaic_gate with
MOSAIC_CONF_WEIGHTED_ARGMAX and mosaic_conf_compact -- against oracle.gate_ext / oracle.conf_gate +
oracle.compact: bit-exact on every output (floats as bit patterns)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_03014_b200 import mosaic
from paper_2606_03014_b200 import workloads as wl

pytestmark = pytest.mark.gpu
SENT = -1


def _d(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _check(r, want, ctx_len):
    oc = oracle.compact(want["bypass"], ctx_len)
    S = int(r["n_survivors"])
    for k in ("mode", "count", "bypass"):
        assert np.array_equal(r[k].cpu().numpy(), want[k]), k
    for k in ("agree", "conf"):
        assert np.array_equal(r[k].cpu().numpy().view(np.uint32), want[k].view(np.uint32)), k
    assert S == oc["n_survivors"] and int(r["total_tokens"]) == oc["total_tokens"]
    assert int(r["max_seqlen"]) == oc["max_seqlen"]
    assert np.array_equal(r["survivor_idx"][:S].cpu().numpy(), oc["survivor_idx"])
    assert np.array_equal(r["cu_seqlens"][:S + 1].cpu().numpy(), oc["cu_seqlens"])


def _inputs(cid, abstain_rate, Q=None):
    cfg = wl.CONFIGS[cid]
    gi = wl.gate_inputs(cfg, 0, Q=Q)
    a = gi.answers.copy()
    g = np.random.default_rng(40 + cid)
    if abstain_rate:
        a[g.random(a.shape) < abstain_rate] = SENT      # failed Extracts
        a[:3] = SENT                                     # questions nobody answered
    w = gi.expert_conf if gi.expert_conf is not None else wl.expert_conf(cfg, 0, Q=a.shape[0])
    return cfg, a, w, gi.ctx_len, gi.tau


@pytest.mark.parametrize("policy", [mosaic.ABSTAIN_NONE, mosaic.ABSTAIN_KEEP_K, mosaic.ABSTAIN_SHRINK_K])
@pytest.mark.parametrize("conf_mode", [0, 1, 2])
@pytest.mark.parametrize("cid", [1, 2, 4])
def test_configs_every_estimator_bit_exact(cid, conf_mode, policy):
    cfg, a, w, ctx, tau = _inputs(cid, 0.15 if policy else 0.0)
    want = oracle.gate_ext(a, tau, w, conf_mode, abstain_policy=policy, abstain_label=SENT)
    r = mosaic.gate_compact_ext(_d(a), _d(ctx), tau, _d(w) if conf_mode else None, conf_mode,
                                abstain_policy=policy, abstain_label=SENT)
    torch.cuda.synchronize()
    _check(r, want, ctx)


@pytest.mark.parametrize("conf_mode,policy", [(2, 0), (0, 1), (1, 2), (2, 1), (2, 2)])
def test_c5_large_bit_exact_with_task_thresholds(conf_mode, policy):
    """configs[4] at its full 2^20 questions (E = 8), a six-entry tau table on top."""
    cfg, a, w, ctx, tau = _inputs(5, 0.2 if policy else 0.0)
    table = np.array([0.5, 2 / 3, 0.75, 1.0, np.nan, -np.inf], np.float32)
    tau_q = table[np.random.default_rng(9).integers(0, len(table), size=a.shape[0])]
    want = oracle.gate_ext(a, 0.0, w, conf_mode, tau_q=tau_q, abstain_policy=policy, abstain_label=SENT)
    r = mosaic.gate_compact_ext(_d(a), _d(ctx), 0.0, _d(w) if conf_mode else None, conf_mode,
                                tau_per_query=_d(tau_q), abstain_policy=policy, abstain_label=SENT)
    torch.cuda.synchronize()
    _check(r, want, ctx)
    assert 0 < int(r["n_survivors"]) < a.shape[0]


@pytest.mark.parametrize("E", [1, 2, 3, 5, 6, 7, 8, 9, 17, 32])
def test_every_expert_count_ragged_sizes(E):
    """Small label alphabets (many ties, in votes and in weight sums), every kernel specialisation
    and the generic E > 8 path, ragged question counts."""
    g = np.random.default_rng(300 + E)
    for Q in (1, 255, 1793, 40001):
        a = g.integers(-1, 3, size=(Q, E), dtype=np.int32)           # -1 doubles as the sentinel
        w = (g.integers(0, 4, size=(Q, E)).astype(np.float32) * 0.25)  # ties and zero rows
        ctx = g.integers(0, 50000, size=Q, dtype=np.int32)
        for conf_mode, policy in ((2, 0), (2, 1), (2, 2), (1, 1), (0, 2)):
            want = oracle.gate_ext(a, 0.5, w, conf_mode, abstain_policy=policy, abstain_label=SENT)
            r = mosaic.gate_compact_ext(_d(a), _d(ctx), 0.5, _d(w) if conf_mode else None, conf_mode,
                                        abstain_policy=policy, abstain_label=SENT)
            torch.cuda.synchronize()
            _check(r, want, ctx)


def test_gate_alone_takes_the_weighted_argmax():
    cfg, a, w, ctx, tau = _inputs(2, 0.0)
    want = oracle.gate_ext(a, tau, w, 2)
    r = mosaic.gate(_d(a), tau, _d(w), mosaic.CONF_WEIGHTED_ARGMAX)
    torch.cuda.synchronize()
    for k in ("mode", "count", "bypass"):
        assert np.array_equal(r[k].cpu().numpy(), want[k]), k
    for k in ("agree", "conf"):
        assert np.array_equal(r[k].cpu().numpy().view(np.uint32), want[k].view(np.uint32)), k


@pytest.mark.parametrize("cid", [1, 2, 4, 5])
def test_conf_compact_bit_exact(cid):
    """A caller-supplied C(q) (here: the weighted share the oracle's gate computes, with NaNs and
    infinities sprinkled in), scalar and per-question thresholds."""
    cfg, a, w, ctx, tau = _inputs(cid, 0.0)
    conf = oracle.gate(a, tau, w, 1)["conf"].copy()
    g = np.random.default_rng(cid)
    conf[g.random(conf.shape) < 0.01] = np.nan
    conf[g.random(conf.shape) < 0.01] = np.inf
    Q = conf.shape[0]
    tau_q = np.array([0.5, 0.75, np.nan, -np.inf], np.float32)[g.integers(0, 4, size=Q)]
    for tq in (None, tau_q):
        by = oracle.conf_gate(conf, tau, tq)
        oc = oracle.compact(by, ctx)
        r = mosaic.conf_compact(_d(conf), _d(ctx), tau, tau_per_query=_d(tq))
        torch.cuda.synchronize()
        S = int(r["n_survivors"])
        assert np.array_equal(r["bypass"].cpu().numpy(), by)
        assert S == oc["n_survivors"] and int(r["total_tokens"]) == oc["total_tokens"]
        assert int(r["max_seqlen"]) == oc["max_seqlen"]
        assert np.array_equal(r["survivor_idx"][:S].cpu().numpy(), oc["survivor_idx"])
        assert np.array_equal(r["cu_seqlens"][:S + 1].cpu().numpy(), oc["cu_seqlens"])


def test_argument_errors():
    a = torch.zeros((4, 3), dtype=torch.int32, device="cuda")
    ctx = torch.ones(4, dtype=torch.int32, device="cuda")
    with pytest.raises(mosaic.MosaicError) as e:
        mosaic.gate_compact_ext(a, ctx, 0.5, None, 0, abstain_policy=3)
    assert e.value.status == mosaic.ERR_INVALID_ARG
    with pytest.raises(mosaic.MosaicError) as e:
        mosaic.gate_compact_ext(a, ctx, 0.5, None, 2)           # weights required
    assert e.value.status == mosaic.ERR_INVALID_ARG
    with pytest.raises(mosaic.MosaicError) as e:
        mosaic.conf_compact(torch.zeros(4, device="cuda"), ctx, float("nan"))
    assert e.value.status == mosaic.ERR_INVALID_ARG
