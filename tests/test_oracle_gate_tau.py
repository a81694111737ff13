"""Pins of oracle.gate_tau_per_query against the already pinned scalar gate:
a constant threshold array reproduces it; mixing two thresholds equals stitching the two scalar
runs by rows; thresholds of -inf / +inf / NaN bypass everything / nothing / nothing; and the
paper's k = 3 rule by hand (agreement 2/3 passes tau = 2/3 but not tau = 0.7)."""
import numpy as np

import oracle
from paper_2606_03014_b200 import workloads as wl


def test_constant_threshold_is_the_scalar_gate():
    for cfg, mode in ((wl.C1, 0), (wl.C2, 1)):
        gi = wl.gate_inputs(cfg, 0)
        a = oracle.gate(gi.answers, gi.tau, gi.expert_conf, mode)
        b = oracle.gate_tau_per_query(gi.answers, np.full(cfg.Q, gi.tau, np.float32), gi.expert_conf, mode)
        for k in a:
            assert np.array_equal(a[k], b[k]), k


def test_two_thresholds_stitch_two_scalar_runs():
    gi = wl.gate_inputs(wl.C4, 1)
    Q = gi.answers.shape[0]
    pick = np.random.default_rng(0).random(Q) < 0.5
    lo, hi = oracle.gate(gi.answers, 0.5), oracle.gate(gi.answers, 0.75)
    tau_q = np.where(pick, 0.5, 0.75).astype(np.float32)
    got = oracle.gate_tau_per_query(gi.answers, tau_q)
    assert np.array_equal(got["bypass"], np.where(pick, lo["bypass"], hi["bypass"]))
    assert np.array_equal(got["mode"], lo["mode"]) and np.array_equal(got["conf"], lo["conf"])


def test_extreme_thresholds_and_the_k3_rule():
    ans = np.array([[1, 1, 2], [1, 2, 3], [4, 4, 4], [5, 6, 5]], np.int32)
    inf = np.float32(np.inf)
    g = oracle.gate_tau_per_query
    assert g(ans, np.full(4, -inf))["bypass"].tolist() == [1, 1, 1, 1]
    assert g(ans, np.full(4, inf))["bypass"].tolist() == [0, 0, 0, 0]
    assert g(ans, np.full(4, np.nan, np.float32))["bypass"].tolist() == [0, 0, 0, 0]
    tau = np.array([2 / 3, 1 / 3, 1.0, 0.7], np.float32)
    assert g(ans, tau)["bypass"].tolist() == [1, 1, 1, 0]
