"""Pins of oracle.gate_ext / oracle.conf_gate (readings N3-1..N3-3),
none of which restates the C loop: hand-worked k = 3 cases under both abstention policies,
reductions to the (already pinned) plain gate, an all-abstaining extra expert that must drop out,
equal weights reducing the weighted argmax to the count plurality, and exact rational arithmetic
for the weighted argmax on weights that are multiples of 2^-24."""
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_2606_03014_b200 import workloads as wl

SENT = -7  # the sentinel a failed Extract returns in these tests


def _f32(x: Fraction) -> np.float32:
    """Nearest fp32 to an exact rational (numpy rounds the binary64 quotient of two exactly
    representable integers; all cases below have numerators and denominators < 2^53 and quotients
    that are not fp32 rounding ties of the binary64 value)."""
    return np.float32(x.numerator / x.denominator)


def test_hand_cases_k3_one_abstention():
    """k = 3 with one failed Extract.  Literal P:L182 divides by k = 3 ("keep k"): a 2:0
    vote has C = 2/3 and just passes tau = 2/3, a 1:1 vote has C = 1/3; dividing by the
    two experts that answered ("shrink k") makes them 1 and 1/2.  The sentinel never wins."""
    a = np.array([[4, 4, SENT], [9, 2, SENT], [SENT, 5, 5], [SENT, SENT, 8], [SENT] * 3], np.int32)
    keep = oracle.gate_ext(a, 2 / 3, abstain_policy=1, abstain_label=SENT)
    assert keep["mode"].tolist() == [4, 2, 5, 8, SENT]
    assert keep["count"].tolist() == [2, 1, 2, 1, 0]
    assert keep["agree"].tolist() == [np.float32(2) / np.float32(3), np.float32(1) / np.float32(3),
                                      np.float32(2) / np.float32(3), np.float32(1) / np.float32(3), 0.0]
    assert keep["bypass"].tolist() == [1, 0, 1, 0, 0]
    shrink = oracle.gate_ext(a, 2 / 3, abstain_policy=2, abstain_label=SENT)
    assert shrink["mode"].tolist() == [4, 2, 5, 8, SENT]
    assert shrink["agree"].tolist() == [1.0, 0.5, 1.0, 1.0, 0.0]
    assert shrink["bypass"].tolist() == [1, 0, 1, 1, 0]
    # every expert abstaining: no answer, C = 0, bypassed only by a threshold <= 0
    assert oracle.gate_ext(a, 0.0, abstain_policy=1, abstain_label=SENT)["bypass"].tolist() == [1] * 5
    # without a policy the sentinel is one more label (reading G-6): [SENT, SENT, 8] is a 2:1 vote
    none = oracle.gate_ext(a, 2 / 3)
    assert none["mode"].tolist() == [4, SENT, 5, SENT, SENT] and none["count"].tolist() == [2, 1, 2, 2, 3]


@pytest.mark.parametrize("cid", [1, 2, 4])
def test_no_sentinel_present_is_the_plain_gate(cid):
    """Policies 1 / 2 with a sentinel that never occurs, and conf modes 0 / 1, reproduce oracle.gate
    bit for bit; a constant tau_q reproduces the scalar threshold."""
    cfg = wl.CONFIGS[cid]
    gi = wl.gate_inputs(cfg, 0)
    for mode in ([0, 1] if cfg.has_conf else [0]):
        want = oracle.gate(gi.answers, gi.tau, gi.expert_conf, mode)
        for pol in (0, 1, 2):
            got = oracle.gate_ext(gi.answers, gi.tau, gi.expert_conf, mode, abstain_policy=pol,
                                  abstain_label=12345)
            for k in want:
                assert np.array_equal(got[k].view(np.uint8), want[k].view(np.uint8)), (k, mode, pol)
        tq = np.full(cfg.Q, gi.tau, np.float32)
        got = oracle.gate_ext(gi.answers, 99.0, gi.expert_conf, mode, tau_q=tq)
        assert np.array_equal(got["bypass"], want["bypass"])


@pytest.mark.parametrize("mode", [0, 1, 2])
def test_an_abstaining_extra_expert_drops_out(mode):
    """Append an expert that always abstains (with any weight).  Shrink-k: every output equals the
    gate on the original E experts.  Keep-k: same mode and count, agree = count / (E + 1), and the
    weight share's denominator gains the abstainer's weight."""
    cfg = wl.C2
    gi = wl.gate_inputs(cfg, 1)
    Q, E = gi.answers.shape
    a2 = np.concatenate([gi.answers, np.full((Q, 1), SENT, np.int32)], axis=1)
    w_extra = wl.expert_conf(cfg, 5)[:, :1]
    w2 = np.concatenate([gi.expert_conf, w_extra], axis=1)
    want = oracle.gate_ext(gi.answers, gi.tau, gi.expert_conf, mode)
    got = oracle.gate_ext(a2, gi.tau, w2, mode, abstain_policy=2, abstain_label=SENT)
    for k in want:
        assert np.array_equal(got[k].view(np.uint8), want[k].view(np.uint8)), k
    keep = oracle.gate_ext(a2, gi.tau, w2, mode, abstain_policy=1, abstain_label=SENT)
    assert np.array_equal(keep["count"], want["count"])
    assert np.array_equal(keep["agree"], keep["count"].astype(np.float32) / np.float32(E + 1))
    if mode == 0:
        assert np.array_equal(keep["mode"], want["mode"])
    else:
        # weights are multiples of 2^-24: every sum is exact, the share is an exact rational
        for q in range(Q):
            st = sum(Fraction(float(x)) for x in w2[q])
            sm = sum(Fraction(float(w2[q, i])) for i in range(E) if a2[q, i] == keep["mode"][q])
            assert keep["conf"][q] == _f32(sm / st), q


def test_weighted_argmax_with_equal_weights_is_the_count_plurality():
    g = np.random.default_rng(3)
    for E in (3, 4, 5, 8):
        a = g.integers(0, 4, size=(4000, E), dtype=np.int32)
        w = np.full((4000, E), 0.5, np.float32)
        vote = oracle.gate(a, 0.5)
        got = oracle.gate_ext(a, 0.5, w, 2)
        assert np.array_equal(got["mode"], vote["mode"]) and np.array_equal(got["count"], vote["count"])
        assert np.array_equal(got["conf"], vote["agree"]) and np.array_equal(got["bypass"], vote["bypass"])
        # weights that do not add up to anything positive: the vote rule, C = the vote fraction
        zero = oracle.gate_ext(a, 0.5, np.zeros_like(w), 2)
        assert np.array_equal(zero["mode"], vote["mode"]) and np.array_equal(zero["conf"], vote["agree"])


def test_weighted_argmax_against_exact_rationals():
    """mode = the label with the largest exact weight sum (ties -> smallest label), C its exact
    share, on 10-option answers with weights on the 2^-24 grid; a minority label with heavy weights
    must beat the plurality."""
    cfg = wl.C5
    a = wl.answers(cfg, 2, Q=3000)
    w = wl.expert_conf(cfg, 2, Q=3000)
    w[::7, 0] = 0.0                      # some zero weights
    a[::11, 1] = a[::11, 0]              # some exact ties between two labels' sums
    w[::11, 1] = w[::11, 0]
    got = oracle.gate_ext(a, 0.4, w, 2)
    vote = oracle.gate(a, 0.4)
    differs = 0
    for q in range(a.shape[0]):
        sums = {}
        for x, ww in zip(a[q].tolist(), w[q]):
            sums[x] = sums.get(x, Fraction(0)) + Fraction(float(ww))
        best = max(sums.values())
        mode = min(x for x, s in sums.items() if s == best)
        assert got["mode"][q] == mode, q
        assert got["count"][q] == int((a[q] == mode).sum())
        assert got["conf"][q] == _f32(best / sum(sums.values())), q
        assert got["bypass"][q] == int(got["conf"][q] >= np.float32(0.4))
        differs += int(mode != vote["mode"][q])
    assert differs > 50                  # the estimator is not the count plurality in disguise
    perm = np.random.default_rng(0).permutation(cfg.E)
    again = oracle.gate_ext(a[:, perm], 0.4, w[:, perm], 2)
    for k in got:
        assert np.array_equal(again[k].view(np.uint8), got[k].view(np.uint8)), k   # exact sums: order-free


def test_conf_gate_is_line_4_of_alg_1():
    """oracle.conf_gate on the confidences the (pinned) gate computed reproduces its mask; NaN on
    either side never bypasses; -inf / +inf thresholds bypass all / none."""
    cfg = wl.C2
    gi = wl.gate_inputs(cfg, 0)
    for mode in (0, 1):
        g = oracle.gate(gi.answers, gi.tau, gi.expert_conf, mode)
        assert np.array_equal(oracle.conf_gate(g["conf"], gi.tau), g["bypass"])
    c = np.array([0.5, np.nan, 1.0, 0.0], np.float32)
    assert oracle.conf_gate(c, 0.5).tolist() == [1, 0, 1, 0]
    assert oracle.conf_gate(c, 0.0, tau_q=np.array([np.nan, 0.0, -np.inf, np.inf], np.float32)).tolist() \
        == [0, 0, 1, 0]
