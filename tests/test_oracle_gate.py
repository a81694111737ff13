"""Pins for the gate + compaction oracle (oracle/mosaic_oracle.c) -- CPU only.

Each test checks the oracle against something other than itself: the values PAPER.md prints
(P:L184-186), invariants the definition fixes, a differently written brute-force restatement,
numpy library routines, exact rational arithmetic, and a closed-form probability.
"""
from fractions import Fraction
from itertools import product
from math import comb, factorial

import numpy as np
import pytest

import oracle
from paper_2606_03014_b200 import workloads as wl


# ------------------------------------------------------------------ paper worked values
def _read_golden(path):
    rows = []
    for line in path.read_text().splitlines():
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        f = line.split()
        rows.append(dict(bucket=f[0], a=[int(x) for x in f[1:4]], c=int(f[4]),
                         C=Fraction(f[5]), by1=int(f[6]), by23=int(f[7])))
    return rows


def test_paper_k3_buckets(golden_dir):
    """3:0, 2:1, 1:1:1 <-> C = 1, 2/3, 1/3.  P:L186: tau=1 gates 3:0 only, tau=2/3 gates
    3:0 and 2:1.  Catches '>' instead of '>=' and mixed-precision compares (reading G-4)."""
    rows = _read_golden(golden_dir / "gate_k3_buckets.txt")
    assert [r["bucket"] for r in rows] == ["3:0", "2:1", "1:1:1"]
    a = np.array([r["a"] for r in rows], np.int32)
    for tau, key in ((1.0, "by1"), (2.0 / 3.0, "by23")):
        out = oracle.gate(a, tau)
        assert out["count"].tolist() == [r["c"] for r in rows]
        assert out["bypass"].tolist() == [r[key] for r in rows]
        for r, agree in zip(rows, out["agree"]):
            assert agree == np.float32(r["C"].numerator) / np.float32(r["C"].denominator)
            assert abs(float(agree) - float(r["C"])) < 2 ** -24
    assert oracle.gate(a, 1.0)["mode"].tolist()[:2] == [4, 4]          # majority of 4,7,4 is 4


def test_fp32_compare_matches_exact_rational_decision():
    """Reading G-4: fl32(c)/fl32(E) >= fl32(p/q) decides exactly like c/E >= p/q for every
    E <= 32 and every threshold p/q with q <= 32 (the paper's 2/3 is not representable)."""
    for E in range(1, 33):
        # one question per attainable c*: c copies of label 0, the rest in runs shorter than c
        tables, cs = [], []
        for c in range(1, E + 1):
            row, lab = [0] * c, 100
            while len(row) < E:
                row += [lab] * max(1, min(c - 1, E - len(row)))
                lab += 1
            tables.append(row[:E])
            cs.append(c)
        a = np.array(tables, np.int32)
        for qd in range(1, 33):
            for pn in range(0, qd + 1):
                tau = Fraction(pn, qd)
                out = oracle.gate(a, np.float32(pn) / np.float32(qd))
                assert out["count"].tolist() == cs
                want = [int(Fraction(c, E) >= tau) for c in cs]
                assert out["bypass"].tolist() == want, (E, pn, qd)


# ------------------------------------------------------------------ invariants
@pytest.mark.parametrize("E", [1, 2, 3, 4, 5, 8, 17, 32])
def test_unanimous_always_bypass_all_distinct_never(E):
    g = np.random.default_rng(E)
    lab = g.integers(-5, 50, size=64, dtype=np.int32)
    una = np.repeat(lab[:, None], E, axis=1)
    for tau in (1.0, 2 / 3, 0.5, 0.01):
        out = oracle.gate(una, tau)
        assert np.all(out["count"] == E) and np.all(out["agree"] == np.float32(1.0))
        assert np.all(out["bypass"] == 1) and np.array_equal(out["mode"], lab)
    assert np.all(oracle.gate(una, np.nextafter(np.float32(1), np.float32(2)))["bypass"] == 0)
    if E > 1:
        dist = np.stack([g.permutation(1000)[:E] for _ in range(64)]).astype(np.int32)
        just_above = float(np.nextafter(np.float32(1.0) / np.float32(E), np.float32(1)))
        for tau in [t for t in (1.0, 2 / 3, 0.5) if Fraction(t) > Fraction(1, E)] + [just_above]:
            out = oracle.gate(dist, tau)
            assert np.all(out["count"] == 1) and np.all(out["bypass"] == 0)
            assert np.array_equal(out["mode"], dist.min(axis=1))       # tie -> smallest label (G-2)
            assert np.all(out["agree"] == np.float32(1) / np.float32(E))
        # C = 1/E exactly reaches tau = 1/E (">=")
        assert np.all(oracle.gate(dist, np.float32(1.0) / np.float32(E))["bypass"] == 1)


@pytest.mark.parametrize("cfg_id", [1, 2, 3, 4])
def test_permuting_experts_changes_nothing(cfg_id):
    cfg = wl.CONFIGS[cfg_id]
    gi = wl.gate_inputs(cfg, seed=1, Q=4096)
    w = wl.expert_conf(cfg, 1, Q=4096)
    g = np.random.default_rng(7)
    perm = np.stack([g.permutation(cfg.E) for _ in range(4096)])
    a2 = np.take_along_axis(gi.answers, perm, axis=1)
    w2 = np.take_along_axis(w, perm, axis=1)
    for mode in (0, 1):
        o1 = oracle.gate(gi.answers, gi.tau, w, mode)
        o2 = oracle.gate(a2, gi.tau, w2, mode)
        for k in o1:
            assert np.array_equal(o1[k], o2[k]), k


def test_tau_monotone_and_tau_independent_outputs():
    gi = wl.gate_inputs(wl.C4, seed=2)
    taus = [-1.0, 0.0, 0.25, 0.26, 0.5, 0.75, 1.0, 1.5]
    outs = [oracle.gate(gi.answers, t) for t in taus]
    assert np.all(outs[0]["bypass"] == 1) and np.all(outs[1]["bypass"] == 1)   # G-8: tau <= 0
    assert np.all(outs[-1]["bypass"] == 0)                                      # tau > 1
    for lo, hi in zip(outs[:-1], outs[1:]):
        assert np.all(hi["bypass"] <= lo["bypass"])
        for k in ("mode", "count", "agree"):
            assert np.array_equal(lo[k], hi[k])


def test_order_preserving_relabel_maps_mode_only():
    gi = wl.gate_inputs(wl.C3, seed=0, Q=2048)
    f = lambda x: 7 * x - 1000                       # strictly increasing
    o1 = oracle.gate(gi.answers, gi.tau)
    o2 = oracle.gate(f(gi.answers).astype(np.int32), gi.tau)
    assert np.array_equal(f(o1["mode"]), o2["mode"])
    for k in ("count", "agree", "conf", "bypass"):
        assert np.array_equal(o1[k], o2[k])


# ------------------------------------------------------------------ brute force
def _restated(row):
    """A second statement of P:L182/L178: sort, run-length encode, take the longest run
    (first longest run of the sorted row = smallest label)."""
    s = sorted(row)
    best_c, best_x, i = 0, None, 0
    while i < len(s):
        j = i
        while j < len(s) and s[j] == s[i]:
            j += 1
        if j - i > best_c:
            best_c, best_x = j - i, s[i]
        i = j
    return best_x, best_c


def test_all_triples_of_ten_options():
    a = np.array(list(product(range(10), repeat=3)), np.int32)
    out = oracle.gate(a, 2 / 3)
    want = [_restated(r) for r in a.tolist()]
    assert out["mode"].tolist() == [w[0] for w in want]
    assert out["count"].tolist() == [w[1] for w in want]
    assert out["bypass"].tolist() == [int(w[1] >= 2) for w in want]
    # bucket census of the 1000 triples: 10 unanimous, 270 two-one, 720 all distinct
    assert np.bincount(out["count"]).tolist() == [0, 720, 270, 10]


@pytest.mark.parametrize("E", [1, 2, 3, 4, 5, 6])
def test_all_tables_over_four_labels(E):
    a = np.array(list(product((3, -2, 11, 5), repeat=E)), np.int32)
    out = oracle.gate(a, 0.5)
    want = [_restated(r) for r in a.tolist()]
    assert out["mode"].tolist() == [w[0] for w in want]
    assert out["count"].tolist() == [w[1] for w in want]
    assert out["bypass"].tolist() == [int(Fraction(w[1], E) >= Fraction(1, 2)) for w in want]


# ------------------------------------------------------------------ weighted confidence (G2')
def test_weighted_conf_reductions():
    cfg = wl.C5
    a = wl.answers(cfg, 3, Q=8192)
    w = wl.expert_conf(cfg, 3, Q=8192)
    vote = oracle.gate(a, 0.5)
    # equal weights -> the vote fraction, bit for bit
    eq = oracle.gate(a, 0.5, np.full_like(w, 0.375), 1)
    for k in vote:
        assert np.array_equal(vote[k], eq[k]), k
    # all-zero weights fall back to the vote fraction
    z = oracle.gate(a, 0.5, np.zeros_like(w), 1)
    assert np.array_equal(z["conf"], vote["agree"])
    # mode / count / agree never depend on the weights
    wt = oracle.gate(a, 0.5, w, 1)
    for k in ("mode", "count", "agree"):
        assert np.array_equal(vote[k], wt[k])
    # exact rational restatement: weights are multiples of 2^-24, so Fractions are exact
    for q in range(0, 8192, 97):
        row, ww = a[q].tolist(), [Fraction(float(x)) for x in w[q]]
        m = vote["mode"][q]
        st = sum(ww)
        if st > 0:
            exact = sum(x for x, lab in zip(ww, row) if lab == m) / st
            assert wt["conf"][q] == np.float32(float(exact)) or abs(
                float(wt["conf"][q]) - float(exact)) <= 2 ** -24
            assert wt["bypass"][q] == int(wt["conf"][q] >= np.float32(0.5))
    una = np.repeat(a[:, :1], cfg.E, axis=1)
    assert np.all(oracle.gate(una, 1.0, w, 1)["conf"] == np.float32(1.0))
    dist = np.tile(np.arange(cfg.E, dtype=np.int32)[::-1], (8192, 1))
    d = oracle.gate(dist, 0.5, w, 1)
    want = (w[:, -1].astype(np.float64) / w.astype(np.float64).sum(axis=1)).astype(np.float32)
    ok = w.astype(np.float64).sum(axis=1) > 0
    assert np.array_equal(d["conf"][ok], want[ok])        # mode = label 0 = last column


# ------------------------------------------------------------------ compaction
@pytest.mark.parametrize("cfg_id,seed", [(1, 0), (2, 0), (3, 1), (4, 2)])
def test_compact_is_flatnonzero_and_cumsum(cfg_id, seed):
    cfg = wl.CONFIGS[cfg_id]
    gi = wl.gate_inputs(cfg, seed)
    by = oracle.gate(gi.answers, gi.tau)["bypass"]
    c = oracle.compact(by, gi.ctx_len)
    idx = np.flatnonzero(by == 0)
    assert np.array_equal(c["survivor_idx"], idx.astype(np.int32))
    assert c["n_survivors"] == cfg.Q - int(by.sum())
    assert np.array_equal(c["cu_seqlens"], np.concatenate([[0], np.cumsum(gi.ctx_len[idx], dtype=np.int64)]))
    assert c["total_tokens"] == int(gi.ctx_len[idx].astype(np.int64).sum())
    assert c["max_seqlen"] == (int(gi.ctx_len[idx].max()) if idx.size else 0)
    assert np.all(np.diff(c["survivor_idx"]) > 0)


def test_compact_degenerate_cases():
    ctx = np.arange(1, 11, dtype=np.int32)
    allb = oracle.compact(np.ones(10, np.uint8), ctx)
    assert allb["n_survivors"] == 0 and allb["cu_seqlens"].tolist() == [0]
    assert allb["total_tokens"] == 0 and allb["max_seqlen"] == 0
    none = oracle.compact(np.zeros(10, np.uint8), ctx)
    assert none["survivor_idx"].tolist() == list(range(10))
    assert none["cu_seqlens"].tolist() == np.concatenate([[0], np.cumsum(ctx)]).tolist()
    empty = oracle.compact(np.zeros(0, np.uint8), np.zeros(0, np.int32))
    assert empty["n_survivors"] == 0 and empty["cu_seqlens"].tolist() == [0]
    # int64 token offsets: 3 survivors of 2^30 tokens exceed int32
    big = oracle.compact(np.zeros(3, np.uint8), np.full(3, 1 << 30, np.int32))
    assert big["total_tokens"] == 3 << 30 and big["cu_seqlens"][-1] == 3 << 30


# ------------------------------------------------------------------ closed form: generator + gate
def _p_max_le(m, bins, c):
    """P(no bin holds more than c of m balls thrown uniformly into `bins` bins)
    = m!/bins^m * [x^m] (sum_{i<=c} x^i/i!)^bins, exact rationals."""
    base = [Fraction(1, factorial(i)) for i in range(min(c, m) + 1)]
    poly = [Fraction(1)]
    for _ in range(bins):
        new = [Fraction(0)] * min(m + 1, len(poly) + len(base) - 1)
        for i, x in enumerate(poly):
            for j, y in enumerate(base):
                if i + j <= m:
                    new[i + j] += x * y
        poly = new
    coeff = poly[m] if m < len(poly) else Fraction(0)
    return coeff * factorial(m) / Fraction(bins) ** m


def _bypass_probability(E, p, cmin):
    p = Fraction(p).limit_denominator(1000)
    tot = Fraction(0)
    for K in range(E + 1):
        pk = comb(E, K) * p ** K * (1 - p) ** (E - K)
        tot += pk * (1 if K >= cmin else 1 - _p_max_le(E - K, 9, cmin - 1))
    return tot


@pytest.mark.parametrize("E,tau,cmin,p,printed", [
    (3, 2 / 3, 2, 0.6, 0.699753), (3, 1.0, 3, 0.6, 0.216790), (4, 0.75, 3, 0.6, 0.478255),
    (5, 0.6, 3, 0.6, 0.689944), (8, 0.5, 4, 0.3, 0.211764), (8, 0.5, 4, 0.6, 0.828138),
    (8, 0.75, 6, 0.6, 0.315396), (8, 0.75, 6, 0.9, 0.961908), (8, 0.5, 4, 0.9, 0.999571),
    (8, 0.75, 6, 0.3, 0.011341),
])
def test_bypass_rate_matches_closed_form(E, tau, cmin, p, printed):
    """The seeded generator (consensus label w.p. p, else one of the other nine) and the gate
    together have an exactly computable bypass probability; SURVEY.md 8(d) prints it."""
    exact = float(_bypass_probability(E, p, cmin))
    assert abs(exact - printed) < 1e-6
    cfg = {3: wl.C2, 4: wl.C4, 5: wl.C3, 8: wl.C5}[E]
    Q = 1 << 18
    a = wl.answers(cfg, seed=0, p_agree=p, Q=Q)
    rate = oracle.gate(a, tau)["bypass"].mean()
    sigma = (exact * (1 - exact) / Q) ** 0.5
    assert abs(rate - exact) < 4 * sigma + 1e-9
