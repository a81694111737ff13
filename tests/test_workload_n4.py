"""the generator reproduces the statistics the paper prints (Table 1 skip rates
P:L205-213; trace lengths by agreement bucket P:L237-243), measured with the oracle's gate."""
import numpy as np
from scipy.stats import spearmanr

import oracle
from paper_2606_03014_b200 import workloads as wl


def test_n4_matches_the_papers_statistics():
    Q = 60000
    a, ctx, t_len = wl.n4_inputs(0, Q)
    g1, g2 = oracle.gate(a, 1.0), oracle.gate(a, 2.0 / 3.0)
    assert abs(g1["bypass"].mean() - 0.4571) < 0.01          # tau = 1 skips the 3:0 bucket
    assert abs(g2["bypass"].mean() - 0.8462) < 0.01          # tau = 2/3 skips 3:0 and 2:1
    c = g1["count"]
    assert set(np.unique(c)) == {1, 2, 3}
    ratio = t_len[c == 1].mean() / t_len[c == 3].mean()
    assert abs(ratio - 2.53) < 0.15                           # the cap trims the 1:1:1 tail a little
    rho = spearmanr(np.repeat(c, 3), t_len.reshape(-1)).correlation
    assert -0.32 < rho < -0.22
    assert np.array_equal(ctx, 256 + t_len.sum(axis=1))
    # the survivors of the aggressive gate hold far more than 15 % of the tokens
    assert ctx[g2["bypass"] == 0].sum() / ctx.sum() > 0.22
