"""GPU parity of mosaic_agg_prefill_attn_kv (q rows = the last Lq positions of
Lk keys) against oracle.attn_kv_full, every row, same tolerances as the plain prefill."""
import numpy as np
import pytest
import torch

import _parity as P
import oracle
from paper_2606_03014_b200 import mosaic

pytestmark = pytest.mark.gpu


def _cu(lengths):
    return np.concatenate([[0], np.cumsum(np.asarray(lengths, np.int64))]).astype(np.int64)


def _case(Lq, Lk, Hq, Hkv, D, seed, k_scale=1.0):
    cq, ck = _cu(Lq), _cu(Lk)
    Tq, Tk = int(cq[-1]), int(ck[-1])
    q = P.randn_bf16((Tq, Hq, D), seed)
    k = P.randn_bf16((Tk, Hkv, D), seed + 1, k_scale)
    v = P.randn_bf16((Tk, Hkv, D), seed + 2)
    scale = 1.0 / np.sqrt(D)
    o, lse = mosaic.agg_prefill_attn_kv(q.cuda(), k.cuda(), v.cuda(), torch.from_numpy(cq).cuda(),
                                        torch.from_numpy(ck).cuda(), len(Lq), int(max(Lq)), scale)
    torch.cuda.synchronize()
    O_ref, lse_ref = oracle.attn_kv_full(P.bf16_bits(q), P.bf16_bits(k), P.bf16_bits(v), cq, ck, scale)
    o_got = o.float().cpu().numpy().astype(np.float64)
    lse_got = lse.cpu().numpy().astype(np.float64)
    assert np.all(np.isfinite(o_got)) and np.all(np.isfinite(lse_got))
    return float(np.abs(o_got - O_ref).max()), float(np.abs(lse_got - lse_ref).max())


@pytest.mark.parametrize("D,Hq,Hkv", [(128, 4, 2), (64, 4, 1), (128, 7, 7)])
def test_offsets_around_every_edge(D, Hq, Hkv):
    """Offsets Lk - Lq that are 0, 1, 63, 64, 65, 127, 128, 129, ... (the diagonal then crosses the
    64-key steps and the 128-key tiles anywhere), decode-like Lq = 1, empty q sequences, q blocks
    of one and of two tiles, plain sequences in between."""
    Lq = [1, 37, 128, 129, 256, 300, 0, 64, 1, 200, 513, 77]
    off = [0, 1, 63, 64, 65, 127, 5, 128, 700, 129, 191, 1000]
    Lk = [a + b for a, b in zip(Lq, off)]
    eo, el = _case(Lq, Lk, Hq, Hkv, D, seed=31)
    assert eo <= P.O_TOL and el <= P.LSE_TOL, (eo, el)


def test_chunked_prefill_of_one_long_sequence():
    """A 2 100-token context prefilled in chunks of 500 q rows against the growing K / V: every
    chunk is one call; together they must reproduce the plain prefill of the whole sequence."""
    L, Hq, Hkv, D = 2100, 4, 2, 128
    q, k, v = P.randn_bf16((L, Hq, D), 41), P.randn_bf16((L, Hkv, D), 42), P.randn_bf16((L, Hkv, D), 43)
    scale = 1.0 / np.sqrt(D)
    O_ref, lse_ref = oracle.attn_full(P.bf16_bits(q), P.bf16_bits(k), P.bf16_bits(v), _cu([L]), scale)
    qd, kd, vd = q.cuda(), k.cuda(), v.cuda()
    for a in range(0, L, 500):
        b = min(L, a + 500)
        o, lse = mosaic.agg_prefill_attn_kv(qd[a:b].contiguous(), kd[:b].contiguous(),
                                            vd[:b].contiguous(), torch.tensor([0, b - a]).cuda(),
                                            torch.tensor([0, b]).cuda(), 1, b - a, scale)
        torch.cuda.synchronize()
        assert np.abs(o.float().cpu().numpy() - O_ref[a:b]).max() <= P.O_TOL
        assert np.abs(lse.cpu().numpy() - lse_ref[:, a:b]).max() <= P.LSE_TOL


def test_sharp_scores_with_offsets():
    eo, el = _case([100, 257], [1124, 300], 2, 1, 128, seed=51, k_scale=8.0)
    assert eo <= P.O_TOL and el <= P.LSE_TOL, (eo, el)
