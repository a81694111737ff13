"""GPU parity of mosaic_agg_decode_attn against oracle.attn_kv_full with one q
row per sequence (a row that sees every key: the pinned Lq = 1 case of the oracle)."""
import numpy as np
import pytest
import torch

import _parity as P
import oracle
from paper_2606_03014_b200 import mosaic

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("D,Hq,Hkv", [(128, 28, 4), (128, 32, 8), (64, 4, 4), (128, 8, 1), (64, 6, 2)])
def test_decode_matches_oracle(D, Hq, Hkv):
    Lk = [1, 63, 64, 65, 127, 128, 129, 700, 2049, 5]
    ck = np.concatenate([[0], np.cumsum(Lk)]).astype(np.int64)
    n, Tk = len(Lk), int(ck[-1])
    q = P.randn_bf16((n, Hq, D), 91)
    k = P.randn_bf16((Tk, Hkv, D), 92)
    v = P.randn_bf16((Tk, Hkv, D), 93)
    scale = 1.0 / np.sqrt(D)
    o, lse = mosaic.agg_decode_attn(q.cuda(), k.cuda(), v.cuda(), torch.from_numpy(ck).cuda(), scale)
    torch.cuda.synchronize()
    cq = np.arange(n + 1, dtype=np.int64)
    O_ref, lse_ref = oracle.attn_kv_full(P.bf16_bits(q), P.bf16_bits(k), P.bf16_bits(v), cq, ck, scale)
    assert np.abs(o.float().cpu().numpy() - O_ref).max() <= P.O_TOL
    assert np.abs(lse.cpu().numpy() - lse_ref).max() <= P.LSE_TOL


def test_decode_few_long_sequences_and_no_keys():
    """Two long sequences (many chunks each: the split-KV merge) and one without keys (O = 0,
    LSE = -inf)."""
    Lk = [9000, 0, 20001]
    ck = np.concatenate([[0], np.cumsum(Lk)]).astype(np.int64)
    Hq, Hkv, D = 8, 2, 128
    q = P.randn_bf16((3, Hq, D), 94)
    k = P.randn_bf16((int(ck[-1]), Hkv, D), 95)
    v = P.randn_bf16((int(ck[-1]), Hkv, D), 96)
    scale = 1.0 / np.sqrt(D)
    o, lse = mosaic.agg_decode_attn(q.cuda(), k.cuda(), v.cuda(), torch.from_numpy(ck).cuda(), scale)
    torch.cuda.synchronize()
    keep = [0, 2]
    ck2 = np.concatenate([[0], np.cumsum([Lk[i] for i in keep])]).astype(np.int64)
    O_ref, lse_ref = oracle.attn_kv_full(P.bf16_bits(q[keep]), P.bf16_bits(k), P.bf16_bits(v),
                                         np.arange(3, dtype=np.int64), ck2, scale)
    og, lg = o.float().cpu().numpy(), lse.cpu().numpy()
    assert np.abs(og[keep] - O_ref).max() <= P.O_TOL
    assert np.abs(lg[:, keep] - lse_ref).max() <= P.LSE_TOL
    assert np.all(og[1] == 0) and np.all(np.isneginf(lg[:, 1]))


def test_decode_empty_batch():
    q = torch.empty((0, 4, 64), dtype=torch.bfloat16, device="cuda")
    k = torch.zeros((8, 2, 64), dtype=torch.bfloat16, device="cuda")
    o, lse = mosaic.agg_decode_attn(q, k, k, torch.zeros(1, dtype=torch.int64, device="cuda"), 0.1)
    assert o.shape == (0, 4, 64) and lse.shape == (4, 0)


def test_decode_keyless_sequence_first_and_more_units_than_ctas():
    """A sequence without keys FIRST in a batch with several times more (chunk, kv head) units than
    the GPU has SMs: the CTA that draws the keyless unit (which visits no KV tile at all) goes on
    to other units afterwards, so every warp role must skip it consistently (a producer that loaded
    Q / K / V for it would leave the K/V ring one item out of step with the consumers)."""
    n_sms = torch.cuda.get_device_properties(0).multi_processor_count
    Hq, Hkv, D = 8, 4, 64
    n = 3 * n_sms // Hkv + 7          # > 2 units per SM (one chunk per sequence at these lengths)
    g = np.random.default_rng(97)
    Lk = g.integers(1, 400, size=n).astype(np.int64)
    Lk[0] = 0
    Lk[n // 2] = 0
    ck = np.concatenate([[0], np.cumsum(Lk)]).astype(np.int64)
    q = P.randn_bf16((n, Hq, D), 98)
    k = P.randn_bf16((int(ck[-1]), Hkv, D), 99)
    v = P.randn_bf16((int(ck[-1]), Hkv, D), 100)
    scale = 1.0 / np.sqrt(D)
    for _ in range(3):                # the hand-out is dynamic: a few draws of who gets the unit
        o, lse = mosaic.agg_decode_attn(q.cuda(), k.cuda(), v.cuda(), torch.from_numpy(ck).cuda(), scale)
        torch.cuda.synchronize()
        keep = np.flatnonzero(Lk > 0)
        ck2 = np.concatenate([[0], np.cumsum(Lk[keep])]).astype(np.int64)
        O_ref, lse_ref = oracle.attn_kv_full(P.bf16_bits(q[keep]), P.bf16_bits(k), P.bf16_bits(v),
                                             np.arange(len(keep) + 1, dtype=np.int64), ck2, scale)
        og, lg = o.float().cpu().numpy(), lse.cpu().numpy()
        assert np.abs(og[keep] - O_ref).max() <= P.O_TOL
        assert np.abs(lg[:, keep] - lse_ref).max() <= P.LSE_TOL
        for s in (0, n // 2):
            assert np.all(og[s] == 0) and np.all(np.isneginf(lg[:, s]))
