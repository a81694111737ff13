"""GPU parity of the SURVEY.md 8(f) N2 entry points built on the prefill kernel: mosaic_lse_merge_n,
mosaic_agg_prefill_attn_chunked and mosaic_agg_prefill_attn_shared_prefix, against the oracle
(north_star's tolerances: max |dO| <= 2e-2, max |dLSE| <= 1e-3)."""
import numpy as np
import pytest
import torch

import _parity as P
import oracle
from paper_2606_03014_b200 import mosaic
from paper_2606_03014_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _cu(lengths):
    return np.concatenate([[0], np.cumsum(np.asarray(lengths, np.int64))]).astype(np.int64)


@pytest.mark.parametrize("n", [1, 2, 3, 7])
def test_merge_n_against_the_oracle(n):
    T, Hq, D = 333, 3, 64
    g = torch.Generator().manual_seed(80 + n)
    op = torch.randn((n, T, Hq, D), generator=g).to(torch.bfloat16)
    lp = torch.randn((n, Hq, T), generator=g) * 3
    lp[0, 0, :7] = float("-inf")
    lp[:, 1, 5:9] = float("-inf")                     # rows without any non-empty partial
    if n > 1:
        lp[1, 2, 100] = float("-inf")
    o, lse = mosaic.lse_merge_n(op.cuda(), lp.cuda())
    torch.cuda.synchronize()
    O_ref, l_ref = oracle.lse_merge_n(op.double().numpy(), lp.double().numpy())
    got, lg = o.float().cpu().numpy(), lse.cpu().numpy()
    assert np.all(np.isfinite(got))
    assert np.abs(got - O_ref).max() <= 2.0 ** -7 * max(1.0, np.abs(O_ref).max())   # one bf16 rounding
    fin = np.isfinite(l_ref)
    assert np.array_equal(np.isneginf(lg), np.isneginf(l_ref))
    assert np.abs(lg[fin] - l_ref[fin]).max() <= 1e-5 * (1 + np.abs(l_ref[fin]).max())
    assert np.all(got[5:9, 1] == 0)


@pytest.mark.parametrize("q_chunk", [1, 100, 128, 256, 500, 4096])
def test_chunked_prefill_is_the_plain_prefill(q_chunk):
    """Ragged lengths around the tile edges, chunk sizes that are and are not multiples of the
    tile, chunks longer than every sequence: every row against the plain-prefill oracle."""
    lengths = [1, 0, 127, 129, 300, 513, 777, 64] if q_chunk > 1 else [3, 0, 70, 129]
    Hq, Hkv, D = 4, 2, 128
    cu = _cu(lengths)
    T = int(cu[-1])
    q, k, v = P.randn_bf16((T, Hq, D), 21), P.randn_bf16((T, Hkv, D), 22), P.randn_bf16((T, Hkv, D), 23)
    scale = 1.0 / np.sqrt(D)
    o, lse = mosaic.agg_prefill_attn_chunked(q.cuda(), k.cuda(), v.cuda(), torch.from_numpy(cu).cuda(),
                                             len(lengths), max(lengths), scale, q_chunk)
    torch.cuda.synchronize()
    eo, el = P.check_attn_full(o, lse, q, k, v, cu, scale)
    assert eo <= P.O_TOL and el <= P.LSE_TOL, (q_chunk, eo, el)


def test_chunked_prefill_of_the_longest_context_configs2_allows():
    """One 45 312-token context (256 + 3 x 4096 + 2 x 16384: the cap of BASELINE configs[2], reading
    G-14) next to a short one, 28 q / 4 kv heads, in chunks of 8192 rows: sampled rows (tile,
    chunk and sequence edges + random) against the O(L^2) oracle."""
    lengths = [45312, 1500]
    Hq, Hkv, D = 28, 4, 128
    cu = _cu(lengths)
    T = int(cu[-1])
    g = torch.Generator(device="cuda").manual_seed(31)
    q = torch.randn((T, Hq, D), device="cuda", generator=g).to(torch.bfloat16)
    k = torch.randn((T, Hkv, D), device="cuda", generator=g).to(torch.bfloat16)
    v = torch.randn((T, Hkv, D), device="cuda", generator=g).to(torch.bfloat16)
    scale = 1.0 / np.sqrt(D)
    o, lse = mosaic.agg_prefill_attn_chunked(q, k, v, torch.from_numpy(cu).cuda(), 2, 45312, scale, 8192)
    torch.cuda.synchronize()
    rs, rh, rp = wl.sample_rows(cu, Hq, Hkv, 0, 33, n_random=96)
    extra = [(0, h, p) for h in (0, 27) for p in (8191, 8192, 8193, 16383, 16384, 40959, 40960, 45311)]
    rs = np.concatenate([rs, np.array([e[0] for e in extra], np.int32)])
    rh = np.concatenate([rh, np.array([e[1] for e in extra], np.int32)])
    rp = np.concatenate([rp, np.array([e[2] for e in extra], np.int64)])
    eo, el = P.check_attn_rows(o, lse, q, k, v, cu, rs, rh, rp, scale)
    assert eo <= P.O_TOL and el <= P.LSE_TOL, (eo, el)
    # and the same rows from the plain prefill, bit for bit where the tiles coincide (8192 = 32 x 256)
    o2, lse2 = P.run_attn(q, k, v, cu, scale)
    assert torch.equal(o, o2) and torch.equal(lse, lse2)


@pytest.mark.parametrize("D,Hq,Hkv", [(128, 4, 2), (64, 4, 1), (128, 7, 7)])
@pytest.mark.parametrize("prefix", [1, 127, 128, 300, 2048])
def test_shared_prefix_against_the_oracle(prefix, D, Hq, Hkv):
    lengths = [1, 130, 0, 64, 257, 500]
    cu = _cu(lengths)
    T = int(cu[-1])
    q, k, v = P.randn_bf16((T, Hq, D), 41), P.randn_bf16((T, Hkv, D), 42), P.randn_bf16((T, Hkv, D), 43)
    kp, vp = P.randn_bf16((prefix, Hkv, D), 44), P.randn_bf16((prefix, Hkv, D), 45)
    scale = 1.0 / np.sqrt(D)
    o, lse = mosaic.agg_prefill_attn_shared_prefix(q.cuda(), kp.cuda(), vp.cuda(), k.cuda(), v.cuda(),
                                                   torch.from_numpy(cu).cuda(), len(lengths),
                                                   max(lengths), scale)
    torch.cuda.synchronize()
    O_ref, l_ref = oracle.attn_shared_prefix(P.bf16_bits(q), P.bf16_bits(kp), P.bf16_bits(vp),
                                             P.bf16_bits(k), P.bf16_bits(v), cu, scale)
    got, lg = o.float().cpu().numpy(), lse.cpu().numpy()
    assert np.all(np.isfinite(got)) and np.all(np.isfinite(lg))
    eo, el = float(np.abs(got - O_ref).max()), float(np.abs(lg - l_ref).max())
    assert eo <= P.O_TOL and el <= P.LSE_TOL, (prefix, eo, el)


def test_shared_prefix_of_length_zero_is_the_plain_prefill():
    lengths, Hq, Hkv, D = [200, 31, 400], 4, 2, 128
    cu = _cu(lengths)
    T = int(cu[-1])
    q, k, v = P.randn_bf16((T, Hq, D), 51), P.randn_bf16((T, Hkv, D), 52), P.randn_bf16((T, Hkv, D), 53)
    scale = 1.0 / np.sqrt(D)
    o, lse = mosaic.agg_prefill_attn_shared_prefix(q.cuda(), None, None, k.cuda(), v.cuda(),
                                                   torch.from_numpy(cu).cuda(), 3, 400, scale)
    o2, lse2 = P.run_attn(q, k, v, cu, scale)
    torch.cuda.synchronize()
    assert torch.equal(o, o2) and torch.equal(lse, lse2)
