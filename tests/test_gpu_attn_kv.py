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


def test_non_causal_block():
    """causal = 0: every row sees all keys (ragged Lk: the tail of the last 64-key step is masked
    by the key count, not by the row)."""
    Lq, Lk = [1, 130, 64, 300], [1, 77, 640, 1000]
    cq, ck = _cu(Lq), _cu(Lk)
    Hq, Hkv, D = 4, 2, 128
    q = P.randn_bf16((int(cq[-1]), Hq, D), 61)
    k = P.randn_bf16((int(ck[-1]), Hkv, D), 62)
    v = P.randn_bf16((int(ck[-1]), Hkv, D), 63)
    scale = 1.0 / np.sqrt(D)
    o, lse = mosaic.agg_prefill_attn_kv(q.cuda(), k.cuda(), v.cuda(), torch.from_numpy(cq).cuda(),
                                        torch.from_numpy(ck).cuda(), len(Lq), max(Lq), scale,
                                        causal=False)
    torch.cuda.synchronize()
    O_ref, lse_ref = oracle.attn_kv_full(P.bf16_bits(q), P.bf16_bits(k), P.bf16_bits(v), cq, ck, scale,
                                         causal=False)
    assert np.abs(o.float().cpu().numpy() - O_ref).max() <= P.O_TOL
    assert np.abs(lse.cpu().numpy() - lse_ref).max() <= P.LSE_TOL


def test_split_kv_prefill_merged_on_the_gpu():
    """A 1 500-token prefill as two key blocks: rows >= a over keys [0, a) (non-causal call), the
    causal prefill over [a, L), mosaic_lse_merge -- against the plain prefill oracle of the whole."""
    L, a, Hq, Hkv, D = 1500, 640, 4, 2, 128
    q, k, v = P.randn_bf16((L, Hq, D), 71), P.randn_bf16((L, Hkv, D), 72), P.randn_bf16((L, Hkv, D), 73)
    scale = 1.0 / np.sqrt(D)
    O_ref, lse_ref = oracle.attn_full(P.bf16_bits(q), P.bf16_bits(k), P.bf16_bits(v), _cu([L]), scale)
    qd, kd, vd = q.cuda(), k.cuda(), v.cuda()
    n = L - a
    cu_n = torch.tensor([0, n]).cuda()
    o1, l1 = mosaic.agg_prefill_attn_kv(qd[a:].contiguous(), kd[:a].contiguous(), vd[:a].contiguous(),
                                        cu_n, torch.tensor([0, a]).cuda(), 1, n, scale, causal=False)
    o2, l2 = mosaic.agg_prefill_attn(qd[a:].contiguous(), kd[a:].contiguous(), vd[a:].contiguous(),
                                     cu_n, 1, n, scale)
    o, lse = mosaic.lse_merge(o1, l1, o2, l2)
    torch.cuda.synchronize()
    # A merged result carries two bf16 roundings of O (the partials, then the merge) instead of
    # one; it is held to north_star's plain tolerance all the same (measured on a B200: 1.6e-3).
    eo = float(np.abs(o.float().cpu().numpy() - O_ref[a:]).max())
    el = float(np.abs(lse.cpu().numpy() - lse_ref[:, a:]).max())
    print(f"split-KV merge: max|dO|={eo:.3e} max|dLSE|={el:.2e} (tolerances {P.O_TOL:.0e} / {P.LSE_TOL:.0e})")
    assert eo <= P.O_TOL and el <= P.LSE_TOL, (eo, el)


def test_merge_against_the_oracle_and_empty_partials():
    T, Hq, D = 333, 3, 64
    g = torch.Generator().manual_seed(81)
    oa = torch.randn((T, Hq, D), generator=g).to(torch.bfloat16)
    ob = torch.randn((T, Hq, D), generator=g).to(torch.bfloat16)
    la = torch.randn((Hq, T), generator=g) * 3
    lb = torch.randn((Hq, T), generator=g) * 3
    la[0, :7] = float("-inf")
    lb[1, 5:9] = float("-inf")
    la[2, 100], lb[2, 100] = float("-inf"), float("-inf")
    o, lse = mosaic.lse_merge(oa.cuda(), la.cuda(), ob.cuda(), lb.cuda())
    torch.cuda.synchronize()
    O_ref, l_ref = oracle.lse_merge(oa.double().numpy(), la.double().numpy(), ob.double().numpy(),
                                    lb.double().numpy())
    got = o.float().cpu().numpy()
    assert np.all(np.isfinite(got))
    assert np.abs(got - O_ref).max() <= 2.0 ** -7 * max(1.0, np.abs(O_ref).max())   # one bf16 rounding
    lg = lse.cpu().numpy()
    fin = np.isfinite(l_ref)
    assert np.array_equal(np.isneginf(lg), np.isneginf(l_ref))
    assert np.abs(lg[fin] - l_ref[fin]).max() <= 1e-5 * (1 + np.abs(l_ref[fin]).max())


@pytest.mark.parametrize("seed", [0, 1, 2, 3, 4, 5])
def test_random_shapes(seed):
    """Seeded random batches: q lengths 0..400, 0..900 more keys than q rows, both head sizes, three
    group sizes, causal and not -- every row against the oracle."""
    g = np.random.default_rng(900 + seed)
    Hq, Hkv = [(4, 2), (6, 1), (8, 8)][seed % 3]
    D = (128, 64)[seed % 2]
    causal = seed % 4 != 3
    n = 14
    Lq = g.integers(0, 401, size=n)
    Lq[g.integers(0, n)] = 0                                   # an empty q sequence somewhere
    Lk = Lq + g.integers(0, 901, size=n) * (g.random(n) < 0.7)  # 30 % plain sequences
    Lk = np.maximum(Lk, 1)                                      # (a q row needs a key)
    cq, ck = _cu(Lq), _cu(Lk)
    q = P.randn_bf16((int(cq[-1]), Hq, D), 7 * seed)
    k = P.randn_bf16((int(ck[-1]), Hkv, D), 7 * seed + 1, 1.5)
    v = P.randn_bf16((int(ck[-1]), Hkv, D), 7 * seed + 2)
    scale = 1.0 / np.sqrt(D)
    o, lse = mosaic.agg_prefill_attn_kv(q.cuda(), k.cuda(), v.cuda(), torch.from_numpy(cq).cuda(),
                                        torch.from_numpy(ck).cuda(), n, int(Lq.max()), scale,
                                        causal=causal)
    torch.cuda.synchronize()
    O_ref, lse_ref = oracle.attn_kv_full(P.bf16_bits(q), P.bf16_bits(k), P.bf16_bits(v), cq, ck, scale,
                                         causal=causal)
    assert np.all(np.isfinite(lse.cpu().numpy()))
    eo = float(np.abs(o.float().cpu().numpy() - O_ref).max())
    el = float(np.abs(lse.cpu().numpy() - lse_ref).max())
    assert eo <= P.O_TOL and el <= P.LSE_TOL, (seed, eo, el)
