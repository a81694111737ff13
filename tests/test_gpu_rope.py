"""GPU parity of mosaic_rope_packed against the binary64 oracle rounded to bf16.  The kernel takes
angle, sine and cosine in binary64 and the two products in fp32, so it differs from the oracle only
where an fp32 rounding error (2^-24) moves a value across a bf16 rounding boundary: at most one bf16
ulp, on a small fraction of the elements (tolerance derived in DESIGN.md section 3)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_03014_b200 import mosaic
from paper_2606_03014_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _bf16_round(x64):
    return torch.from_numpy(x64).to(torch.float32).to(torch.bfloat16)


def _check(T, Hq, Hkv, D, pos, theta, seed):
    g = torch.Generator().manual_seed(seed)
    q = torch.randn((T, Hq, D), generator=g).to(torch.bfloat16)
    k = torch.randn((T, Hkv, D), generator=g).to(torch.bfloat16)
    want_q = _bf16_round(oracle.rope(q.double().numpy(), pos, theta))
    want_k = _bf16_round(oracle.rope(k.double().numpy(), pos, theta))
    qd, kd = q.cuda(), k.cuda()
    mosaic.rope_packed(qd, kd, torch.from_numpy(np.asarray(pos, np.int32)).cuda(), theta)
    torch.cuda.synchronize()
    for got, want in ((qd.cpu(), want_q), (kd.cpu(), want_k)):
        g32, w32 = got.float(), want.float()
        ulp = torch.maximum(w32.abs(), torch.tensor(2.0 ** -126)) * 2.0 ** -7   # >= 1 bf16 ulp
        assert bool(((g32 - w32).abs() <= ulp).all())
        assert float((got.view(torch.int16) != want.view(torch.int16)).float().mean()) < 2e-3


@pytest.mark.parametrize("D,Hq,Hkv", [(128, 28, 4), (64, 4, 2), (128, 3, 1)])
def test_rope_random_positions(D, Hq, Hkv):
    rng = np.random.default_rng(D + Hq)
    T = 777
    pos = rng.integers(0, 45312, size=T)      # the longest context configs[2] allows
    pos[:3] = [0, 1, 45311]
    _check(T, Hq, Hkv, D, pos, 1e6, seed=1)


def test_rope_on_assembled_positions():
    """End of the N1 row: positions from mosaic_assemble_context on configs[0]."""
    cfg = wl.C1
    gi = wl.gate_inputs(cfg, 0)
    oc = oracle.compact(oracle.gate(gi.answers, gi.tau)["bypass"], gi.ctx_len)
    pt, po, tt, to = wl.context_parts(cfg, 0)
    pos = oracle.assemble_context(oc["survivor_idx"], oc["cu_seqlens"], pt, po, tt, to, cfg.E)[
        "position_ids"]
    _check(oc["total_tokens"], cfg.Hq, cfg.Hkv, cfg.D, pos, 1e4, seed=2)


def test_rope_empty_and_identity():
    q = torch.randn((5, 2, 64)).to(torch.bfloat16).cuda()
    k = torch.randn((5, 1, 64)).to(torch.bfloat16).cuda()
    q0, k0 = q.clone(), k.clone()
    mosaic.rope_packed(q, k, torch.zeros(5, dtype=torch.int32, device="cuda"), 1e6)
    torch.cuda.synchronize()
    assert torch.equal(q, q0) and torch.equal(k, k0)      # position 0: exact identity
    mosaic.rope_packed(q[:0], k[:0], torch.zeros(1, dtype=torch.int32, device="cuda"), 1e6)
