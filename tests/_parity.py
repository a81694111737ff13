"""Helpers shared by the GPU parity tests: run the CUDA path through the binding and the oracle on
the same seeded inputs.  (Test infrastructure; imports both sides, shares arithmetic with neither.)"""
import numpy as np
import torch

import oracle
from paper_2606_03014_b200 import mosaic
from paper_2606_03014_b200 import workloads as wl

O_TOL = 2e-2      # BASELINE.json north_star: max abs error on O
LSE_TOL = 1e-3    # ... and on logsumexp


def bf16_bits(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)


def gpu_gate_compact_all(gi: wl.GateInputs, conf_mode: int):
    """Runs mosaic_gate + mosaic_compact and mosaic_gate_compact; returns both as numpy dicts."""
    dev = "cuda"
    a = torch.from_numpy(gi.answers).to(dev)
    w = torch.from_numpy(gi.expert_conf).to(dev) if conf_mode == 1 else None
    cl = torch.from_numpy(gi.ctx_len).to(dev)
    g = mosaic.gate(a, gi.tau, w, conf_mode)
    c = mosaic.compact(g["bypass"], cl)
    f = mosaic.gate_compact(a, cl, gi.tau, w, conf_mode, want_count=True, want_agree=True)
    torch.cuda.synchronize()

    def pack(gd, cd):
        S = int(cd["n_survivors"].item())
        return dict(mode=gd["mode"].cpu().numpy(), count=gd["count"].cpu().numpy(),
                    agree=gd["agree"].cpu().numpy(), conf=gd["conf"].cpu().numpy(),
                    bypass=gd["bypass"].cpu().numpy(),
                    survivor_idx=cd["survivor_idx"][:S].cpu().numpy(),
                    cu_seqlens=cd["cu_seqlens"][:S + 1].cpu().numpy(), n_survivors=S,
                    total_tokens=int(cd["total_tokens"].item()),
                    max_seqlen=int(cd["max_seqlen"].item()))
    return pack(g, c), pack(f, f)


def oracle_gate_compact(gi: wl.GateInputs, conf_mode: int):
    og = oracle.gate(gi.answers, gi.tau, gi.expert_conf, conf_mode)
    oc = oracle.compact(og["bypass"], gi.ctx_len)
    return {**og, **oc}


def assert_gate_equal(got: dict, want: dict):
    """Bit-exact on every output (floats compared as bit patterns)."""
    for k in ("mode", "count", "bypass", "survivor_idx", "cu_seqlens"):
        assert got[k].dtype == want[k].dtype, k
        assert np.array_equal(got[k], want[k]), k
    for k in ("agree", "conf"):
        assert np.array_equal(got[k].view(np.uint32), want[k].view(np.uint32)), k
    for k in ("n_survivors", "total_tokens", "max_seqlen"):
        assert got[k] == want[k], (k, got[k], want[k])


def run_attn(q, k, v, cu_seqlens, scale):
    """q,k,v torch bf16 (any device), cu_seqlens numpy int64.  Returns (o, lse) torch on the GPU."""
    cu = torch.from_numpy(np.asarray(cu_seqlens, np.int64)).cuda()
    L = np.diff(cu_seqlens)
    o, lse = mosaic.agg_prefill_attn(q.cuda(), k.cuda(), v.cuda(), cu, len(L),
                                     int(L.max()) if len(L) else 0, scale)
    torch.cuda.synchronize()
    return o, lse


def check_attn_rows(o, lse, q, k, v, cu_seqlens, rs, rh, rp, scale):
    """Compares the sampled rows with the O(L^2) oracle; returns (max |dO|, max |dLSE|)."""
    qb, kb, vb = bf16_bits(q), bf16_bits(k), bf16_bits(v)
    O_ref, lse_ref, _ = oracle.attn_rows(qb, kb, vb, cu_seqlens, rs, rh, rp, scale)
    t = torch.from_numpy(np.asarray(cu_seqlens)[rs] + rp).to(o.device)
    hh = torch.from_numpy(rh.astype(np.int64)).to(o.device)
    o_got = o[t, hh].float().cpu().numpy().astype(np.float64)
    lse_got = lse[hh, t].cpu().numpy().astype(np.float64)
    assert np.all(np.isfinite(o_got)) and np.all(np.isfinite(lse_got))
    return float(np.abs(o_got - O_ref).max()), float(np.abs(lse_got - lse_ref).max())


def check_attn_full(o, lse, q, k, v, cu_seqlens, scale):
    qb, kb, vb = bf16_bits(q), bf16_bits(k), bf16_bits(v)
    O_ref, lse_ref = oracle.attn_full(qb, kb, vb, cu_seqlens, scale)
    o_got = o.float().cpu().numpy().astype(np.float64)
    lse_got = lse.cpu().numpy().astype(np.float64)
    assert np.all(np.isfinite(o_got)) and np.all(np.isfinite(lse_got))
    return float(np.abs(o_got - O_ref).max()), float(np.abs(lse_got - lse_ref).max())


def randn_bf16(shape, seed, scale=1.0):
    g = torch.Generator().manual_seed(seed)
    return (torch.randn(shape, generator=g, dtype=torch.float32) * scale).to(torch.bfloat16)
