#!/usr/bin/env python
"""bench.py -- one JSON line for the confidence-gated aggregator stage (MOSAIC, Alg. 1) on B200.

A "step" is one pass of the whole hot path over one batch of BASELINE.json configs[1] (C2):
mosaic_gate_compact over the Q questions, then mosaic_agg_prefill_attn over the survivors'
packed contexts.  `value` = algorithmic attention FLOPs (4*Hq*D*sum_s L_s(L_s+1)/2, causal pairs
only) of all ranks / the max-over-ranks device time of the timed steps, inputs resident in HBM.
`e2e` = the same through mosaic_stage_host from pinned HOST buffers (H2D + D2H inside the timed
region).  `roofline` is the attention kernel alone (CUDA events around its launches) against the
measured dense-bf16 peak; `gate` is the gate+compaction kernel on configs[4] (2^20 questions,
E = 8, weighted confidences) against the measured HBM copy bandwidth, L2-cold by rotating buffer
sets.  `cpu_baseline` times the fp64 oracle on a bounded row sample of the same workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "gated agg-prefill attn TFLOP/s"
UNIT = "TFLOP/s"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0}


def peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return d, "measured (MEASURED_PEAKS.json)"
    return dict(FALLBACK_PEAKS), "fallback (B200_PROFILING.md)"


def attn_flops(lengths, Hq, D) -> float:
    L = np.asarray(lengths, np.float64)
    return float(4.0 * Hq * D * np.sum(L * (L + 1.0) / 2.0))


def gate_bytes_per_query(E, weighted, survive_frac):
    """Algorithmic bytes of the fused gate+compaction pass (kernel G): answers (+
    weights) + ctx_len read; mode, conf, bypass written; survivor_idx + cu_seqlens per survivor."""
    return 4 * E * (2 if weighted else 1) + 4 + (4 + 4 + 1) + survive_frac * (4 + 8)


def whole_job(secs: float, units: float, world: int, device="cpu"):
    """Whole-job aggregate over the ranks: (max over ranks of the timed seconds, sum over ranks of
    the units processed).  Weak scaling, no data-path collective: every rank works on its own
    batch, these two reductions are the only communication.  Works on any backend (gloo on CPU in
    tests/test_multi_rank.py, nccl in the bench)."""
    if world <= 1:
        return float(secs), float(units)
    import torch
    import torch.distributed as dist
    mx = torch.tensor([secs], dtype=torch.float64, device=device)
    sm = torch.tensor([units], dtype=torch.float64, device=device)
    dist.all_reduce(mx, op=dist.ReduceOp.MAX)
    dist.all_reduce(sm, op=dist.ReduceOp.SUM)
    return float(mx[0]), float(sm[0])


def rank_seed(rank: int) -> int:
    """Seed of the batch rank `rank` generates for itself (weak scaling: one batch per rank)."""
    return int(rank)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [r.split(", ") for r in Path(self.f.name).read_text().splitlines() if r.strip()]
        os.unlink(self.f.name)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.strip().lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(np.max(mx)) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def bf16_bits(t):
    import torch
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)


# ------------------------------------------------------------------------------ reference arm
_ORACLE_INPUTS = {}


def oracle_inputs(cfg, seed):
    """Seeded inputs of the workload as numpy arrays for the oracle (generated once per process)."""
    if (cfg.config_id, seed) not in _ORACLE_INPUTS:
        import oracle
        from paper_2606_03014_b200 import workloads as wl
        gi = wl.gate_inputs(cfg, seed)
        oc = oracle.compact(oracle.gate(gi.answers, gi.tau)["bypass"], gi.ctx_len)
        cu = oc["cu_seqlens"]
        q, k, v = wl.qkv(cfg, seed, int(cu[-1]))
        _ORACLE_INPUTS[(cfg.config_id, seed)] = (gi, cu, bf16_bits(q), bf16_bits(k), bf16_bits(v))
    return _ORACLE_INPUTS[(cfg.config_id, seed)]


def oracle_sample(cfg, seed, budget_rows):
    """A bounded sample of the workload for the CPU oracle: the whole gate + compaction, and
    `budget_rows` random attention rows (plus the tile / sequence edge rows) of the survivors'
    batch.  Returns (flops, seconds, threads, description)."""
    import oracle
    from paper_2606_03014_b200 import workloads as wl

    gi, cu, qb, kb, vb = oracle_inputs(cfg, seed)
    rs, rh, rp = wl.sample_rows(cu, cfg.Hq, cfg.Hkv, seed, cfg.config_id, n_random=budget_rows)
    t0 = time.perf_counter()
    og = oracle.gate(gi.answers, gi.tau)
    oracle.compact(og["bypass"], gi.ctx_len)
    t_gate = time.perf_counter() - t0
    t0 = time.perf_counter()
    oracle.attn_rows(qb, kb, vb, cu, rs, rh, rp, wl.softmax_scale(cfg))
    t_attn = time.perf_counter() - t0
    flops = float(4.0 * cfg.D * np.sum(rp.astype(np.float64) + 1.0))
    desc = (f"oracle gate+compact over all {cfg.Q} questions ({t_gate * 1e3:.2f} ms) + "
            f"{len(rp)} sampled attention rows of {cfg.name} (tile/sequence edges + random), "
            f"{flops / 1e9:.1f} GFLOP in {t_attn:.2f} s")
    return flops, t_gate + t_attn, oracle.num_threads(), desc


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_2606_03014_b200 import workloads as wl
    cfg = wl.C2
    for _ in range(args.warmup):
        oracle_sample(cfg, 0, 64)
    flops = secs = 0.0
    threads, desc = 1, ""
    for _ in range(args.steps):
        f, t, threads, desc = oracle_sample(cfg, 0, args.ref_rows)
        flops += f
        secs += t
    value = flops / secs / 1e12
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": secs / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": cfg.name + " (BASELINE.json configs[1])",
                   "note": "each step = a bounded sample of the workload, see cpu_baseline.sample"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------- product arm
def bench_gate_c5(torch, mosaic, wl, pk, steps, warmup):
    """Gate + compaction on configs[4] (2^20 questions, E = 8, weighted confidences, p = 0.6,
    tau = 0.75), L2-cold: 4 disjoint buffer sets (> 2x the 126 MB L2) used round-robin."""
    cfg = wl.C5
    gi = wl.gate_inputs(cfg, 0)
    nsets = 4
    sets = []
    for _ in range(nsets):
        a = torch.from_numpy(gi.answers).cuda()
        w = torch.from_numpy(gi.expert_conf).cuda()
        cl = torch.from_numpy(gi.ctx_len).cuda()
        out = mosaic.gate_compact(a, cl, gi.tau, w, mosaic.CONF_WEIGHTED)
        sets.append((a, w, cl, out))
    torch.cuda.synchronize()
    S = int(sets[0][3]["n_survivors"])
    bytes_per_call = gate_bytes_per_query(cfg.E, True, S / cfg.Q) * cfg.Q

    def call(i):
        a, w, cl, out = sets[i % nsets]
        mosaic.gate_compact(a, cl, gi.tau, w, mosaic.CONF_WEIGHTED, out=out)

    # The call is ~15 us of GPU work: replay a CUDA graph of one round over the buffer sets so
    # that the measurement is the device's, not the Python launch path's.
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        for i in range(nsets):
            call(i)
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        for i in range(nsets):
            call(i)
    for _ in range(max(1, warmup // nsets)):
        graph.replay()
    rounds = max(1, steps // nsets)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
           for _ in range(rounds)]
    torch.cuda.synchronize()
    for e0, e1 in evs:
        e0.record()
        graph.replay()
        e1.record()
    torch.cuda.synchronize()
    ms = np.array([e0.elapsed_time(e1) for e0, e1 in evs]) / nsets
    t = float(np.mean(ms)) * 1e-3
    gbs = bytes_per_call / t / 1e9
    traffic = None
    tj = ROOT / "profiles" / "traffic.json"
    if tj.exists():
        traffic = json.loads(tj.read_text()).get("gate_compact_dram_bytes_per_launch")
    return {"workload": "C5-large-sweep gate+compaction: Q=2^20, E=8, weighted conf, p=0.6, tau=0.75",
            "call": "mosaic_gate_compact (memset + 1 kernel), CUDA-graph replay of 4 calls", "mqueries_per_s": cfg.Q / t / 1e6,
            "us_per_call": t * 1e6, "us_best": float(ms.min()) * 1e3, "survivors": S,
            "l2": "cold: 4 buffer sets (~93 MB each) used round-robin",
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": pk["hbm_gbs"], "unit": "GB/s",
                         "frac": gbs / pk["hbm_gbs"], "traffic": traffic,
                         "algorithmic_bytes": bytes_per_call}}


def bench_gate_q24(torch, mosaic, pk):
    """Supplementary point: the same fused call at 2^24 questions, where launch, ramp
    and tail stop mattering.  Inputs of the C5 recipe drawn with torch on the device (no parity
    claim is attached to this point; parity at this kernel configuration is tests/test_gpu_gate.py)."""
    Q, E, p_agree, tau = 1 << 24, 8, 0.6, 0.75
    g = torch.Generator(device="cuda").manual_seed(24)
    cons = torch.randint(0, 10, (Q, 1), device="cuda", generator=g, dtype=torch.int32)
    other = torch.randint(0, 9, (Q, E), device="cuda", generator=g, dtype=torch.int32)
    other = other + (other >= cons).to(torch.int32)
    hit = torch.rand((Q, E), device="cuda", generator=g) < p_agree
    a = torch.where(hit, cons.expand(Q, E), other).contiguous()
    w = torch.rand((Q, E), device="cuda", generator=g)
    cl = torch.randint(8192, 32769, (Q,), device="cuda", generator=g, dtype=torch.int32)
    del cons, other, hit
    out = mosaic.gate_compact(a, cl, tau, w, mosaic.CONF_WEIGHTED)
    torch.cuda.synchronize()
    S = int(out["n_survivors"])
    byts = gate_bytes_per_query(E, True, S / Q) * Q
    for _ in range(2):
        mosaic.gate_compact(a, cl, tau, w, mosaic.CONF_WEIGHTED, out=out)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
           for _ in range(5)]
    torch.cuda.synchronize()
    for e0, e1 in evs:   # inputs (1.1 GB) are far larger than L2: every call is cold
        e0.record()
        mosaic.gate_compact(a, cl, tau, w, mosaic.CONF_WEIGHTED, out=out)
        e1.record()
    torch.cuda.synchronize()
    t = float(np.mean([e0.elapsed_time(e1) for e0, e1 in evs])) * 1e-3
    return {"workload": "supplementary: Q=2^24, E=8, weighted conf (torch-drawn inputs, C5 recipe)",
            "us_per_call": t * 1e6, "mqueries_per_s": Q / t / 1e6, "survivors": S,
            "achieved_gbs": byts / t / 1e9, "frac_of_measured_hbm": byts / t / 1e9 / pk["hbm_gbs"]}


def bench_assemble(torch, mosaic, pk, traffic=None):
    """SURVEY 8(f) N1 (a "next" row): mosaic_assemble_context over 2048 survivors of the C5 context
    recipe (U{8192..32768} tokens each, E = 8, prompt 256 + 8 traces at seeded cut points).
    Algorithmic bytes: 4 read + 8 written per token.  Parity: tests/test_gpu_assemble.py."""
    S, E = 2048, 8
    g = np.random.default_rng(31)
    n = g.integers(8192, 32769, size=S).astype(np.int64)
    p_len = np.full(S, 256, np.int64)
    cuts = np.sort((g.random((S, E - 1)) * (n - 256 + 1)[:, None]).astype(np.int64), axis=1)
    edges = np.concatenate([np.zeros((S, 1), np.int64), cuts, (n - 256)[:, None]], axis=1)
    t_len = np.diff(edges, axis=1)
    po = np.concatenate([[0], np.cumsum(p_len)]).astype(np.int64)
    to = np.concatenate([[0], np.cumsum(t_len.reshape(-1))]).astype(np.int64)
    cu = np.concatenate([[0], np.cumsum(n)]).astype(np.int64)
    T = int(cu[-1])
    dev = "cuda"
    gt = torch.Generator(device=dev).manual_seed(31)
    pt = torch.randint(0, 151936, (int(po[-1]),), device=dev, generator=gt, dtype=torch.int32)
    tt = torch.randint(0, 151936, (int(to[-1]),), device=dev, generator=gt, dtype=torch.int32)
    idx = torch.arange(S, device=dev, dtype=torch.int32)
    cu_d, po_d, to_d = (torch.from_numpy(x).to(dev) for x in (cu, po, to))
    ids = torch.empty(T, dtype=torch.int32, device=dev)
    pos = torch.empty(T, dtype=torch.int32, device=dev)
    mm = torch.empty(1, dtype=torch.int32, device=dev)
    call = lambda: mosaic.assemble_context(idx, cu_d, S, int(n.max()), T, pt, po_d, tt, to_d, E,
                                           input_ids=ids, position_ids=pos, n_mismatch=mm)
    for _ in range(2):
        call()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
           for _ in range(5)]
    torch.cuda.synchronize()
    for e0, e1 in evs:   # 0.5 GB per call: every call is L2-cold
        e0.record()
        call()
        e1.record()
    torch.cuda.synchronize()
    assert int(mm.item()) == 0
    t = float(np.mean([e0.elapsed_time(e1) for e0, e1 in evs])) * 1e-3
    byts = 12.0 * T
    return {"workload": "SURVEY 8(f) N1: 2048 contexts of U{8192..32768} tokens, E=8", "tokens": T,
            "us_per_call": t * 1e6, "gtokens_per_s": T / t / 1e9,
            "roofline": {"bound": "hbm", "achieved": byts / t / 1e9, "peak": pk["hbm_gbs"],
                         "unit": "GB/s", "frac": byts / t / 1e9 / pk["hbm_gbs"], "traffic": traffic,
                         "algorithmic_bytes": byts}}


def bench_rope(torch, mosaic, pk, T, Hq, Hkv, D, traffic=None):
    """SURVEY 8(f) N1, second half: mosaic_rope_packed in place on a packed Q / K of the bench
    config's shape (positions 0..L-1 of ~2 k-token sequences).  Algorithmic bytes: every element of
    Q and K read and written once.  Parity: tests/test_gpu_rope.py."""
    dev = "cuda"
    g = torch.Generator(device=dev).manual_seed(41)
    q = torch.randn((T, Hq, D), device=dev, generator=g).to(torch.bfloat16)
    k = torch.randn((T, Hkv, D), device=dev, generator=g).to(torch.bfloat16)
    pos = (torch.arange(T, device=dev, dtype=torch.int32) % 2090).contiguous()
    for _ in range(2):
        mosaic.rope_packed(q, k, pos, 1e6)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
           for _ in range(5)]
    torch.cuda.synchronize()
    for e0, e1 in evs:   # 1.3 GB of Q + K: every call is L2-cold
        e0.record()
        mosaic.rope_packed(q, k, pos, 1e6)
        e1.record()
    torch.cuda.synchronize()
    t = float(np.mean([e0.elapsed_time(e1) for e0, e1 in evs])) * 1e-3
    byts = 4.0 * T * (Hq + Hkv) * D + 4.0 * T
    return {"workload": "SURVEY 8(f) N1: RoPE in place on packed Q/K, T=%d, Hq/Hkv/D=%d/%d/%d" %
                        (T, Hq, Hkv, D),
            "us_per_call": t * 1e6, "gtokens_per_s": T / t / 1e9,
            "roofline": {"bound": "hbm", "achieved": byts / t / 1e9, "peak": pk["hbm_gbs"],
                         "unit": "GB/s", "frac": byts / t / 1e9 / pk["hbm_gbs"], "traffic": traffic,
                         "algorithmic_bytes": byts}}


def bench_attn_kv(torch, mosaic, pk):
    """the last 8192 q rows of two 32768-token contexts against all their keys
    (the last chunk of a chunked prefill), Hq/Hkv/D = 32/8/128.  Algorithmic flops: 4 Hq D per
    visible (row, key) pair.  Parity: tests/test_gpu_attn_kv.py."""
    Lq, Lk, n, Hq, Hkv, D = 8192, 32768, 2, 32, 8, 128
    dev = "cuda"
    g = torch.Generator(device=dev).manual_seed(51)
    q = torch.randn((n * Lq, Hq, D), device=dev, generator=g).to(torch.bfloat16)
    k = torch.randn((n * Lk, Hkv, D), device=dev, generator=g).to(torch.bfloat16)
    v = torch.randn((n * Lk, Hkv, D), device=dev, generator=g).to(torch.bfloat16)
    cq = torch.arange(0, (n + 1) * Lq, Lq, device=dev, dtype=torch.int64)
    ck = torch.arange(0, (n + 1) * Lk, Lk, device=dev, dtype=torch.int64)
    o = torch.empty_like(q)
    lse = torch.empty((Hq, n * Lq), dtype=torch.float32, device=dev)
    ws = torch.empty(mosaic.attn_workspace_bytes(n, n * Lq, Hq, Hkv, D), dtype=torch.uint8, device=dev)
    call = lambda: mosaic.agg_prefill_attn_kv(q, k, v, cq, ck, n, Lq, D ** -0.5, o=o, lse=lse,
                                              workspace=ws)
    for _ in range(2):
        call()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
           for _ in range(3)]
    torch.cuda.synchronize()
    for e0, e1 in evs:
        e0.record()
        call()
        e1.record()
    torch.cuda.synchronize()
    t = float(np.mean([e0.elapsed_time(e1) for e0, e1 in evs])) * 1e-3
    pairs = n * sum(float(Lk - Lq + i + 1) for i in range(Lq))
    fl = 4.0 * Hq * D * pairs
    return {"workload": "SURVEY 8(f) N2: last 8192 rows of 2 x 32768-token contexts, Hq/Hkv/D=32/8/128",
            "ms_per_call": t * 1e3, "tflops": fl / t / 1e12,
            "roofline": {"bound": "tensor", "achieved": fl / t / 1e12, "peak": pk["bf16_tflops"],
                         "unit": "TFLOP/s", "frac": fl / t / 1e12 / pk["bf16_tflops"], "traffic": None}}


def bench_lse_merge(torch, mosaic, pk, T, Hq, D, traffic=None):
    """mosaic_lse_merge on two partial results of the bench config's shape.
    Algorithmic bytes: two bf16 reads and one write per element of O, three fp32 LSE values per row."""
    dev = "cuda"
    g = torch.Generator(device=dev).manual_seed(61)
    oa = torch.randn((T, Hq, D), device=dev, generator=g).to(torch.bfloat16)
    ob = torch.randn((T, Hq, D), device=dev, generator=g).to(torch.bfloat16)
    la = torch.randn((Hq, T), device=dev, generator=g)
    lb = torch.randn((Hq, T), device=dev, generator=g)
    o, lse = torch.empty_like(oa), torch.empty_like(la)
    for _ in range(2):
        mosaic.lse_merge(oa, la, ob, lb, o=o, lse=lse)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
           for _ in range(5)]
    torch.cuda.synchronize()
    for e0, e1 in evs:   # 3.4 GB per call: L2-cold
        e0.record()
        mosaic.lse_merge(oa, la, ob, lb, o=o, lse=lse)
        e1.record()
    torch.cuda.synchronize()
    t = float(np.mean([e0.elapsed_time(e1) for e0, e1 in evs])) * 1e-3
    byts = 6.0 * T * Hq * D + 12.0 * T * Hq
    return {"workload": "SURVEY 8(f) N2: LSE merge of two partials, T=%d, Hq/D=%d/%d" % (T, Hq, D),
            "us_per_call": t * 1e6,
            "roofline": {"bound": "hbm", "achieved": byts / t / 1e9, "peak": pk["hbm_gbs"],
                         "unit": "GB/s", "frac": byts / t / 1e9 / pk["hbm_gbs"], "traffic": traffic,
                         "algorithmic_bytes": byts}}


def bench_decode(torch, mosaic, pk):
    """mosaic_agg_decode_attn, one new token for each of 64 sequences of
    U{8192..32768} cached keys, Hq/Hkv/D = 32/8/128.  Algorithmic bytes: K and V read once."""
    n, Hq, Hkv, D = 64, 32, 8, 128
    g = np.random.default_rng(71)
    Lk = g.integers(8192, 32769, size=n).astype(np.int64)
    ck = np.concatenate([[0], np.cumsum(Lk)]).astype(np.int64)
    Tk = int(ck[-1])
    dev = "cuda"
    gt = torch.Generator(device=dev).manual_seed(71)
    q = torch.randn((n, Hq, D), device=dev, generator=gt).to(torch.bfloat16)
    k = torch.randn((Tk, Hkv, D), device=dev, generator=gt).to(torch.bfloat16)
    v = torch.randn((Tk, Hkv, D), device=dev, generator=gt).to(torch.bfloat16)
    ck_d = torch.from_numpy(ck).to(dev)
    o = torch.empty_like(q)
    lse = torch.empty((Hq, n), dtype=torch.float32, device=dev)
    ws = torch.empty(int(mosaic.load().mosaic_agg_decode_attn_workspace_bytes(n, Tk, Hq, Hkv, D)),
                     dtype=torch.uint8, device=dev)
    call = lambda: mosaic.agg_decode_attn(q, k, v, ck_d, D ** -0.5, o=o, lse=lse, workspace=ws)
    for _ in range(2):
        call()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
           for _ in range(5)]
    torch.cuda.synchronize()
    for e0, e1 in evs:   # K + V = 5 GB: L2-cold
        e0.record()
        call()
        e1.record()
    torch.cuda.synchronize()
    t = float(np.mean([e0.elapsed_time(e1) for e0, e1 in evs])) * 1e-3
    byts = 4.0 * Tk * Hkv * D
    return {"workload": "SURVEY 8(f) N2: decode, 64 sequences of U{8192..32768} keys, Hq/Hkv/D=32/8/128",
            "cached_tokens": Tk, "us_per_call": t * 1e6,
            "roofline": {"bound": "hbm", "achieved": byts / t / 1e9, "peak": pk["hbm_gbs"],
                         "unit": "GB/s", "frac": byts / t / 1e9 / pk["hbm_gbs"], "traffic": None,
                         "algorithmic_bytes": byts}}


def bench_gated_stage(torch, mosaic, wl):
    """what the gate buys on a workload with the paper's statistics (MMLU-Pro bucket
    rates, survivors' traces 2.53 x longer): the aggregator prefill attention over ALL 768 contexts
    against gate + compaction + attention over the survivors of tau = 2/3 (61 GB of Q / K / V / O).  The paper reports 1.74 x
    for its whole aggregator stage on MMLU-Pro with 84.62 % of the calls skipped."""
    Q, Hq, Hkv, D = 768, 28, 4, 128   # 768 questions: the sample's token shares are the population's
    a, ctx, _ = wl.n4_inputs(0, Q)
    dev = "cuda"
    T_all = int(ctx.sum())
    g = torch.Generator(device=dev).manual_seed(81)
    q = torch.randn((T_all, Hq, D), device=dev, generator=g).to(torch.bfloat16)
    k = torch.randn((T_all, Hkv, D), device=dev, generator=g).to(torch.bfloat16)
    v = torch.randn((T_all, Hkv, D), device=dev, generator=g).to(torch.bfloat16)
    o = torch.empty_like(q)
    lse = torch.empty((Hq, T_all), dtype=torch.float32, device=dev)
    ws = torch.empty(mosaic.attn_workspace_bytes(Q, T_all, Hq, Hkv, D), dtype=torch.uint8, device=dev)
    a_d, ctx_d = torch.from_numpy(a).to(dev), torch.from_numpy(ctx).to(dev)
    cu_all = torch.from_numpy(np.concatenate([[0], np.cumsum(ctx.astype(np.int64))])).to(dev)
    scale = D ** -0.5

    def timed(fn, n=3):
        fn()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
               for _ in range(n)]
        torch.cuda.synchronize()
        for e0, e1 in evs:
            e0.record()
            fn()
            e1.record()
        torch.cuda.synchronize()
        return float(np.mean([e0.elapsed_time(e1) for e0, e1 in evs]))

    t_all = timed(lambda: mosaic.agg_prefill_attn(q, k, v, cu_all, Q, int(ctx.max()), scale, o=o,
                                                  lse=lse, workspace=ws))
    out = mosaic.gate_compact(a_d, ctx_d, 2.0 / 3.0)
    torch.cuda.synchronize()
    S, T, mx = int(out["n_survivors"]), int(out["total_tokens"]), int(out["max_seqlen"])

    def gated():   # the survivors' Q / K / V are the first T rows of the same buffers (synthetic)
        mosaic.gate_compact(a_d, ctx_d, 2.0 / 3.0, out=out)
        mosaic.agg_prefill_attn(q[:T], k[:T], v[:T], out["cu_seqlens"], S, mx, scale, o=o[:T],
                                lse=lse.view(-1)[:Hq * T].view(Hq, T), workspace=ws)

    t_gated = timed(gated)
    return {"workload": "SURVEY 8(f) N4: 768 questions, k=3, MMLU-Pro bucket rates, traces 2.53x longer "
                        "for 1:1:1 than 3:0, Hq/Hkv/D=28/4/128",
            "skip_rate": 1.0 - S / Q, "survivor_token_share": T / T_all,
            "survivor_cost_share": float((ctx[out["bypass"].cpu().numpy() == 0].astype(np.float64) ** 2).sum()
                                         / (ctx.astype(np.float64) ** 2).sum()),
            "ms_ungated": t_all, "ms_gated": t_gated, "speedup": t_all / t_gated,
            "paper_aggregator_stage_speedup_mmlu_pro": 1.74}


def run_product(args):
    import torch
    import torch.distributed as dist

    from paper_2606_03014_b200 import mosaic
    from paper_2606_03014_b200 import workloads as wl

    mosaic.load()  # fails loudly when the CUDA library is missing: there is no fallback
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    pk, pk_src = peaks()
    cfg = wl.C2
    seed = rank_seed(rank)  # weak scaling: every rank gates and attends its own batch, no collective
    gi = wl.gate_inputs(cfg, seed)
    a = torch.from_numpy(gi.answers).cuda()
    cl = torch.from_numpy(gi.ctx_len).cuda()
    gout = mosaic.gate_compact(a, cl, gi.tau)
    torch.cuda.synchronize()
    S, T, max_len = int(gout["n_survivors"]), int(gout["total_tokens"]), int(gout["max_seqlen"])
    cu_host = gout["cu_seqlens"][:S + 1].cpu().numpy()
    lengths = np.diff(cu_host)
    flops = attn_flops(lengths, cfg.Hq, cfg.D)
    q, k, v = wl.qkv(cfg, seed, T, device="cuda")
    o = torch.empty_like(q)
    lse = torch.empty((cfg.Hq, T), dtype=torch.float32, device="cuda")
    ws = torch.empty(mosaic.attn_workspace_bytes(S, T, cfg.Hq, cfg.Hkv, cfg.D), dtype=torch.uint8,
                     device="cuda")
    scale = wl.softmax_scale(cfg)
    ev_attn = []

    def step(timed):
        mosaic.gate_compact(a, cl, gi.tau, out=gout)
        if timed:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
        mosaic.agg_prefill_attn(q, k, v, gout["cu_seqlens"], S, max_len, scale, o=o, lse=lse,
                                workspace=ws)
        if timed:
            e1.record()
            ev_attn.append((e0, e1))

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step(False)
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    l0 = mosaic.kernel_launch_count()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    for _ in range(args.steps):
        step(True)
    t1.record()
    barrier()
    launches = mosaic.kernel_launch_count() - l0
    clocks = sampler.stop() if sampler else None
    secs = t0.elapsed_time(t1) * 1e-3
    attn_ms = float(np.mean([e0.elapsed_time(e1) for e0, e1 in ev_attn]))
    secs_max, flops_all = whole_job(secs, flops * args.steps, world, "cuda")
    value = flops_all / secs_max / 1e12

    # ---- end to end through the host-buffer call (pinned host memory, copies timed) ----------
    qh, kh, vh = (t.cpu().pin_memory() for t in (q, k, v))
    ah, clh = torch.from_numpy(gi.answers).pin_memory(), torch.from_numpy(gi.ctx_len).pin_memory()
    del q, k, v, o, lse
    torch.cuda.empty_cache()
    out_h = {"o": torch.empty((T, cfg.Hq, cfg.D), dtype=torch.bfloat16).pin_memory(),
             "lse": torch.empty(cfg.Hq * T, dtype=torch.float32).pin_memory(),
             "mode": torch.empty(cfg.Q, dtype=torch.int32).pin_memory(),
             "conf": torch.empty(cfg.Q, dtype=torch.float32).pin_memory(),
             "bypass": torch.empty(cfg.Q, dtype=torch.uint8).pin_memory()}
    arena = torch.empty(mosaic.stage_host_arena_bytes(cfg.Q, cfg.E, T, cfg.Hq, cfg.Hkv, cfg.D),
                        dtype=torch.uint8, device="cuda")
    e2e_steps = max(3, min(args.steps, 10))
    for _ in range(2):
        mosaic.stage_host(ah, None, clh, gi.tau, 0, qh, kh, vh, scale, out_h=out_h, arena=arena)
    barrier()
    w0 = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(e2e_steps):
        mosaic.stage_host(ah, None, clh, gi.tau, 0, qh, kh, vh, scale, out_h=out_h, arena=arena)
    e1.record()
    barrier()
    e2e_secs = max(e0.elapsed_time(e1) * 1e-3, 0.0)
    e2e_wall = time.perf_counter() - w0
    e2e_max, _ = whole_job(e2e_secs, 0.0, world, "cuda")
    tt = [e2e_max]
    e2e_value = flops_all / args.steps * e2e_steps / float(tt[0]) / 1e12
    h2d = gi.answers.nbytes + gi.ctx_len.nbytes + (qh.numel() + kh.numel() + vh.numel()) * 2
    d2h = (16 + cfg.Q * 9 + S * 4 + (S + 1) * 8 + T * cfg.Hq * cfg.D * 2 + T * cfg.Hq * 4)
    del arena
    torch.cuda.empty_cache()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    gate_info = bench_gate_c5(torch, mosaic, wl, pk, steps=40, warmup=8)
    gate_info["q24"] = bench_gate_q24(torch, mosaic, pk)
    tj0 = ROOT / "profiles" / "traffic.json"
    asm_traffic = (json.loads(tj0.read_text()).get("assemble_dram_bytes_per_launch")
                   if tj0.exists() else None)
    assemble_info = bench_assemble(torch, mosaic, pk, asm_traffic)
    rope_traffic = (json.loads(tj0.read_text()).get("rope_dram_bytes_per_launch")
                    if tj0.exists() else None)
    attn_kv_info = bench_attn_kv(torch, mosaic, pk)
    decode_info = bench_decode(torch, mosaic, pk)
    gated_info = bench_gated_stage(torch, mosaic, wl)
    merge_info = bench_lse_merge(torch, mosaic, pk, T, cfg.Hq, cfg.D,
                                 json.loads(tj0.read_text()).get("lse_merge_dram_bytes_per_launch")
                                 if tj0.exists() else None)
    rope_info = bench_rope(torch, mosaic, pk, T, cfg.Hq, cfg.Hkv, cfg.D, rope_traffic)
    f, t, threads, desc = oracle_sample(cfg, 0, args.cpu_rows)
    attn_tflops = flops / (attn_ms * 1e-3) / 1e12
    traffic = None
    tj = ROOT / "profiles" / "traffic.json"
    if tj.exists():
        traffic = json.loads(tj.read_text()).get("attn_fwd_dram_bytes_per_launch")
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": secs_max / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic",
        "config": {"workload": cfg.name + " (BASELINE.json configs[1])", "Q": cfg.Q, "E": cfg.E,
                   "tau": cfg.tau, "survivors": S, "total_tokens": T, "max_seqlen": max_len,
                   "Hq": cfg.Hq, "Hkv": cfg.Hkv, "D": cfg.D, "per_rank_seed": "rank",
                   "algorithmic_tflop_per_step": flops / 1e12,
                   "l2": "inputs larger than L2 (Q+K+V+O = %.2f GB per step)" %
                         ((2 * T * cfg.Hq + 2 * T * cfg.Hkv) * cfg.D * 2 / 1e9),
                   "peaks": pk_src},
        "roofline": {"bound": "tensor", "achieved": attn_tflops, "peak": pk["bf16_tflops"],
                     "unit": "TFLOP/s", "frac": attn_tflops / pk["bf16_tflops"],
                     "traffic": traffic, "kernel": "attn_fwd (+ schedule_kernel)",
                     "ms_per_launch": attn_ms, "peak_kind": "burst bf16_tflops"},
        "gate": gate_info,
        "assemble": assemble_info,
        "rope": rope_info,
        "attn_kv": attn_kv_info,
        "lse_merge": merge_info,
        "decode": decode_info,
        "gated_stage": gated_info,
        "cpu_baseline": {"value": f / t / 1e12, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "sample": desc},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h), "steps": e2e_steps,
                "ms_per_step": float(tt[0]) / e2e_steps * 1e3,
                "wall_ms_per_step": e2e_wall / e2e_steps * 1e3,
                "call": "mosaic_stage_host (pinned host buffers)"},
        "gpu_launches": int(launches),
        "clocks": clocks,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="mosaic", choices=["mosaic", "reference"])
    ap.add_argument("--ref-rows", type=int, default=4096, help="reference arm: rows per step")
    ap.add_argument("--cpu-rows", type=int, default=524288, help="cpu_baseline: sampled rows")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_product(args)


if __name__ == "__main__":
    main()
