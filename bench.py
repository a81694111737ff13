#!/usr/bin/env python
"""bench.py -- one JSON line for the confidence-gated aggregator stage (MOSAIC, Alg. 1) on B200.

A "step" is one pass of the whole hot path over one batch of BASELINE.json configs[4] (C5, the
largest single-GPU configuration): mosaic_gate_compact over the 2^20 questions (E = 8, weighted
confidences), then mosaic_agg_prefill_attn over the packed contexts of the first 16 survivors
(64 q / 8 kv heads, head_dim 128, 8-32 k tokens each).  `value` = algorithmic attention FLOPs
(4*Hq*D*sum_s L_s(L_s+1)/2, causal pairs only) of all ranks / the max-over-ranks device time of
the timed steps, inputs resident in HBM.  `e2e` = the same through mosaic_stage_host from pinned
HOST buffers (H2D + D2H inside the timed region).  `roofline` is the attention kernel alone (CUDA
events around its launches) against the measured dense-bf16 peak (the sustained figure: the timed
region is seconds long; `frac_burst` is the same against the burst figure).  `gate` is the
gate+compaction call on the same 2^20 questions against the measured HBM copy bandwidth, L2-cold
by rotating buffer sets.  `per_config` times the attention of configs[1..4] (C2..C5) alone.
`next` holds the SURVEY 8(f) legs (shapes in DESIGN.md section 7; `gbs` legs are HBM-bound, against
the measured copy bandwidth, `tflops` legs tensor-bound).  `cpu_baseline` times the fp64
oracle on a bounded row sample of the same workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--legs a,b,...]
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
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}
TRAFFIC_SOURCE = "profiles/traffic.json (ncu, static)"
ALL_LEGS = ("gate", "q24", "lse_merge", "lse_merge_n", "rope", "assemble", "decode", "attn_kv",
            "prefix", "chunked", "per_config", "gated_stage", "e2e", "cpu")


def peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        d.setdefault("bf16_tflops_sustained", d["bf16_tflops"])
        return d, "MEASURED_PEAKS.json"
    return dict(FALLBACK_PEAKS), "fallback (B200_PROFILING.md)"


def static_traffic(key):
    tj = ROOT / "profiles" / "traffic.json"
    return json.loads(tj.read_text()).get(key) if tj.exists() else None


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


def spawn_ranks(n: int, target, args=(), port: int = 0):
    """`--gpus N` without a launcher (no WORLD_SIZE in the environment): start the N ranks here,
    one process per GPU, with the environment torchrun would have set.  Returns when all ranks have
    exited; raises if any rank failed (a box with fewer than N GPUs fails in the rank that cannot
    select its device -- loudly, never as a silent N = 1 run)."""
    import torch.multiprocessing as mp
    if not port:
        import socket
        with socket.socket() as s:
            s.bind(("127.0.0.1", 0))
            port = s.getsockname()[1]
    mp.spawn(_rank_main, args=(n, port, target, args), nprocs=n, join=True)


def _rank_main(rank, n, port, target, args):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(n),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    target(*args)


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


def r3(x):
    """Three significant decimals are plenty for a report line (keeps the JSON line short)."""
    return None if x is None else float(f"{x:.4g}")


# ------------------------------------------------------------------------------ reference arm
_ORACLE_INPUTS = {}


def oracle_inputs(cfg, seed, n_random):
    """Seeded inputs of the workload for the oracle, as numpy arrays (once per process): the gate
    inputs in full, K and V of the attended sequences in full, and Q ONLY at the sampled rows --
    the [T, Hq, D] array is calloc'ed and untouched pages are never committed, so the 5.8 GB of
    configs[4]'s Q costs what the sampled rows cost.  Timing inputs only (no parity claim)."""
    key = (cfg.config_id, seed, n_random)
    if key not in _ORACLE_INPUTS:
        import torch

        import oracle
        from paper_2606_03014_b200 import workloads as wl
        gi = wl.gate_inputs(cfg, seed)
        w = gi.expert_conf if cfg.has_conf else None
        oc = oracle.compact(oracle.gate(gi.answers, gi.tau, w, 1 if cfg.has_conf else 0)["bypass"],
                            gi.ctx_len)
        n = oc["n_survivors"] if cfg.max_attn_seqs is None else min(cfg.max_attn_seqs,
                                                                    oc["n_survivors"])
        cu = oc["cu_seqlens"][:n + 1]
        T = int(cu[-1])
        rs, rh, rp = wl.sample_rows(cu, cfg.Hq, cfg.Hkv, seed, cfg.config_id, n_random=n_random)
        g = torch.Generator().manual_seed(1000 + seed)
        bits = lambda t: t.contiguous().view(torch.int16).numpy().view(np.uint16)
        kb = bits((torch.randn((T, cfg.Hkv, cfg.D), generator=g) * cfg.k_scale).to(torch.bfloat16))
        vb = bits(torch.randn((T, cfg.Hkv, cfg.D), generator=g).to(torch.bfloat16))
        qb = np.zeros((T, cfg.Hq, cfg.D), np.uint16)
        qrows = bits(torch.randn((len(rp), cfg.D), generator=g).to(torch.bfloat16))
        qb[cu[rs] + rp, rh] = qrows
        _ORACLE_INPUTS[key] = (gi, w, cu, qb, kb, vb, rs, rh, rp)
    return _ORACLE_INPUTS[key]


def oracle_sample(cfg, seed, budget_rows):
    """A bounded sample of the workload for the CPU oracle: the whole gate + compaction, and
    `budget_rows` random attention rows (plus the tile / sequence edge rows) of the attended
    sequences.  Returns (flops, seconds, threads, description)."""
    import oracle
    from paper_2606_03014_b200 import workloads as wl

    gi, w, cu, qb, kb, vb, rs, rh, rp = oracle_inputs(cfg, seed, budget_rows)
    t0 = time.perf_counter()
    og = oracle.gate(gi.answers, gi.tau, w, 1 if w is not None else 0)
    oracle.compact(og["bypass"], gi.ctx_len)
    t_gate = time.perf_counter() - t0
    t0 = time.perf_counter()
    oracle.attn_rows(qb, kb, vb, cu, rs, rh, rp, wl.softmax_scale(cfg))
    t_attn = time.perf_counter() - t0
    flops = float(4.0 * cfg.D * np.sum(rp.astype(np.float64) + 1.0))
    desc = (f"oracle gate+compact over all {cfg.Q} questions ({t_gate * 1e3:.0f} ms) + "
            f"{len(rp)} sampled attention rows of {cfg.name} ({flops / 1e9:.1f} GFLOP, {t_attn:.2f} s)")
    return flops, t_gate + t_attn, oracle.num_threads(), desc


def workload_name(cfg):
    return (f"{cfg.name} (configs[{cfg.config_id - 1}]): gate+compaction of 2^20 questions "
            f"(E=8, weighted) + attention of the first {cfg.max_attn_seqs} survivors "
            f"({cfg.Hq}/{cfg.Hkv}/{cfg.D}, 8-32 k tokens)")


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_2606_03014_b200 import workloads as wl
    cfg = wl.C5
    for _ in range(args.warmup):
        oracle_sample(cfg, 0, args.ref_rows)
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
        "config": {"workload": workload_name(cfg),
                   "note": "each step = a bounded sample of the workload, see cpu_baseline.sample"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------- product arm
def timed(torch, fn, n, warm=2):
    """ms of n launches of fn, CUDA events on the current stream, after `warm` untimed ones."""
    for _ in range(warm):
        fn()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
           for _ in range(n)]
    torch.cuda.synchronize()
    for e0, e1 in evs:
        e0.record()
        fn()
        e1.record()
    torch.cuda.synchronize()
    return np.array([e0.elapsed_time(e1) for e0, e1 in evs])


def hbm_leg(ms, byts, pk, traffic=None):
    t = float(np.median(ms)) * 1e-3
    leg = {"us": r3(t * 1e6), "us_best": r3(float(ms.min()) * 1e3), "gbs": r3(byts / t / 1e9),
           "frac": r3(byts / t / 1e9 / pk["hbm_gbs"]), "bytes": int(byts)}
    if traffic is not None:
        leg["traffic"] = traffic
    return leg


def tensor_leg(ms, fl, pk):
    """A leg whose timed launches add up to more than 0.3 s runs under the power cap and is held
    against the sustained bf16 peak; a shorter one (timed after an idle second) against the burst
    peak -- MEASURED_PEAKS.json's two figures, B200_PROFILING.md."""
    t = float(np.median(ms)) * 1e-3
    kind = "sustained" if float(ms.sum()) > 300.0 else "burst"
    peak = pk["bf16_tflops_sustained"] if kind == "sustained" else pk["bf16_tflops"]
    return {"ms": r3(t * 1e3), "ms_best": r3(float(ms.min())), "tflop": r3(fl / 1e12),
            "tflops": r3(fl / t / 1e12), "frac": r3(fl / t / 1e12 / peak), "peak_kind": kind}


def bench_gate_c5(torch, mosaic, wl, pk, gi, steps=80, warmup=8):
    """Gate + compaction on configs[4] (2^20 questions, E = 8, weighted confidences, p = 0.6,
    tau = 0.75), L2-cold: 4 disjoint buffer sets (> 2x the 126 MB L2) used round-robin, one CUDA
    graph replay = one round over the sets, so that the time is the device's and not Python's."""
    cfg = wl.C5
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
    byts = gate_bytes_per_query(cfg.E, True, S / cfg.Q) * cfg.Q

    def call(i):
        a, w, cl, out = sets[i % nsets]
        mosaic.gate_compact(a, cl, gi.tau, w, mosaic.CONF_WEIGHTED, out=out)

    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        for i in range(nsets):
            call(i)
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    l0 = mosaic.kernel_launch_count()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        for i in range(nsets):
            call(i)
    launches_per_call = (mosaic.kernel_launch_count() - l0) // nsets
    ms = timed(torch, graph.replay, max(3, steps // nsets), max(1, warmup // nsets)) / nsets
    t = float(np.median(ms)) * 1e-3
    gbs = byts / t / 1e9
    # Context for a 90 MB call (Kernel G): the simplest kernel there is -- torch's
    # elementwise fp32 copy -- moving the same number of bytes in the same harness.  Not ours, not
    # counted in gpu_launches; it says what fraction of the copy bandwidth ANY kernel reaches here.
    n = int(byts) // 8 // 1024 * 1024
    cp = [(torch.empty(n, dtype=torch.float32, device="cuda").normal_(),
           torch.empty(n, dtype=torch.float32, device="cuda")) for _ in range(nsets)]
    with torch.cuda.stream(side):
        for x, y in cp:
            torch.mul(x, 1.0, out=y)
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    cgraph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(cgraph):
        for x, y in cp:
            torch.mul(x, 1.0, out=y)
    cms = timed(torch, cgraph.replay, max(3, steps // nsets), max(1, warmup // nsets)) / nsets
    copy_us = float(np.median(cms)) * 1e3
    return {"workload": "configs[4]: Q=2^20, E=8, weighted conf, p=0.6, tau=0.75",
            "copy_same_bytes_us": r3(copy_us),
            "mqueries_per_s": r3(cfg.Q / t / 1e6), "us_per_call": r3(t * 1e6),
            "us_best": r3(float(ms.min()) * 1e3), "survivors": S,
            "kernels_per_call": int(launches_per_call),
            "l2": "cold: 4 buffer sets round-robin, CUDA-graph replay",
            "roofline": {"bound": "hbm", "achieved": r3(gbs), "peak": pk["hbm_gbs"], "unit": "GB/s",
                         "frac": r3(gbs / pk["hbm_gbs"]), "frac_of_8tbs": r3(gbs / 8000.0),
                         "traffic": static_traffic("gate_compact_dram_bytes_per_launch"),
                         "algorithmic_bytes": int(byts)}}


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
    # inputs (1.1 GB) are far larger than L2: every call is cold
    ms = timed(torch, lambda: mosaic.gate_compact(a, cl, tau, w, mosaic.CONF_WEIGHTED, out=out), 10)
    return hbm_leg(ms, byts, pk)


def bench_assemble(torch, mosaic, pk):
    """mosaic_assemble_context over 2048 survivors of the C5 context recipe
    (U{8192..32768} tokens each, E = 8, prompt 256 + 8 traces at seeded cut points).
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
    ms = timed(torch, call, 20)   # 0.5 GB per call: every call is L2-cold
    assert int(mm.item()) == 0
    return hbm_leg(ms, 12.0 * T, pk, static_traffic("assemble_dram_bytes_per_launch"))


def bench_rope(torch, mosaic, pk, T, Hq, Hkv, D):
    """SURVEY 8(f) N1, second half: mosaic_rope_packed in place on a packed Q / K of configs[1]'s
    shape (positions 0..L-1 of ~2 k-token sequences).  Algorithmic bytes: every element of Q and K
    read and written once.  Parity: tests/test_gpu_rope.py."""
    dev = "cuda"
    g = torch.Generator(device=dev).manual_seed(41)
    q = torch.randn((T, Hq, D), device=dev, generator=g).to(torch.bfloat16)
    k = torch.randn((T, Hkv, D), device=dev, generator=g).to(torch.bfloat16)
    pos = (torch.arange(T, device=dev, dtype=torch.int32) % 2090).contiguous()
    ms = timed(torch, lambda: mosaic.rope_packed(q, k, pos, 1e6), 20)   # 1.3 GB: L2-cold
    return hbm_leg(ms, 4.0 * T * (Hq + Hkv) * D + 4.0 * T, pk,
                   static_traffic("rope_dram_bytes_per_launch"))


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
    ms = timed(torch, call, 5)
    pairs = n * sum(float(Lk - Lq + i + 1) for i in range(Lq))
    return tensor_leg(ms, 4.0 * Hq * D * pairs, pk)


def bench_lse_merge(torch, mosaic, pk, T, Hq, D):
    """mosaic_lse_merge on two partial results of configs[1]'s shape.  Algorithmic
    bytes: two bf16 reads and one write per element of O, three fp32 LSE values per row."""
    dev = "cuda"
    g = torch.Generator(device=dev).manual_seed(61)
    oa = torch.randn((T, Hq, D), device=dev, generator=g).to(torch.bfloat16)
    ob = torch.randn((T, Hq, D), device=dev, generator=g).to(torch.bfloat16)
    la = torch.randn((Hq, T), device=dev, generator=g)
    lb = torch.randn((Hq, T), device=dev, generator=g)
    o, lse = torch.empty_like(oa), torch.empty_like(la)
    ms = timed(torch, lambda: mosaic.lse_merge(oa, la, ob, lb, o=o, lse=lse), 20)   # 3.4 GB: cold
    return hbm_leg(ms, 6.0 * T * Hq * D + 12.0 * T * Hq, pk,
                   static_traffic("lse_merge_dram_bytes_per_launch"))


def bench_lse_merge_n(torch, mosaic, pk, T, Hq, D, n=4):
    """mosaic_lse_merge_n on n = 4 partial results of configs[1]'s shape.
    Algorithmic bytes: n bf16 reads and one write per element of O, n + 1 fp32 LSE values per row."""
    dev = "cuda"
    g = torch.Generator(device=dev).manual_seed(62)
    op = torch.randn((n, T, Hq, D), device=dev, generator=g).to(torch.bfloat16)
    lp = torch.randn((n, Hq, T), device=dev, generator=g)
    o = torch.empty((T, Hq, D), dtype=torch.bfloat16, device=dev)
    lse = torch.empty((Hq, T), dtype=torch.float32, device=dev)
    ms = timed(torch, lambda: mosaic.lse_merge_n(op, lp, o=o, lse=lse), 20)   # 5.7 GB: cold
    return hbm_leg(ms, 2.0 * (n + 1) * T * Hq * D + 4.0 * (n + 1) * T * Hq, pk,
                   static_traffic("lse_merge_n_dram_bytes_per_launch"))


def bench_prefix(torch, mosaic, pk):
    """mosaic_agg_prefill_attn_shared_prefix, 64 contexts of a shared 2048-token block
    + U{2048..8192} own tokens, Hq/Hkv/D = 28/4/128.  Algorithmic flops: 4 Hq D per visible (row, key)
    pair = sum_s L_s (L_s + 1) / 2 + T P.  Parity: tests/test_gpu_cascade.py."""
    n, P_, Hq, Hkv, D = 64, 2048, 28, 4, 128
    L = np.random.default_rng(91).integers(2048, 8193, size=n).astype(np.int64)
    cu = np.concatenate([[0], np.cumsum(L)]).astype(np.int64)
    T = int(cu[-1])
    dev = "cuda"
    g = torch.Generator(device=dev).manual_seed(91)
    q = torch.randn((T, Hq, D), device=dev, generator=g).to(torch.bfloat16)
    k = torch.randn((T, Hkv, D), device=dev, generator=g).to(torch.bfloat16)
    v = torch.randn((T, Hkv, D), device=dev, generator=g).to(torch.bfloat16)
    kp = torch.randn((P_, Hkv, D), device=dev, generator=g).to(torch.bfloat16)
    vp = torch.randn((P_, Hkv, D), device=dev, generator=g).to(torch.bfloat16)
    o = torch.empty_like(q)
    lse = torch.empty((Hq, T), dtype=torch.float32, device=dev)
    ws = torch.empty(int(mosaic.load().mosaic_agg_prefill_attn_shared_prefix_workspace_bytes(
        n, T, Hq, Hkv, D)), dtype=torch.uint8, device=dev)
    cu_d = torch.from_numpy(cu).to(dev)
    call = lambda: mosaic.agg_prefill_attn_shared_prefix(q, kp, vp, k, v, cu_d, n, int(L.max()),
                                                         D ** -0.5, o=o, lse=lse, workspace=ws)
    ms = timed(torch, call, 5)
    pairs = float(np.sum(L.astype(np.float64) * (L + 1.0) / 2.0) + float(T) * P_)
    leg = tensor_leg(ms, 4.0 * Hq * D * pairs, pk)
    leg["tokens"] = T
    return leg


def bench_chunked(torch, mosaic, pk):
    """mosaic_agg_prefill_attn_chunked, 4 contexts of 45 312 tokens (the longest
    configs[2] allows) in chunks of 8192 rows, Hq/Hkv/D = 28/4/128, one launch."""
    n, Lmax, Hq, Hkv, D = 4, 45312, 28, 4, 128
    cu = np.arange(0, (n + 1) * Lmax, Lmax, dtype=np.int64)
    T = int(cu[-1])
    dev = "cuda"
    g = torch.Generator(device=dev).manual_seed(92)
    q = torch.randn((T, Hq, D), device=dev, generator=g).to(torch.bfloat16)
    k = torch.randn((T, Hkv, D), device=dev, generator=g).to(torch.bfloat16)
    v = torch.randn((T, Hkv, D), device=dev, generator=g).to(torch.bfloat16)
    o = torch.empty_like(q)
    lse = torch.empty((Hq, T), dtype=torch.float32, device=dev)
    ws = torch.empty(int(mosaic.load().mosaic_agg_prefill_attn_chunked_workspace_bytes(
        n, T, 8192, Hq, Hkv, D)), dtype=torch.uint8, device=dev)
    cu_d = torch.from_numpy(cu).to(dev)
    call = lambda: mosaic.agg_prefill_attn_chunked(q, k, v, cu_d, n, Lmax, D ** -0.5, 8192, o=o,
                                                   lse=lse, workspace=ws)
    ms = timed(torch, call, 4, 1)
    return tensor_leg(ms, attn_flops([Lmax] * n, Hq, D), pk)


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
    ms = timed(torch, call, 20)   # K + V = 5 GB: L2-cold
    return hbm_leg(ms, 4.0 * Tk * Hkv * D, pk)


def bench_per_config(torch, mosaic, wl, pk, cids=(2, 3, 4)):
    """The attention of BASELINE.json configs[1..3] (C2, C3, C4) alone, at full size on seed 0, in
    the launch configuration the parity tests check (tests/test_gpu_attn.py); C5 is the headline."""
    out = {}
    for cid in cids:
        cfg = wl.CONFIGS[cid]
        gi = wl.gate_inputs(cfg, 0)
        g = mosaic.gate_compact(torch.from_numpy(gi.answers).cuda(),
                                torch.from_numpy(gi.ctx_len).cuda(), gi.tau)
        torch.cuda.synchronize()
        S, T, mx = int(g["n_survivors"]), int(g["total_tokens"]), int(g["max_seqlen"])
        L = np.diff(g["cu_seqlens"][:S + 1].cpu().numpy())
        q, k, v = wl.qkv(cfg, 0, T, device="cuda")
        o = torch.empty_like(q)
        lse = torch.empty((cfg.Hq, T), dtype=torch.float32, device="cuda")
        ws = torch.empty(mosaic.attn_workspace_bytes(S, T, cfg.Hq, cfg.Hkv, cfg.D),
                         dtype=torch.uint8, device="cuda")
        call = lambda: mosaic.agg_prefill_attn(q, k, v, g["cu_seqlens"], S, mx,
                                               wl.softmax_scale(cfg), o=o, lse=lse, workspace=ws)
        n = {2: 20, 3: 6, 4: 12}.get(cid, 6)
        for _ in range(3):
            call()
        torch.cuda.synchronize()
        time.sleep(1.0)   # a kernel timed alone: let the power budget recover from the previous leg
        leg = tensor_leg(timed(torch, call, n, 1), attn_flops(L, cfg.Hq, cfg.D), pk)
        leg.update(seqs=S, tokens=T)
        out[f"C{cid}"] = leg
        del q, k, v, o, lse, ws
        torch.cuda.empty_cache()
    return out


def bench_gated_stage(torch, mosaic, wl):
    """what the gate buys on a workload with the paper's statistics (MMLU-Pro bucket
    rates, survivors' traces 2.53 x longer): the aggregator prefill attention over ALL 768 contexts
    against gate + compaction + attention over the survivors of tau = 2/3 (61 GB of Q / K / V / O).
    The paper reports 1.74 x for its whole aggregator stage on MMLU-Pro with 84.62 % of the calls
    skipped."""
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
    t_all = float(np.mean(timed(torch, lambda: mosaic.agg_prefill_attn(
        q, k, v, cu_all, Q, int(ctx.max()), scale, o=o, lse=lse, workspace=ws), 3, 1)))
    out = mosaic.gate_compact(a_d, ctx_d, 2.0 / 3.0)
    torch.cuda.synchronize()
    S, T, mx = int(out["n_survivors"]), int(out["total_tokens"]), int(out["max_seqlen"])

    def gated():   # the survivors' Q / K / V are the first T rows of the same buffers (synthetic)
        mosaic.gate_compact(a_d, ctx_d, 2.0 / 3.0, out=out)
        mosaic.agg_prefill_attn(q[:T], k[:T], v[:T], out["cu_seqlens"], S, mx, scale, o=o[:T],
                                lse=lse.view(-1)[:Hq * T].view(Hq, T), workspace=ws)

    t_gated = float(np.mean(timed(torch, gated, 3, 1)))
    surv = out["bypass"].cpu().numpy() == 0
    return {"skip_rate": r3(1.0 - S / Q), "survivor_token_share": r3(T / T_all),
            "survivor_cost_share": r3(float((ctx[surv].astype(np.float64) ** 2).sum()
                                            / (ctx.astype(np.float64) ** 2).sum())),
            "ms_ungated": r3(t_all), "ms_gated": r3(t_gated), "speedup": r3(t_all / t_gated),
            "paper_speedup_mmlu_pro": 1.74}


def run_product(args):
    import torch
    import torch.distributed as dist

    from paper_2606_03014_b200 import mosaic
    from paper_2606_03014_b200 import workloads as wl

    mosaic.load()  # fails loudly when the CUDA library is missing: there is no fallback
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}")
    torch.cuda.set_device(local_rank)   # raises on a box with fewer GPUs than ranks
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    legs = set(args.legs.split(",")) if args.legs else set(ALL_LEGS)
    pk, pk_src = peaks()
    cfg = wl.C5
    seed = rank_seed(rank)  # weak scaling: every rank gates and attends its own batch, no collective
    gi = wl.gate_inputs(cfg, seed)
    a = torch.from_numpy(gi.answers).cuda()
    w = torch.from_numpy(gi.expert_conf).cuda()
    cl = torch.from_numpy(gi.ctx_len).cuda()
    gout = mosaic.gate_compact(a, cl, gi.tau, w, mosaic.CONF_WEIGHTED)
    torch.cuda.synchronize()
    S_all = int(gout["n_survivors"])
    S = min(cfg.max_attn_seqs, S_all)
    cu_host = gout["cu_seqlens"][:S + 1].cpu().numpy()
    lengths = np.diff(cu_host)
    T, max_len = int(cu_host[-1]), int(lengths.max())
    flops = attn_flops(lengths, cfg.Hq, cfg.D)
    q, k, v = wl.qkv(cfg, seed, T, device="cuda")
    o = torch.empty_like(q)
    lse = torch.empty((cfg.Hq, T), dtype=torch.float32, device="cuda")
    ws = torch.empty(mosaic.attn_workspace_bytes(S, T, cfg.Hq, cfg.Hkv, cfg.D), dtype=torch.uint8,
                     device="cuda")
    scale = wl.softmax_scale(cfg)
    ev_attn, ev_gate = [], []

    def step(is_timed):
        if is_timed:
            e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            e0.record()
        mosaic.gate_compact(a, cl, gi.tau, w, mosaic.CONF_WEIGHTED, out=gout)
        if is_timed:
            e1.record()
        mosaic.agg_prefill_attn(q, k, v, gout["cu_seqlens"], S, max_len, scale, o=o, lse=lse,
                                workspace=ws)
        if is_timed:
            e2.record()
            ev_gate.append((e0, e1))
            ev_attn.append((e1, e2))

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
    attn_ms = np.array([e0.elapsed_time(e1) for e0, e1 in ev_attn])
    gate_ms = np.array([e0.elapsed_time(e1) for e0, e1 in ev_gate])
    secs_max, flops_all = whole_job(secs, flops * args.steps, world, "cuda")
    value = flops_all / secs_max / 1e12

    # ---- end to end through the host-buffer call (pinned host memory, copies timed) ----------
    e2e = None
    if "e2e" in legs:
        pin = lambda t: torch.empty(t.shape, dtype=t.dtype, pin_memory=True).copy_(t)
        qh, kh, vh = pin(q), pin(k), pin(v)
        ah, wh, clh = (pin(torch.from_numpy(x)) for x in (gi.answers, gi.expert_conf, gi.ctx_len))
        del q, k, v, o, lse
        torch.cuda.empty_cache()
        out_h = {"o": torch.empty((T, cfg.Hq, cfg.D), dtype=torch.bfloat16, pin_memory=True),
                 "lse": torch.empty(cfg.Hq * T, dtype=torch.float32, pin_memory=True),
                 "mode": torch.empty(cfg.Q, dtype=torch.int32, pin_memory=True),
                 "conf": torch.empty(cfg.Q, dtype=torch.float32, pin_memory=True),
                 "bypass": torch.empty(cfg.Q, dtype=torch.uint8, pin_memory=True),
                 "survivor_idx": torch.empty(cfg.Q, dtype=torch.int32, pin_memory=True),
                 "cu_seqlens": torch.empty(cfg.Q + 1, dtype=torch.int64, pin_memory=True)}
        arena = torch.empty(mosaic.stage_host_arena_bytes(cfg.Q, cfg.E, T, cfg.Hq, cfg.Hkv, cfg.D),
                            dtype=torch.uint8, device="cuda")
        host_call = lambda: mosaic.stage_host(ah, wh, clh, gi.tau, mosaic.CONF_WEIGHTED, qh, kh, vh,
                                              scale, max_attn_seqs=S, out_h=out_h, arena=arena)
        e2e_steps = max(3, min(args.steps, 5))
        host_call()
        barrier()
        w0 = time.perf_counter()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(e2e_steps):
            host_call()
        e1.record()
        barrier()
        e2e_wall = time.perf_counter() - w0
        e2e_max, fl_e2e = whole_job(e0.elapsed_time(e1) * 1e-3, flops * e2e_steps, world, "cuda")
        h2d = (gi.answers.nbytes + gi.expert_conf.nbytes + gi.ctx_len.nbytes
               + (qh.numel() + kh.numel() + vh.numel()) * 2)
        d2h = 16 + cfg.Q * 9 + S_all * 4 + (S_all + 1) * 8 + T * cfg.Hq * cfg.D * 2 + T * cfg.Hq * 4
        e2e = {"value": r3(fl_e2e / e2e_max / 1e12), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "steps": e2e_steps,
               "ms_per_step": r3(e2e_max / e2e_steps * 1e3),
               "wall_ms_per_step": r3(e2e_wall / e2e_steps * 1e3),
               "call": "mosaic_stage_host (pinned host buffers)"}
        del arena, qh, kh, vh, out_h
    else:
        del q, k, v, o, lse
    torch.cuda.empty_cache()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    C2T, C2 = 158817, wl.C2   # configs[1]'s seed-0 token count: the shape of the HBM-bound legs
    gate_info = bench_gate_c5(torch, mosaic, wl, pk, gi) if "gate" in legs else None
    if gate_info is not None and "q24" in legs:
        gate_info["q24"] = bench_gate_q24(torch, mosaic, pk)
    nxt = {}

    def leg(name, key, fn):
        """A supplementary leg: a failure is recorded in the line, loudly, and does
        not take the headline measurements down with it."""
        if name not in legs:
            return
        try:
            nxt[key] = fn()
        except Exception as e:  # noqa: BLE001
            print(f"bench.py: leg {key} failed: {e!r}", file=sys.stderr, flush=True)
            nxt[key] = {"error": repr(e)[:120]}
            torch.cuda.empty_cache()

    leg("lse_merge", "lse_merge", lambda: bench_lse_merge(torch, mosaic, pk, C2T, C2.Hq, C2.D))
    leg("lse_merge_n", "lse_merge_n", lambda: bench_lse_merge_n(torch, mosaic, pk, C2T, C2.Hq, C2.D))
    leg("rope", "rope", lambda: bench_rope(torch, mosaic, pk, C2T, C2.Hq, C2.Hkv, C2.D))
    leg("assemble", "assemble", lambda: bench_assemble(torch, mosaic, pk))
    leg("decode", "decode", lambda: bench_decode(torch, mosaic, pk))
    leg("attn_kv", "attn_kv", lambda: bench_attn_kv(torch, mosaic, pk))
    leg("prefix", "shared_prefix", lambda: bench_prefix(torch, mosaic, pk))
    leg("chunked", "chunked", lambda: bench_chunked(torch, mosaic, pk))
    per_config = bench_per_config(torch, mosaic, wl, pk) if "per_config" in legs else {}
    attn_t = float(np.median(attn_ms)) * 1e-3
    attn_tflops = flops / attn_t / 1e12
    c5 = tensor_leg(attn_ms, flops, pk)
    c5.update(seqs=S, tokens=T)
    per_config["C5"] = c5
    leg("gated_stage", "gated_stage", lambda: bench_gated_stage(torch, mosaic, wl))
    cpu = None
    if "cpu" in legs:
        f, t, threads, desc = oracle_sample(cfg, 0, args.cpu_rows)
        cpu = {"value": f / t / 1e12, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": desc}
    sustained = secs_max > 0.3
    peak = pk["bf16_tflops_sustained"] if sustained else pk["bf16_tflops"]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": secs_max / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic", "gpu_launches": int(launches),
        "config": {"workload": workload_name(cfg), "Q": cfg.Q, "E": cfg.E, "tau": cfg.tau,
                   "survivors": S_all, "attn_seqs": S, "total_tokens": T, "max_seqlen": max_len,
                   "per_rank_seed": "rank", "tflop_per_step": r3(flops / 1e12),
                   "l2": "inputs > L2 (Q+K+V+O = %.1f GB per step)" %
                         ((2 * T * cfg.Hq + 2 * T * cfg.Hkv) * cfg.D * 2 / 1e9),
                   "gate_ms_in_step": r3(float(np.median(gate_ms))), "peaks": pk_src},
        "roofline": {"bound": "tensor", "achieved": r3(attn_tflops), "peak": peak,
                     "unit": "TFLOP/s", "frac": r3(attn_tflops / peak),
                     "traffic": static_traffic("attn_fwd_c5_dram_bytes_per_launch"),
                     "traffic_source": TRAFFIC_SOURCE, "kernel": "attn_fwd<128> (+ schedule_kernel)",
                     "ms_per_launch": r3(attn_t * 1e3),
                     "peak_kind": ("sustained" if sustained else "burst") + " (timed region %.1f s)" % secs_max,
                     "frac_burst": r3(attn_tflops / pk["bf16_tflops"]),
                     "frac_nominal_2250": r3(attn_tflops / 2250.0)},
        "gate": gate_info,
        "per_config": per_config,
        "next": nxt,
        "cpu_baseline": cpu,
        "e2e": e2e,
        "clocks": clocks,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="mosaic", choices=["mosaic", "reference"])
    ap.add_argument("--ref-rows", type=int, default=1024, help="reference arm: rows per step")
    ap.add_argument("--cpu-rows", type=int, default=32768, help="cpu_baseline: sampled rows")
    ap.add_argument("--legs", default="", help="comma-separated subset of " + ",".join(ALL_LEGS))
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args.gpus, run_product, (args,))
    else:
        run_product(args)


if __name__ == "__main__":
    main()
