"""Seeded synthetic workloads shaped like MOSAIC's (BASELINE.json configs[0..4] = C1..C5).

This module only draws INPUTS.  It holds none of the method's arithmetic (no vote, no scan, no
softmax) and is the one module the tests hand to both the CUDA path and the oracle.  The recipe
is stated in DESIGN.md ("Input recipe"); the paper's own benchmarks (MMLU-Pro, MedMCQA, GPQA;
PAPER.md P:L331-346) and expert traces are not available, these inputs stand in for them with
their shapes: 10-option multiple-choice labels, k = 3..8 experts, instruction-length vs
long-reasoning traces, 32k-class contexts.

Every array comes from numpy.random.Generator(PCG64(SeedSequence([seed, config_id, array_id]))).
Q/K/V come from a seeded torch generator on the device that will consume them (CPU for the small
configs, CUDA for the large ones) -- a fixed bit pattern for a given (seed, config, device kind).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

# array ids (third word of the seed sequence)
_A_CONSENSUS, _A_AGREE, _A_OTHER, _A_WEIGHT, _A_CTX, _A_CTX2, _A_CTX3, _A_QKV = range(8)


def rng(seed: int, config_id: int, array_id: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([seed, config_id, array_id])))


@dataclass(frozen=True)
class Config:
    """One BASELINE.json config.  `name` is what bench.py prints in config.workload."""
    config_id: int
    name: str
    Q: int                      # questions entering the gate
    E: int                      # experts per question (the paper's k)
    p_agree: float              # P(an expert gives the consensus answer)
    tau: float                  # gate threshold (1 and 2/3 are the paper's points)
    has_conf: bool              # fp32 expert confidences present (conf_mode 1 also run)
    Hq: int
    Hkv: int
    D: int
    ctx: str                    # context-length recipe, see ctx_len()
    k_scale: float = 1.0        # C4 multiplies K by 2 to sharpen the softmax
    max_attn_seqs: Optional[int] = None   # C5: attention over the first 16 survivors only
    n_options: int = 10


C1 = Config(1, "C1-tiny", 8, 3, 0.6, 2.0 / 3.0, False, 4, 2, 64, "uniform64_256")
C2 = Config(2, "C2-instruction", 256, 3, 0.6, 2.0 / 3.0, True, 28, 4, 128, "prompt256+3xLN600")
C3 = Config(3, "C3-reasoning-heavy", 64, 5, 0.6, 0.6, False, 28, 4, 128,
            "prompt256+3xLN600+2xLN6000")
C4 = Config(4, "C4-skewed", 512, 4, 0.6, 0.75, False, 32, 8, 128, "mix_1in8_long", k_scale=2.0)
C5 = Config(5, "C5-large-sweep", 1 << 20, 8, 0.6, 0.75, True, 64, 8, 128, "uniform8k_32k",
            max_attn_seqs=16)
CONFIGS = {c.config_id: c for c in (C1, C2, C3, C4, C5)}
C5_SWEEP = [(p, tau) for p in (0.3, 0.6, 0.9) for tau in (0.5, 0.75)]


def answers(cfg: Config, seed: int, p_agree: Optional[float] = None, Q: Optional[int] = None):
    """int32 [Q,E]: a consensus label g ~ U{0..9} per question; each expert independently
    answers g with probability p, otherwise one of the other nine labels uniformly."""
    Q = cfg.Q if Q is None else Q
    p = cfg.p_agree if p_agree is None else p_agree
    g = rng(seed, cfg.config_id, _A_CONSENSUS).integers(0, cfg.n_options, size=Q, dtype=np.int32)
    hit = rng(seed, cfg.config_id, _A_AGREE).random((Q, cfg.E)) < p
    other = rng(seed, cfg.config_id, _A_OTHER).integers(0, cfg.n_options - 1, size=(Q, cfg.E),
                                                        dtype=np.int32)
    other = other + (other >= g[:, None])
    return np.where(hit, g[:, None], other).astype(np.int32)


def expert_conf(cfg: Config, seed: int, Q: Optional[int] = None):
    """fp32 [Q,E] ~ U[0,1) on the 2^-24 grid, so binary64 sums of a row are exact."""
    Q = cfg.Q if Q is None else Q
    u = rng(seed, cfg.config_id, _A_WEIGHT).integers(0, 1 << 32, size=(Q, cfg.E), dtype=np.uint64)
    return ((u >> 8).astype(np.float64) * 2.0 ** -24).astype(np.float32)


def _lognormal_len(g: np.random.Generator, median: float, sigma: float, cap: int, size):
    x = np.rint(g.lognormal(np.log(median), sigma, size=size))
    return np.minimum(cap, np.maximum(1, x)).astype(np.int64)


def ctx_len(cfg: Config, seed: int, Q: Optional[int] = None):
    """int32 [Q]: tokens in question q's aggregator context = prompt + all expert traces."""
    Q = cfg.Q if Q is None else Q
    g = rng(seed, cfg.config_id, _A_CTX)
    if cfg.ctx == "uniform64_256":
        n = g.integers(64, 257, size=Q)
    elif cfg.ctx == "prompt256+3xLN600":
        n = 256 + _lognormal_len(g, 600.0, 0.5, 4096, (Q, 3)).sum(axis=1)
    elif cfg.ctx == "prompt256+3xLN600+2xLN6000":
        g2 = rng(seed, cfg.config_id, _A_CTX2)
        n = (256 + _lognormal_len(g, 600.0, 0.5, 4096, (Q, 3)).sum(axis=1)
             + _lognormal_len(g2, 6000.0, 0.5, 16384, (Q, 2)).sum(axis=1))
    elif cfg.ctx == "mix_1in8_long":
        g2 = rng(seed, cfg.config_id, _A_CTX2)
        g3 = rng(seed, cfg.config_id, _A_CTX3)
        is_long = g.random(Q) < 0.125
        n = np.where(is_long, g2.integers(4000, 10001, size=Q), g3.integers(300, 801, size=Q))
    elif cfg.ctx == "uniform8k_32k":
        n = g.integers(8192, 32769, size=Q)
    else:
        raise ValueError(cfg.ctx)
    return n.astype(np.int32)


_A_PARTS, _A_TOKENS = 21, 22
VOCAB = 151936  # the aggregator models the paper runs are Qwen-family; any vocabulary would do


def context_parts(cfg: Config, seed: int, Q: Optional[int] = None, E: Optional[int] = None):
    """SURVEY 8(f) N1 inputs: every question's context split into a prompt and E expert traces
    whose lengths add up to ctx_len(cfg, seed)[q] (so cu_seqlens is the one every other step sees).
    The prompt is min(256, n // 4) tokens, as in the ctx recipes of configs 2-3; E - 1 seeded cut
    points split the rest (a trace may be empty).  Returns (prompt_tokens int32, prompt_off int64
    [Q+1], trace_tokens int32, trace_off int64 [Q*E+1]) with seeded token ids in [0, VOCAB)."""
    Q = cfg.Q if Q is None else Q
    E = cfg.E if E is None else E
    n = ctx_len(cfg, seed, Q).astype(np.int64)
    g = rng(seed, cfg.config_id, _A_PARTS)
    p_len = np.minimum(256, n // 4)
    rest = n - p_len
    cuts = np.sort((g.random((Q, max(E - 1, 0))) * (rest[:, None] + 1)).astype(np.int64), axis=1)
    edges = np.concatenate([np.zeros((Q, 1), np.int64), cuts, rest[:, None]], axis=1)
    t_len = np.diff(edges, axis=1)  # [Q, E]
    prompt_off = np.concatenate([[0], np.cumsum(p_len)]).astype(np.int64)
    trace_off = np.concatenate([[0], np.cumsum(t_len.reshape(-1))]).astype(np.int64)
    gt = rng(seed, cfg.config_id, _A_TOKENS)
    prompt_tokens = gt.integers(0, VOCAB, size=int(prompt_off[-1]), dtype=np.int32)
    trace_tokens = gt.integers(0, VOCAB, size=int(trace_off[-1]), dtype=np.int32)
    return prompt_tokens, prompt_off, trace_tokens, trace_off


_A_N4 = 31
# MMLU-Pro-shaped gate statistics (Table 1: 45.71 % of the questions are
# 3:0 and 84.62 % are 3:0 or 2:1) and trace lengths that fall with agreement (mean
# output 1 064 tokens for 3:0 against 2 696 for 1:1:1, 2.53 x, Spearman rho = -0.27).
N4_BUCKET_RATES = (0.4571, 0.8462 - 0.4571, 1.0 - 0.8462)       # 3:0, 2:1, 1:1:1
N4_MEAN_TOKENS = (1064.0, (1064.0 * 2696.0) ** 0.5, 2696.0)   # 2:1 is not printed: geometric mean
N4_SIGMA, N4_CAP, N4_PROMPT = 1.15, 16384, 256


def n4_inputs(seed: int, Q: int):
    """k = 3 answers with the paper's bucket rates and, per expert trace, a lognormal length whose
    mean depends on the question's bucket (sigma = 1.15 puts the Spearman correlation between
    agreement and trace length, per (question, expert) sample, at the paper's -0.27).  Returns
    (answers int32 [Q,3], ctx_len int32 [Q] = 256-token prompt + three traces, trace_len [Q,3])."""
    g = rng(seed, 6, _A_N4)
    b = g.choice(3, size=Q, p=np.asarray(N4_BUCKET_RATES) / sum(N4_BUCKET_RATES))
    first = g.integers(0, 10, size=Q)
    second = (first + g.integers(1, 10, size=Q)) % 10
    third = (first + g.integers(1, 10, size=Q)) % 10
    third = np.where(third == second, (third + 1) % 10, third)
    third = np.where(third == first, (third + 1) % 10, third)
    third = np.where(third == second, (third + 1) % 10, third)
    odd = g.integers(0, 3, size=Q)  # which expert dissents in a 2:1 question
    a = np.repeat(first[:, None], 3, axis=1)
    two = b == 1
    a[two, odd[two]] = second[two]
    three = b == 2
    a[three, 1] = second[three]
    a[three, 2] = third[three]
    mean = np.asarray(N4_MEAN_TOKENS)[b]
    mu = np.log(mean) - N4_SIGMA ** 2 / 2
    t_len = np.exp(mu[:, None] + N4_SIGMA * g.standard_normal((Q, 3)))
    t_len = np.clip(np.rint(t_len), 1, N4_CAP).astype(np.int64)
    ctx = (N4_PROMPT + t_len.sum(axis=1)).astype(np.int32)
    return a.astype(np.int32), ctx, t_len


@dataclass
class GateInputs:
    answers: np.ndarray
    expert_conf: Optional[np.ndarray]
    ctx_len: np.ndarray
    tau: float
    E: int
    extra: dict = field(default_factory=dict)


def gate_inputs(cfg: Config, seed: int, p_agree: Optional[float] = None,
                tau: Optional[float] = None, Q: Optional[int] = None) -> GateInputs:
    return GateInputs(answers(cfg, seed, p_agree, Q),
                      expert_conf(cfg, seed, Q) if cfg.has_conf else None,
                      ctx_len(cfg, seed, Q), cfg.tau if tau is None else tau, cfg.E)


def softmax_scale(cfg: Config) -> float:
    return 1.0 / float(np.sqrt(cfg.D))


def qkv(cfg: Config, seed: int, total_tokens: int, device="cpu"):
    """bf16 Q [T,Hq,D], K,V [T,Hkv,D] ~ N(0,1) (fp32 draws rounded to nearest-even), K times
    cfg.k_scale.  torch is used for the bf16 dtype and, on CUDA, to draw in place in HBM."""
    import torch

    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(int(np.random.SeedSequence([seed, cfg.config_id, _A_QKV]).generate_state(1)[0]))

    def draw(H, scale):
        out = torch.empty((total_tokens, H, cfg.D), dtype=torch.bfloat16, device=dev)
        step = max(1, (1 << 26) // (H * cfg.D))          # fp32 staging of <= 256 MiB
        for t0 in range(0, total_tokens, step):
            t1 = min(total_tokens, t0 + step)
            x = torch.randn((t1 - t0, H, cfg.D), dtype=torch.float32, device=dev, generator=gen)
            if scale != 1.0:
                x = x * scale
            out[t0:t1] = x.to(torch.bfloat16)
        return out

    return draw(cfg.Hq, 1.0), draw(cfg.Hkv, cfg.k_scale), draw(cfg.Hkv, 1.0)


def sample_rows(cu_seqlens: np.ndarray, Hq: int, Hkv: int, seed: int, config_id: int,
                n_random: int = 2048, tile: int = 128):
    """Output rows (seq, head, pos) the O(L^2) oracle is asked for on the large configs:
    tile-edge and sequence-edge rows of every sequence for one head per KV group, plus
    n_random uniform draws half of which go to the shortest and the longest sequence."""
    cu = np.asarray(cu_seqlens, np.int64)
    L = np.diff(cu)
    n_seqs = L.shape[0]
    G = Hq // Hkv
    g = rng(seed, config_id, 100)
    rows = set()
    for s in range(n_seqs):
        if L[s] == 0:
            continue
        last_tile = tile * ((int(L[s]) - 1) // tile)
        cand = {0, 1, tile - 1, tile, tile + 1, int(L[s]) - 2, int(L[s]) - 1, last_tile,
                last_tile - 1, 2 * tile - 1, 2 * tile}
        for i in cand:
            if 0 <= i < L[s]:
                for kvh in range(Hkv):
                    h = kvh * G + int(g.integers(0, G))
                    rows.add((s, h, int(i)))
    nz = np.flatnonzero(L > 0)
    if nz.size and n_random:
        shortest, longest = nz[np.argmin(L[nz])], nz[np.argmax(L[nz])]
        for r in range(n_random):
            if r % 4 == 0:
                s = int(shortest)
            elif r % 4 == 1:
                s = int(longest)
            else:
                s = int(nz[g.integers(0, nz.size)])
            rows.add((s, int(g.integers(0, Hq)), int(g.integers(0, L[s]))))
    rows = sorted(rows)
    return (np.array([r[0] for r in rows], np.int32), np.array([r[1] for r in rows], np.int32),
            np.array([r[2] for r in rows], np.int64))
