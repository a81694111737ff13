"""oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes front end of ``oracle/mosaic_oracle.c``: the plain CPU (integer / binary64) statement of
MOSAIC's confidence-gated aggregator stage (Sec. 4.2, Alg. 1, and
the attention definition BASELINE.json's north_star fixes).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import this package.  It imports nothing from ``paper_2606_03014_b200`` and the CUDA path imports
nothing from here.

All arrays are numpy.  bf16 tensors are passed as ``uint16`` bit patterns.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "mosaic_oracle.c"
_LIB = _HERE / "libmosaic_oracle.so"
# No -ffast-math, no -march: the arithmetic is the C source's, in source order.
_CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-fno-fast-math", "-ffp-contract=off"]

_lib = None


def build(force: bool = False) -> Path:
    """Compile the C oracle with gcc (building the checker is not using it)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".{os.getpid()}.tmp")
        subprocess.run(["gcc", *_CFLAGS, str(_SRC), "-o", str(tmp), "-lm"], check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        p = ctypes.c_void_p
        lib.oracle_gate.argtypes = [p, p, ctypes.c_int64, ctypes.c_int32, ctypes.c_float,
                                    ctypes.c_int32, p, p, p, p, p]
        lib.oracle_gate.restype = None
        lib.oracle_gate_ext.argtypes = [p, p, ctypes.c_int64, ctypes.c_int32, ctypes.c_float, p,
                                        ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, p, p, p, p, p]
        lib.oracle_gate_ext.restype = None
        lib.oracle_compact.argtypes = [p, p, ctypes.c_int64, p, p, p, p]
        lib.oracle_compact.restype = ctypes.c_int64
        lib.oracle_attn_rows.argtypes = [p, p, p, p, ctypes.c_int64, p, p, p, ctypes.c_int32,
                                         ctypes.c_int32, ctypes.c_int32, ctypes.c_float, p, p, p]
        lib.oracle_attn_rows.restype = ctypes.c_int
        lib.oracle_attn_full.argtypes = [p, p, p, p, ctypes.c_int32, ctypes.c_int32,
                                         ctypes.c_int32, ctypes.c_int32, ctypes.c_float, p, p]
        lib.oracle_attn_full.restype = ctypes.c_int
        lib.oracle_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _c(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a


def num_threads() -> int:
    """Threads the attention oracle's OpenMP loops use (OMP_NUM_THREADS or all cores)."""
    return int(_load().oracle_num_threads())


def gate(answers, tau, expert_conf=None, conf_mode: int = 0):
    """Alg. 1 lines 2-4 for every question.

    answers int32 [Q,E]; tau is rounded to fp32 (reading G-4); expert_conf fp32 [Q,E] for
    conf_mode 1.  Returns dict(mode, count, agree, conf, bypass).
    """
    answers = _c(answers, np.int32)
    Q, E = answers.shape
    if conf_mode not in (0, 1):
        raise ValueError("conf_mode")
    w = None
    if conf_mode == 1:
        w = _c(expert_conf, np.float32)
        assert w.shape == (Q, E)
    out = dict(mode=np.empty(Q, np.int32), count=np.empty(Q, np.int32),
               agree=np.empty(Q, np.float32), conf=np.empty(Q, np.float32),
               bypass=np.empty(Q, np.uint8))
    _load().oracle_gate(_ptr(answers), _ptr(w), Q, E, ctypes.c_float(np.float32(tau)),
                        conf_mode, _ptr(out["mode"]), _ptr(out["count"]), _ptr(out["agree"]),
                        _ptr(out["conf"]), _ptr(out["bypass"]))
    return out


def gate_tau_per_query(answers, tau_q, expert_conf=None, conf_mode: int = 0):
    """the gate with a threshold per question (a per-task tau table gathered by
    the caller's task ids; the paper names its single static threshold as a limitation).
    Vote, mode and confidence do not depend on the threshold (Alg. 1 lines 2-3): they are the
    scalar gate's; line 4 becomes bypass[q] = conf[q] >= tau_q[q], compared in fp32 like reading
    G-4 compares the scalar.  A NaN threshold never bypasses."""
    tau_q = _c(tau_q, np.float32)
    out = gate(answers, 0.0, expert_conf, conf_mode)
    assert tau_q.shape == out["conf"].shape
    out["bypass"] = (out["conf"] >= tau_q).astype(np.uint8)
    return out


def gate_ext(answers, tau, expert_conf=None, conf_mode: int = 0, tau_q=None,
             abstain_policy: int = 0, abstain_label: int = -1):
    """the gate with the optional estimator settings (oracle_gate_ext in the C
    source states them): conf_mode 2 = the answer is the label with the largest weight sum
    (reading N3-3); tau_q = a threshold per question (N3-1); abstain_policy 1 / 2 = an expert
    whose label is abstain_label did not answer, C still divides by E (1) or by the experts that
    answered (2) (N3-2).  Returns dict(mode, count, agree, conf, bypass)."""
    answers = _c(answers, np.int32)
    Q, E = answers.shape
    if conf_mode not in (0, 1, 2) or abstain_policy not in (0, 1, 2):
        raise ValueError("conf_mode / abstain_policy")
    w = None
    if conf_mode != 0:
        w = _c(expert_conf, np.float32)
        assert w.shape == (Q, E)
    tq = None
    if tau_q is not None:
        tq = _c(tau_q, np.float32)
        assert tq.shape == (Q,)
    out = dict(mode=np.empty(Q, np.int32), count=np.empty(Q, np.int32),
               agree=np.empty(Q, np.float32), conf=np.empty(Q, np.float32),
               bypass=np.empty(Q, np.uint8))
    _load().oracle_gate_ext(_ptr(answers), _ptr(w), Q, E, ctypes.c_float(np.float32(tau)), _ptr(tq),
                            conf_mode, abstain_policy, int(abstain_label), _ptr(out["mode"]),
                            _ptr(out["count"]), _ptr(out["agree"]), _ptr(out["conf"]),
                            _ptr(out["bypass"]))
    return out


def conf_gate(conf, tau, tau_q=None):
    """Alg. 1 line 4 on a confidence C(q) the caller computed:
    bypass[q] = conf[q] >= tau (or tau_q[q]) in fp32; a NaN on either side never bypasses."""
    c = _c(conf, np.float32)
    t = np.float32(tau) if tau_q is None else _c(tau_q, np.float32)
    with np.errstate(invalid="ignore"):
        return (c >= t).astype(np.uint8)


def compact(bypass, ctx_len):
    """Alg. 1 line 6 survivors as a ragged batch (BJ:north_star).

    Returns dict(survivor_idx int32 [S], cu_seqlens int64 [S+1], n_survivors, total_tokens,
    max_seqlen).
    """
    bypass = _c(bypass, np.uint8)
    ctx_len = _c(ctx_len, np.int32)
    Q = bypass.shape[0]
    assert ctx_len.shape == (Q,)
    idx = np.empty(max(Q, 1), np.int32)
    cu = np.empty(Q + 1, np.int64)
    tot = np.zeros(1, np.int64)
    mx = np.zeros(1, np.int32)
    S = int(_load().oracle_compact(_ptr(bypass), _ptr(ctx_len), Q, _ptr(idx), _ptr(cu),
                                   _ptr(tot), _ptr(mx)))
    return dict(survivor_idx=idx[:S].copy(), cu_seqlens=cu[:S + 1].copy(), n_survivors=S,
                total_tokens=int(tot[0]), max_seqlen=int(mx[0]))


def attn_kv_full(q, k, v, cu_seqlens_q, cu_seqlens_k, softmax_scale, causal: bool = True):
    """SURVEY.md 8(f) N2 (prefix-cached / chunked prefill): the q rows of a sequence are the LAST
    Lq of its Lk positions, so row i sees keys j <= i + (Lk - Lq) ("bottom-right" causal alignment,
    DESIGN.md reading N2-1; Lk = Lq is the plain prefill of north_star).  The definition written
    out per (sequence, q head) with numpy in binary64: S = scale Q K^T, mask, row softmax, O = P V,
    LSE = ln sum_j exp(S_ij).  q uint16 [Tq,Hq,D], k/v uint16 [Tk,Hkv,D] (bf16 bits).
    causal = False: every q row sees all Lk keys (a block of earlier keys in a split-KV prefill).
    Returns (O float64 [Tq,Hq,D], LSE float64 [Hq,Tq])."""
    def f64(bits):
        return (_c(bits, np.uint16).astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    Q, K, V = f64(q), f64(k), f64(v)
    cq, ck = _c(cu_seqlens_q, np.int64), _c(cu_seqlens_k, np.int64)
    Tq, Hq, D = Q.shape
    Hkv = K.shape[1]
    assert cq.shape == ck.shape and Hq % Hkv == 0
    O = np.zeros((Tq, Hq, D), np.float64)
    lse = np.zeros((Hq, Tq), np.float64)
    scale = float(np.float32(softmax_scale))
    for s_ in range(cq.shape[0] - 1):
        a, b = int(cq[s_]), int(cq[s_ + 1])
        c, d = int(ck[s_]), int(ck[s_ + 1])
        Lq, Lk = b - a, d - c
        if Lq == 0:
            continue
        assert Lk >= (Lq if causal else 1)
        visible = np.arange(Lk)[None, :] <= (np.arange(Lq)[:, None] + (Lk - Lq))
        if not causal:
            visible = np.ones((Lq, Lk), bool)
        for h in range(Hq):
            g = h // (Hq // Hkv)
            S = scale * (Q[a:b, h] @ K[c:d, g].T)
            S = np.where(visible, S, -np.inf)
            M = S.max(axis=1, keepdims=True)
            P = np.exp(S - M)
            Z = P.sum(axis=1, keepdims=True)
            O[a:b, h] = (P / Z) @ V[c:d, g]
            lse[h, a:b] = (M + np.log(Z))[:, 0]
    return O, lse


def lse_merge(o_a, lse_a, o_b, lse_b):
    """the attention result over the union of two disjoint key sets from the
    partial results over each (binary64): LSE = ln(e^LSE_a + e^LSE_b), O = O_a e^(LSE_a - LSE) +
    O_b e^(LSE_b - LSE).  o_* float64 [T,Hq,D], lse_* float64 [Hq,T]; -inf = empty partial."""
    o_a, o_b = np.asarray(o_a, np.float64), np.asarray(o_b, np.float64)
    la, lb = np.asarray(lse_a, np.float64), np.asarray(lse_b, np.float64)
    lse = np.logaddexp(la, lb)
    with np.errstate(invalid="ignore"):
        wa = np.where(np.isneginf(la), 0.0, np.exp(la - lse))
        wb = np.where(np.isneginf(lb), 0.0, np.exp(lb - lse))
    o = np.where(wa.T[:, :, None] != 0, o_a * wa.T[:, :, None], 0.0) + \
        np.where(wb.T[:, :, None] != 0, o_b * wb.T[:, :, None], 0.0)
    return o, lse


def lse_merge_n(o_parts, lse_parts):
    """the n-way form of lse_merge (reading N2-2): partial results over n
    pairwise disjoint key sets -> LSE = ln sum_p e^LSE_p, O = sum_p O_p e^(LSE_p - LSE), binary64.
    o_parts float64 [n,T,Hq,D], lse_parts float64 [n,Hq,T]; -inf marks an empty partial; a row with
    no non-empty partial gets O = 0, LSE = -inf."""
    o_parts = np.asarray(o_parts, np.float64)
    lp = np.asarray(lse_parts, np.float64)
    with np.errstate(invalid="ignore", divide="ignore"):
        m = lp.max(axis=0)
        z = np.where(np.isneginf(lp), 0.0, np.exp(lp - np.where(np.isneginf(m), 0.0, m))).sum(axis=0)
        lse = np.where(z > 0, m + np.log(np.where(z > 0, z, 1.0)), -np.inf)
        w = np.where(np.isneginf(lp), 0.0, np.exp(lp - np.where(np.isneginf(lse), 0.0, lse)))  # [n,Hq,T]
    wt = np.transpose(w, (0, 2, 1))[..., None]                                     # [n,T,Hq,1]
    o = np.where(wt != 0, o_parts * wt, 0.0).sum(axis=0)
    return o, lse


def attn_shared_prefix(q, k_prefix, v_prefix, k, v, cu_seqlens, softmax_scale):
    """SURVEY.md 8(f) N2, shared-prefix cascade (reading N2-5): sequence s is the shared
    block of P keys followed by its own L_s tokens; the rows computed are those of the own tokens,
    row i seeing all P prefix keys and its own keys j <= i.  Written as the definition: every
    sequence's keys are concatenated EXPLICITLY (prefix ++ own) and handed to attn_kv_full with
    Lq = L_s, Lk = P + L_s (bottom-right alignment: key j visible iff j <= i + P).
    q uint16 [T,Hq,D]; k_prefix, v_prefix uint16 [P,Hkv,D]; k, v uint16 [T,Hkv,D]."""
    cu = _c(cu_seqlens, np.int64)
    kp, vp = _c(k_prefix, np.uint16), _c(v_prefix, np.uint16)
    k, v = _c(k, np.uint16), _c(v, np.uint16)
    P = kp.shape[0]
    ks, vs, ck = [], [], [0]
    for s_ in range(cu.shape[0] - 1):
        a, b = int(cu[s_]), int(cu[s_ + 1])
        if b > a:
            ks += [kp, k[a:b]]
            vs += [vp, v[a:b]]
        ck.append(ck[-1] + ((P + b - a) if b > a else 0))
    kcat = np.concatenate(ks) if ks else np.zeros((0,) + k.shape[1:], np.uint16)
    vcat = np.concatenate(vs) if vs else np.zeros((0,) + v.shape[1:], np.uint16)
    return attn_kv_full(q, kcat, vcat, cu, np.asarray(ck, np.int64), softmax_scale, causal=True)


def assemble_context(survivor_idx, cu_seqlens, prompt_tokens, prompt_off, trace_tokens, trace_off,
                     E: int):
    """the survivors' aggregator contexts as one packed token batch.  The
    aggregator reads "the combined output or reasoning traces of its experts" (Alg. 1
    `Aggregator(q, {a_i})`); reading N1-1 fixes the order the paper leaves open:
    context of survivor j (question q = survivor_idx[j]) = prompt(q) ++ trace(q,0) ++ ... ++
    trace(q,E-1).  Written out sequence by sequence, segment by segment (plain slices, no
    arithmetic to get wrong beyond the offsets).  A sequence whose cu_seqlens length differs from
    prompt + traces is truncated, or padded with -1, and counted in n_mismatch.

    Returns dict(input_ids int32 [T], position_ids int32 [T], n_mismatch int).
    """
    idx = _c(survivor_idx, np.int32)
    cu = _c(cu_seqlens, np.int64)
    pt, po = _c(prompt_tokens, np.int32), _c(prompt_off, np.int64)
    tt, to = _c(trace_tokens, np.int32), _c(trace_off, np.int64)
    S = idx.shape[0]
    assert cu.shape == (S + 1,)
    T = int(cu[S]) if S else 0
    ids = np.full(T, -1, np.int32)
    pos = np.empty(T, np.int32)
    n_mismatch = 0
    for j in range(S):
        q = int(idx[j])
        parts = [pt[po[q]:po[q + 1]]]
        for e in range(E):
            parts.append(tt[to[q * E + e]:to[q * E + e + 1]])
        seq = np.concatenate(parts) if parts else np.empty(0, np.int32)
        a, b = int(cu[j]), int(cu[j + 1])
        L = b - a
        if seq.shape[0] != L:
            n_mismatch += 1
        m = min(L, seq.shape[0])
        ids[a:a + m] = seq[:m]
        pos[a:b] = np.arange(L, dtype=np.int32)
    return dict(input_ids=ids, position_ids=pos, n_mismatch=n_mismatch)


def rope(x, position_ids, theta: float):
    """SURVEY.md 8(f) N1, second half: rotary position embedding of a packed [T, H, D] tensor
    (binary64 values in, binary64 out; the caller rounds to bf16).  DESIGN.md reading N1-4: pairs
    (i, i + D/2), w_i = theta^(-2i/D), a = position * w_i,
    out[i] = x[i] cos a - x[i+D/2] sin a, out[i+D/2] = x[i+D/2] cos a + x[i] sin a."""
    x = np.asarray(x, np.float64)
    T, H, D = x.shape
    pos = np.asarray(position_ids, np.float64).reshape(T)
    half = D // 2
    w = np.float64(theta) ** (-2.0 * np.arange(half, dtype=np.float64) / D)
    a = pos[:, None] * w[None, :]                      # [T, D/2]
    c, s = np.cos(a)[:, None, :], np.sin(a)[:, None, :]
    lo, hi = x[..., :half], x[..., half:]
    return np.concatenate([lo * c - hi * s, hi * c + lo * s], axis=-1)


def _check_qkv(q, k, v, cu_seqlens):
    q = _c(q, np.uint16)
    k = _c(k, np.uint16)
    v = _c(v, np.uint16)
    cu = _c(cu_seqlens, np.int64)
    T, Hq, D = q.shape
    Tk, Hkv, Dk = k.shape
    assert v.shape == k.shape and Tk == T and Dk == D and Hq % Hkv == 0
    assert cu[0] == 0 and cu[-1] == T and np.all(np.diff(cu) >= 0)
    return q, k, v, cu, T, Hq, Hkv, D


def attn_rows(q, k, v, cu_seqlens, row_seq, row_head, row_pos, softmax_scale):
    """Selected output rows (sequence, q head, position) of the attention definition.

    q uint16 [T,Hq,D], k/v uint16 [T,Hkv,D] (bf16 bits).  Returns (O float64 [n,D],
    LSE float64 [n], psum float64 [n]) where psum is the sum of the row's softmax weights.
    """
    q, k, v, cu, T, Hq, Hkv, D = _check_qkv(q, k, v, cu_seqlens)
    rs = _c(row_seq, np.int32)
    rh = _c(row_head, np.int32)
    rp = _c(row_pos, np.int64)
    n = rs.shape[0]
    assert rh.shape == (n,) and rp.shape == (n,)
    if n:
        L = np.diff(cu)[rs]
        assert np.all((rp >= 0) & (rp < L)) and np.all((rh >= 0) & (rh < Hq))
    O = np.empty((n, D), np.float64)
    lse = np.empty(n, np.float64)
    ps = np.empty(n, np.float64)
    rc = _load().oracle_attn_rows(_ptr(q), _ptr(k), _ptr(v), _ptr(cu), n, _ptr(rs), _ptr(rh),
                                  _ptr(rp), Hq, Hkv, D, ctypes.c_float(np.float32(softmax_scale)),
                                  _ptr(O), _ptr(lse), _ptr(ps))
    if rc:
        raise MemoryError("oracle_attn_rows")
    return O, lse, ps


def attn_full(q, k, v, cu_seqlens, softmax_scale):
    """Every row: returns (O float64 [T,Hq,D], LSE float64 [Hq,T])."""
    q, k, v, cu, T, Hq, Hkv, D = _check_qkv(q, k, v, cu_seqlens)
    O = np.empty((T, Hq, D), np.float64)
    lse = np.empty((Hq, T), np.float64)
    rc = _load().oracle_attn_full(_ptr(q), _ptr(k), _ptr(v), _ptr(cu), cu.shape[0] - 1, Hq, Hkv,
                                  D, ctypes.c_float(np.float32(softmax_scale)), _ptr(O), _ptr(lse))
    if rc:
        raise MemoryError("oracle_attn_full")
    return O, lse
