"""ctypes binding over libmosaic.so (include/mosaic.h).  Argument marshalling only: every step of
the path runs in the library's kernels.  torch is used for device memory and streams.

There is no fallback: if the library is missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes
from pathlib import Path
from typing import Optional

import torch

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libmosaic.so"

OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_WORKSPACE_TOO_SMALL, ERR_CUDA = range(5)
CONF_VOTE, CONF_WEIGHTED, CONF_WEIGHTED_ARGMAX = 0, 1, 2
ABSTAIN_NONE, ABSTAIN_KEEP_K, ABSTAIN_SHRINK_K = 0, 1, 2

_vp, _i32, _i64, _f32, _sz = (ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_float,
                              ctypes.c_size_t)

# name -> (restype, argtypes): every symbol include/mosaic.h declares
SIGNATURES = {
    "mosaic_gate": (ctypes.c_int, [_vp, _vp, _i64, _i32, _f32, _i32, _vp, _vp, _vp, _vp, _vp, _vp]),
    "mosaic_compact_workspace_bytes": (_sz, [_i64]),
    "mosaic_compact": (ctypes.c_int, [_vp, _vp, _i64, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]),
    "mosaic_compact_static": (ctypes.c_int, [_vp, _vp, _i64, _vp, _vp, _vp, _vp, _vp, _vp]),
    "mosaic_gate_compact": (ctypes.c_int, [_vp, _vp, _vp, _i64, _i32, _f32, _i32, _vp, _vp, _vp,
                                           _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]),
    "mosaic_gate_compact_tau": (ctypes.c_int, [_vp, _vp, _vp, _i64, _i32, _vp, _i32, _vp, _vp, _vp,
                                               _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]),
    "mosaic_gate_compact_ext": (ctypes.c_int, [_vp, _vp, _vp, _i64, _i32, _f32, _vp, _i32, _i32, _i32,
                                               _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp,
                                               _sz, _vp]),
    "mosaic_conf_compact": (ctypes.c_int, [_vp, _vp, _i64, _f32, _vp, _vp, _vp, _vp, _vp, _vp, _vp,
                                           _vp, _sz, _vp]),
    "mosaic_agg_prefill_attn_workspace_bytes": (_sz, [_i32, _i64, _i32, _i32, _i32]),
    "mosaic_agg_prefill_attn": (ctypes.c_int, [_vp, _vp, _vp, _vp, _i32, _i64, _i32, _i32, _i32,
                                               _i32, _f32, _vp, _vp, _vp, _sz, _vp]),
    "mosaic_agg_prefill_attn_kv": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp, _i32, _i64, _i64, _i32,
                                                  _i32, _i32, _i32, _f32, _i32, _vp, _vp, _vp, _sz,
                                                  _vp]),
    "mosaic_agg_decode_attn_workspace_bytes": (_sz, [_i32, _i64, _i32, _i32, _i32]),
    "mosaic_agg_decode_attn": (ctypes.c_int, [_vp, _vp, _vp, _vp, _i32, _i64, _i32, _i32, _i32, _f32,
                                              _vp, _vp, _vp, _sz, _vp]),
    "mosaic_lse_merge": (ctypes.c_int, [_vp, _vp, _vp, _vp, _i64, _i32, _i32, _vp, _vp, _vp]),
    "mosaic_lse_merge_n": (ctypes.c_int, [_vp, _vp, _i32, _i64, _i32, _i32, _vp, _vp, _vp]),
    "mosaic_agg_prefill_attn_chunked_workspace_bytes": (_sz, [_i32, _i64, _i32, _i32, _i32, _i32]),
    "mosaic_agg_prefill_attn_chunked": (ctypes.c_int, [_vp, _vp, _vp, _vp, _i32, _i64, _i32, _i32,
                                                       _i32, _i32, _f32, _i32, _vp, _vp, _vp, _sz,
                                                       _vp]),
    "mosaic_agg_prefill_attn_shared_prefix_workspace_bytes": (_sz, [_i32, _i64, _i32, _i32, _i32]),
    "mosaic_agg_prefill_attn_shared_prefix": (ctypes.c_int, [_vp, _vp, _vp, _i32, _vp, _vp, _vp, _i32,
                                                             _i64, _i32, _i32, _i32, _i32, _f32, _vp,
                                                             _vp, _vp, _sz, _vp]),
    "mosaic_assemble_context": (ctypes.c_int, [_vp, _vp, _i32, _i32, _vp, _vp, _vp, _vp, _i32, _vp,
                                               _vp, _vp, _vp]),
    "mosaic_rope_packed": (ctypes.c_int, [_vp, _vp, _vp, _i64, _i32, _i32, _i32, _f32, _vp]),
    "mosaic_stage_host_arena_bytes": (_sz, [_i64, _i32, _i64, _i32, _i32, _i32]),
    "mosaic_stage_host": (ctypes.c_int, [_vp, _vp, _vp, _i64, _i32, _f32, _i32, _vp, _vp, _vp, _vp,
                                         _vp, _vp, _vp, _vp, _i32, _vp, _vp, _vp, _i64, _i32, _i32,
                                         _i32, _f32, _vp, _vp, _vp, _sz, _vp]),
    "mosaic_status_string": (ctypes.c_char_p, [ctypes.c_int]),
    "mosaic_version": (ctypes.c_int, []),
    "mosaic_last_cuda_error": (ctypes.c_int, []),
    "mosaic_kernel_launch_count": (_i64, []),
}

_lib = None


class MosaicError(RuntimeError):
    def __init__(self, call: str, status: int):
        lib = load()
        name = lib.mosaic_status_string(status).decode()
        extra = f" (cudaError {lib.mosaic_last_cuda_error()})" if status == ERR_CUDA else ""
        super().__init__(f"{call} failed: {name}{extra}")
        self.status = status


def load() -> ctypes.CDLL:
    """Loads libmosaic.so; raises if it has not been built (python -m paper_2606_03014_b200.build)."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise RuntimeError(f"{LIB_PATH} is missing: build it with "
                               "`python -m paper_2606_03014_b200.build` (no CPU fallback exists)")
        lib = ctypes.CDLL(str(LIB_PATH))
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def _check(call: str, status: int):
    if status != OK:
        raise MosaicError(call, status)


def _dptr(t: Optional[torch.Tensor], dtype=None, name="tensor"):
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError(f"{name} must be a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"{name} must be {dtype}, got {t.dtype}")
    return t.data_ptr()


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def version() -> int:
    return load().mosaic_version()


def kernel_launch_count() -> int:
    return int(load().mosaic_kernel_launch_count())


def gate(answers, tau, expert_conf=None, conf_mode=CONF_VOTE, *, want_count=True, want_agree=True,
         out=None, stream=None):
    """mosaic_gate.  answers int32 [Q,E] on the GPU.  Returns dict(mode,count,agree,conf,bypass)."""
    Q, E = answers.shape
    dev = answers.device
    o = out or {}
    mode = o.get("mode", torch.empty(Q, dtype=torch.int32, device=dev))
    count = o.get("count", torch.empty(Q, dtype=torch.int32, device=dev) if want_count else None)
    agree = o.get("agree", torch.empty(Q, dtype=torch.float32, device=dev) if want_agree else None)
    conf = o.get("conf", torch.empty(Q, dtype=torch.float32, device=dev))
    bypass = o.get("bypass", torch.empty(Q, dtype=torch.uint8, device=dev))
    st = load().mosaic_gate(_dptr(answers, torch.int32, "answers"),
                            _dptr(expert_conf, torch.float32, "expert_conf"), Q, E, float(tau),
                            conf_mode, _dptr(mode), _dptr(count), _dptr(agree), _dptr(conf),
                            _dptr(bypass), _stream(stream))
    _check("mosaic_gate", st)
    return dict(mode=mode, count=count, agree=agree, conf=conf, bypass=bypass)


def compact_workspace_bytes(Q: int) -> int:
    return int(load().mosaic_compact_workspace_bytes(Q))


def _compact_outputs(Q, dev, out):
    o = out or {}
    return dict(
        survivor_idx=o.get("survivor_idx", torch.empty(max(Q, 1), dtype=torch.int32, device=dev)),
        cu_seqlens=o.get("cu_seqlens", torch.empty(Q + 1, dtype=torch.int64, device=dev)),
        n_survivors=o.get("n_survivors", torch.empty(1, dtype=torch.int32, device=dev)),
        total_tokens=o.get("total_tokens", torch.empty(1, dtype=torch.int64, device=dev)),
        max_seqlen=o.get("max_seqlen", torch.empty(1, dtype=torch.int32, device=dev)),
        workspace=o.get("workspace", torch.empty(compact_workspace_bytes(Q), dtype=torch.uint8,
                                                 device=dev)))


def compact(bypass, ctx_len, *, out=None, stream=None):
    """mosaic_compact.  Returns device tensors (full-capacity survivor_idx / cu_seqlens plus the
    three device scalars); nothing is copied to the host."""
    Q = bypass.shape[0]
    r = _compact_outputs(Q, bypass.device, out)
    st = load().mosaic_compact(_dptr(bypass, torch.uint8, "bypass"),
                               _dptr(ctx_len, torch.int32, "ctx_len"), Q,
                               _dptr(r["survivor_idx"]), _dptr(r["cu_seqlens"]),
                               _dptr(r["n_survivors"]), _dptr(r["total_tokens"]),
                               _dptr(r["max_seqlen"]), _dptr(r["workspace"]),
                               r["workspace"].numel(), _stream(stream))
    _check("mosaic_compact", st)
    return r


COMPACT_STATIC_MAX_Q = 1 << 22


def compact_static(bypass, ctx_len, *, out, stream=None):
    """mosaic_compact_static: mosaic_compact with the scan state in the library's own device array.
    The call allocates nothing, so neither does this wrapper: `out` must hold survivor_idx [Q]
    int32, cu_seqlens [Q+1] int64 and the device scalars n_survivors, total_tokens, max_seqlen."""
    Q = bypass.shape[0]
    st = load().mosaic_compact_static(_dptr(bypass, torch.uint8, "bypass"),
                                      _dptr(ctx_len, torch.int32, "ctx_len"), Q,
                                      _dptr(out["survivor_idx"], torch.int32, "survivor_idx"),
                                      _dptr(out["cu_seqlens"], torch.int64, "cu_seqlens"),
                                      _dptr(out["n_survivors"], torch.int32, "n_survivors"),
                                      _dptr(out["total_tokens"], torch.int64, "total_tokens"),
                                      _dptr(out["max_seqlen"], torch.int32, "max_seqlen"),
                                      _stream(stream))
    _check("mosaic_compact_static", st)
    return out


def gate_compact(answers, ctx_len, tau, expert_conf=None, conf_mode=CONF_VOTE, *, want_count=False,
                 want_agree=False, want_bypass=True, out=None, stream=None):
    """mosaic_gate_compact: both steps in one launch."""
    Q, E = answers.shape
    dev = answers.device
    o = out or {}
    r = _compact_outputs(Q, dev, out)
    r["mode"] = o.get("mode", torch.empty(Q, dtype=torch.int32, device=dev))
    r["count"] = o.get("count", torch.empty(Q, dtype=torch.int32, device=dev) if want_count else None)
    r["agree"] = o.get("agree", torch.empty(Q, dtype=torch.float32, device=dev) if want_agree else None)
    r["conf"] = o.get("conf", torch.empty(Q, dtype=torch.float32, device=dev))
    r["bypass"] = o.get("bypass", torch.empty(Q, dtype=torch.uint8, device=dev) if want_bypass else None)
    st = load().mosaic_gate_compact(
        _dptr(answers, torch.int32, "answers"), _dptr(expert_conf, torch.float32, "expert_conf"),
        _dptr(ctx_len, torch.int32, "ctx_len"), Q, E, float(tau), conf_mode, _dptr(r["mode"]),
        _dptr(r["count"]), _dptr(r["agree"]), _dptr(r["conf"]), _dptr(r["bypass"]),
        _dptr(r["survivor_idx"]), _dptr(r["cu_seqlens"]), _dptr(r["n_survivors"]),
        _dptr(r["total_tokens"]), _dptr(r["max_seqlen"]), _dptr(r["workspace"]),
        r["workspace"].numel(), _stream(stream))
    _check("mosaic_gate_compact", st)
    return r


def gate_compact_tau(answers, ctx_len, tau_per_query, expert_conf=None, conf_mode=CONF_VOTE, *,
                     out=None, stream=None):
    """mosaic_gate_compact_tau: a threshold per question (fp32 [Q])."""
    Q, E = answers.shape
    dev = answers.device
    o = out or {}
    r = _compact_outputs(Q, dev, out)
    r["mode"] = o.get("mode", torch.empty(Q, dtype=torch.int32, device=dev))
    r["conf"] = o.get("conf", torch.empty(Q, dtype=torch.float32, device=dev))
    r["bypass"] = o.get("bypass", torch.empty(Q, dtype=torch.uint8, device=dev))
    st = load().mosaic_gate_compact_tau(
        _dptr(answers, torch.int32, "answers"), _dptr(expert_conf, torch.float32, "expert_conf"),
        _dptr(ctx_len, torch.int32, "ctx_len"), Q, E, _dptr(tau_per_query, torch.float32, "tau"),
        conf_mode, _dptr(r["mode"]), None, None, _dptr(r["conf"]), _dptr(r["bypass"]),
        _dptr(r["survivor_idx"]), _dptr(r["cu_seqlens"]), _dptr(r["n_survivors"]),
        _dptr(r["total_tokens"]), _dptr(r["max_seqlen"]), _dptr(r["workspace"]),
        r["workspace"].numel(), _stream(stream))
    _check("mosaic_gate_compact_tau", st)
    return r


def gate_compact_ext(answers, ctx_len, tau, expert_conf=None, conf_mode=CONF_VOTE, *,
                     tau_per_query=None, abstain_policy=ABSTAIN_NONE, abstain_label=-1,
                     want_count=True, want_agree=True, out=None, stream=None):
    """mosaic_gate_compact_ext: per-question thresholds, the weighted-argmax
    estimator and the abstention sentinel of a failed Extract, all optional, in one launch."""
    Q, E = answers.shape
    dev = answers.device
    o = out or {}
    r = _compact_outputs(Q, dev, out)
    r["mode"] = o.get("mode", torch.empty(Q, dtype=torch.int32, device=dev))
    r["count"] = o.get("count", torch.empty(Q, dtype=torch.int32, device=dev) if want_count else None)
    r["agree"] = o.get("agree", torch.empty(Q, dtype=torch.float32, device=dev) if want_agree else None)
    r["conf"] = o.get("conf", torch.empty(Q, dtype=torch.float32, device=dev))
    r["bypass"] = o.get("bypass", torch.empty(Q, dtype=torch.uint8, device=dev))
    st = load().mosaic_gate_compact_ext(
        _dptr(answers, torch.int32, "answers"), _dptr(expert_conf, torch.float32, "expert_conf"),
        _dptr(ctx_len, torch.int32, "ctx_len"), Q, E, float(tau),
        _dptr(tau_per_query, torch.float32, "tau_per_query"), conf_mode, int(abstain_policy),
        int(abstain_label), _dptr(r["mode"]), _dptr(r["count"]), _dptr(r["agree"]), _dptr(r["conf"]),
        _dptr(r["bypass"]), _dptr(r["survivor_idx"]), _dptr(r["cu_seqlens"]), _dptr(r["n_survivors"]),
        _dptr(r["total_tokens"]), _dptr(r["max_seqlen"]), _dptr(r["workspace"]),
        r["workspace"].numel(), _stream(stream))
    _check("mosaic_gate_compact_ext", st)
    return r


def conf_compact(conf, ctx_len, tau, *, tau_per_query=None, out=None, stream=None):
    """mosaic_conf_compact: threshold + compaction on a confidence C(q) the
    caller computed (fp32 [Q])."""
    Q = conf.shape[0]
    o = out or {}
    r = _compact_outputs(Q, conf.device, out)
    r["bypass"] = o.get("bypass", torch.empty(Q, dtype=torch.uint8, device=conf.device))
    st = load().mosaic_conf_compact(
        _dptr(conf, torch.float32, "conf"), _dptr(ctx_len, torch.int32, "ctx_len"), Q, float(tau),
        _dptr(tau_per_query, torch.float32, "tau_per_query"), _dptr(r["bypass"]),
        _dptr(r["survivor_idx"]), _dptr(r["cu_seqlens"]), _dptr(r["n_survivors"]),
        _dptr(r["total_tokens"]), _dptr(r["max_seqlen"]), _dptr(r["workspace"]),
        r["workspace"].numel(), _stream(stream))
    _check("mosaic_conf_compact", st)
    return r


def attn_workspace_bytes(n_seqs, total_tokens, Hq, Hkv, D) -> int:
    return int(load().mosaic_agg_prefill_attn_workspace_bytes(n_seqs, total_tokens, Hq, Hkv, D))


def agg_prefill_attn(q, k, v, cu_seqlens, n_seqs, max_seqlen, softmax_scale, *, o=None, lse=None,
                     workspace=None, stream=None):
    """mosaic_agg_prefill_attn.  q bf16 [T,Hq,D], k/v bf16 [T,Hkv,D], cu_seqlens int64 (device,
    at least n_seqs+1 entries).  Returns (o bf16 [T,Hq,D], lse fp32 [Hq,T])."""
    T, Hq, D = q.shape
    Hkv = k.shape[1]
    if k.shape != (T, Hkv, D) or v.shape != k.shape:
        raise ValueError("k/v shape")
    dev = q.device
    if o is None:
        o = torch.empty_like(q)
    if lse is None:
        lse = torch.empty((Hq, T), dtype=torch.float32, device=dev)
    if workspace is None:
        workspace = torch.empty(max(attn_workspace_bytes(n_seqs, T, Hq, Hkv, D), 16),
                                dtype=torch.uint8, device=dev)
    st = load().mosaic_agg_prefill_attn(
        _dptr(q, torch.bfloat16, "q"), _dptr(k, torch.bfloat16, "k"), _dptr(v, torch.bfloat16, "v"),
        _dptr(cu_seqlens, torch.int64, "cu_seqlens"), int(n_seqs), int(T), int(max_seqlen), Hq, Hkv,
        D, float(softmax_scale), _dptr(o, torch.bfloat16, "o"), _dptr(lse, torch.float32, "lse"),
        _dptr(workspace), workspace.numel(), _stream(stream))
    _check("mosaic_agg_prefill_attn", st)
    return o, lse


def agg_prefill_attn_kv(q, k, v, cu_seqlens_q, cu_seqlens_k, n_seqs, max_seqlen_q, softmax_scale, *,
                        causal=True, o=None, lse=None, workspace=None, stream=None):
    """mosaic_agg_prefill_attn_kv: q bf16 [Tq,Hq,D], k/v bf16 [Tk,Hkv,D],
    row i of a sequence sees keys j <= i + (Lk - Lq).  Returns (o bf16 [Tq,Hq,D], lse fp32 [Hq,Tq])."""
    Tq, Hq, D = q.shape
    Tk, Hkv = k.shape[0], k.shape[1]
    if k.shape != (Tk, Hkv, D) or v.shape != k.shape:
        raise ValueError("k/v shape")
    dev = q.device
    if o is None:
        o = torch.empty_like(q)
    if lse is None:
        lse = torch.empty((Hq, Tq), dtype=torch.float32, device=dev)
    if workspace is None:
        workspace = torch.empty(max(attn_workspace_bytes(n_seqs, Tq, Hq, Hkv, D), 16),
                                dtype=torch.uint8, device=dev)
    st = load().mosaic_agg_prefill_attn_kv(
        _dptr(q, torch.bfloat16, "q"), _dptr(k, torch.bfloat16, "k"), _dptr(v, torch.bfloat16, "v"),
        _dptr(cu_seqlens_q, torch.int64, "cu_seqlens_q"), _dptr(cu_seqlens_k, torch.int64, "cu_seqlens_k"),
        int(n_seqs), int(Tq), int(Tk), int(max_seqlen_q), Hq, Hkv, D, float(softmax_scale),
        1 if causal else 0, _dptr(o, torch.bfloat16, "o"), _dptr(lse, torch.float32, "lse"),
        _dptr(workspace), workspace.numel(), _stream(stream))
    _check("mosaic_agg_prefill_attn_kv", st)
    return o, lse


def agg_decode_attn(q, k, v, cu_seqlens_k, softmax_scale, *, o=None, lse=None, workspace=None,
                    stream=None):
    """mosaic_agg_decode_attn: q bf16 [n_seqs,Hq,D] (one token per sequence) against k/v bf16
    [Tk,Hkv,D].  Returns (o bf16 [n_seqs,Hq,D], lse fp32 [Hq,n_seqs])."""
    n, Hq, D = q.shape
    Tk, Hkv = k.shape[0], k.shape[1]
    dev = q.device
    if o is None:
        o = torch.empty_like(q)
    if lse is None:
        lse = torch.empty((Hq, n), dtype=torch.float32, device=dev)
    if workspace is None:
        nb = int(load().mosaic_agg_decode_attn_workspace_bytes(n, Tk, Hq, Hkv, D))
        workspace = torch.empty(max(nb, 16), dtype=torch.uint8, device=dev)
    st = load().mosaic_agg_decode_attn(
        _dptr(q, torch.bfloat16, "q"), _dptr(k, torch.bfloat16, "k"), _dptr(v, torch.bfloat16, "v"),
        _dptr(cu_seqlens_k, torch.int64, "cu_seqlens_k"), int(n), int(Tk), Hq, Hkv, D,
        float(softmax_scale), _dptr(o, torch.bfloat16, "o"), _dptr(lse, torch.float32, "lse"),
        _dptr(workspace), workspace.numel(), _stream(stream))
    _check("mosaic_agg_decode_attn", st)
    return o, lse


def lse_merge(o_a, lse_a, o_b, lse_b, *, o=None, lse=None, stream=None):
    """mosaic_lse_merge: partial results over two disjoint key sets -> the result over their union."""
    T, Hq, D = o_a.shape
    if o is None:
        o = torch.empty_like(o_a)
    if lse is None:
        lse = torch.empty_like(lse_a)
    st = load().mosaic_lse_merge(_dptr(o_a, torch.bfloat16, "o_a"), _dptr(lse_a, torch.float32, "lse_a"),
                                 _dptr(o_b, torch.bfloat16, "o_b"), _dptr(lse_b, torch.float32, "lse_b"),
                                 int(T), Hq, D, _dptr(o, torch.bfloat16, "o"),
                                 _dptr(lse, torch.float32, "lse"), _stream(stream))
    _check("mosaic_lse_merge", st)
    return o, lse


def lse_merge_n(o_parts, lse_parts, *, o=None, lse=None, stream=None):
    """mosaic_lse_merge_n: o_parts bf16 [n, T, Hq, D], lse_parts fp32 [n, Hq, T] -> (o, lse)."""
    n, T, Hq, D = o_parts.shape
    if o is None:
        o = torch.empty((T, Hq, D), dtype=torch.bfloat16, device=o_parts.device)
    if lse is None:
        lse = torch.empty((Hq, T), dtype=torch.float32, device=o_parts.device)
    st = load().mosaic_lse_merge_n(_dptr(o_parts, torch.bfloat16, "o_parts"),
                                   _dptr(lse_parts, torch.float32, "lse_parts"), int(n), int(T), Hq, D,
                                   _dptr(o, torch.bfloat16, "o"), _dptr(lse, torch.float32, "lse"),
                                   _stream(stream))
    _check("mosaic_lse_merge_n", st)
    return o, lse


def agg_prefill_attn_chunked(q, k, v, cu_seqlens, n_seqs, max_seqlen, softmax_scale, q_chunk, *,
                             o=None, lse=None, workspace=None, stream=None):
    """mosaic_agg_prefill_attn_chunked: the plain prefill with every sequence taken in chunks of
    q_chunk query rows, all chunks in one launch."""
    T, Hq, D = q.shape
    Hkv = k.shape[1]
    dev = q.device
    if o is None:
        o = torch.empty_like(q)
    if lse is None:
        lse = torch.empty((Hq, T), dtype=torch.float32, device=dev)
    if workspace is None:
        nb = int(load().mosaic_agg_prefill_attn_chunked_workspace_bytes(int(n_seqs), T, int(q_chunk),
                                                                        Hq, Hkv, D))
        workspace = torch.empty(max(nb, 16), dtype=torch.uint8, device=dev)
    st = load().mosaic_agg_prefill_attn_chunked(
        _dptr(q, torch.bfloat16, "q"), _dptr(k, torch.bfloat16, "k"), _dptr(v, torch.bfloat16, "v"),
        _dptr(cu_seqlens, torch.int64, "cu_seqlens"), int(n_seqs), int(T), int(max_seqlen), Hq, Hkv, D,
        float(softmax_scale), int(q_chunk), _dptr(o, torch.bfloat16, "o"),
        _dptr(lse, torch.float32, "lse"), _dptr(workspace), workspace.numel(), _stream(stream))
    _check("mosaic_agg_prefill_attn_chunked", st)
    return o, lse


def agg_prefill_attn_shared_prefix(q, k_prefix, v_prefix, k, v, cu_seqlens, n_seqs, max_seqlen,
                                   softmax_scale, *, o=None, lse=None, workspace=None, stream=None):
    """mosaic_agg_prefill_attn_shared_prefix: every sequence = the shared block k_prefix / v_prefix
    bf16 [P, Hkv, D] followed by its own tokens (q, k, v packed by cu_seqlens)."""
    T, Hq, D = q.shape
    Hkv = k.shape[1]
    P = 0 if k_prefix is None else k_prefix.shape[0]
    dev = q.device
    if o is None:
        o = torch.empty_like(q)
    if lse is None:
        lse = torch.empty((Hq, T), dtype=torch.float32, device=dev)
    if workspace is None:
        nb = int(load().mosaic_agg_prefill_attn_shared_prefix_workspace_bytes(int(n_seqs), T, Hq, Hkv, D))
        workspace = torch.empty(max(nb, 16), dtype=torch.uint8, device=dev)
    st = load().mosaic_agg_prefill_attn_shared_prefix(
        _dptr(q, torch.bfloat16, "q"), _dptr(k_prefix, torch.bfloat16, "k_prefix"),
        _dptr(v_prefix, torch.bfloat16, "v_prefix"), int(P), _dptr(k, torch.bfloat16, "k"),
        _dptr(v, torch.bfloat16, "v"), _dptr(cu_seqlens, torch.int64, "cu_seqlens"), int(n_seqs),
        int(T), int(max_seqlen), Hq, Hkv, D, float(softmax_scale), _dptr(o, torch.bfloat16, "o"),
        _dptr(lse, torch.float32, "lse"), _dptr(workspace), workspace.numel(), _stream(stream))
    _check("mosaic_agg_prefill_attn_shared_prefix", st)
    return o, lse


def assemble_context(survivor_idx, cu_seqlens, n_survivors, max_seqlen, total_tokens,
                     prompt_tokens, prompt_off, trace_tokens, trace_off, E, *, input_ids=None,
                     position_ids=None, n_mismatch=None, stream=None):
    """mosaic_assemble_context.  All tensors on the device; returns
    (input_ids int32 [total_tokens], position_ids int32 [total_tokens], n_mismatch int32 [1])."""
    dev = cu_seqlens.device
    if input_ids is None:
        input_ids = torch.empty(max(int(total_tokens), 1), dtype=torch.int32, device=dev)
    if position_ids is None:
        position_ids = torch.empty(max(int(total_tokens), 1), dtype=torch.int32, device=dev)
    if n_mismatch is None:
        n_mismatch = torch.empty(1, dtype=torch.int32, device=dev)
    st = load().mosaic_assemble_context(
        _dptr(survivor_idx, torch.int32, "survivor_idx"), _dptr(cu_seqlens, torch.int64, "cu_seqlens"),
        int(n_survivors), int(max_seqlen), _dptr(prompt_tokens, torch.int32, "prompt_tokens"),
        _dptr(prompt_off, torch.int64, "prompt_off"), _dptr(trace_tokens, torch.int32, "trace_tokens"),
        _dptr(trace_off, torch.int64, "trace_off"), int(E), _dptr(input_ids, torch.int32, "input_ids"),
        _dptr(position_ids, torch.int32, "position_ids"), _dptr(n_mismatch, torch.int32, "n_mismatch"),
        _stream(stream))
    _check("mosaic_assemble_context", st)
    return input_ids[:int(total_tokens)], position_ids[:int(total_tokens)], n_mismatch


def rope_packed(q, k, position_ids, theta, *, stream=None):
    """mosaic_rope_packed: rotates q bf16 [T,Hq,D] and k bf16 [T,Hkv,D] in place by position_ids."""
    T, Hq, D = q.shape
    Hkv = k.shape[1]
    st = load().mosaic_rope_packed(_dptr(q, torch.bfloat16, "q"), _dptr(k, torch.bfloat16, "k"),
                                   _dptr(position_ids, torch.int32, "position_ids"), int(T), Hq, Hkv,
                                   D, float(theta), _stream(stream))
    _check("mosaic_rope_packed", st)
    return q, k


def stage_host_arena_bytes(Q, E, T_cap, Hq, Hkv, D) -> int:
    return int(load().mosaic_stage_host_arena_bytes(Q, E, T_cap, Hq, Hkv, D))


def _hptr(t: Optional[torch.Tensor], name="tensor"):
    if t is None:
        return None
    if t.is_cuda or not t.is_contiguous():
        raise ValueError(f"{name} must be a contiguous host tensor")
    return t.data_ptr()


def stage_host(answers_h, expert_conf_h, ctx_len_h, tau, conf_mode, q_h, k_h, v_h, softmax_scale,
               *, max_attn_seqs=-1, out_h=None, arena=None, stream=None):
    """mosaic_stage_host: the whole stage from (ideally pinned) host tensors; synchronous.
    out_h may carry preallocated pinned host outputs.  Returns the dict of host outputs."""
    Q, E = answers_h.shape
    T_cap, Hq, D = q_h.shape
    Hkv = k_h.shape[1]
    o = dict(out_h or {})

    def host(name, shape, dtype):
        if name not in o:
            o[name] = torch.empty(shape, dtype=dtype)
        return o[name]

    host("mode", Q, torch.int32)
    host("conf", Q, torch.float32)
    host("bypass", Q, torch.uint8)
    host("survivor_idx", max(Q, 1), torch.int32)
    host("cu_seqlens", Q + 1, torch.int64)
    host("n_survivors", 1, torch.int32)
    host("total_tokens", 1, torch.int64)
    host("max_seqlen", 1, torch.int32)
    host("o", (T_cap, Hq, D), torch.bfloat16)
    host("lse", Hq * T_cap, torch.float32)
    if arena is None:
        arena = torch.empty(stage_host_arena_bytes(Q, E, T_cap, Hq, Hkv, D), dtype=torch.uint8,
                            device="cuda")
    st = load().mosaic_stage_host(
        _hptr(answers_h), _hptr(expert_conf_h), _hptr(ctx_len_h), Q, E, float(tau), conf_mode,
        _hptr(o["mode"]), _hptr(o["conf"]), _hptr(o["bypass"]), _hptr(o["survivor_idx"]),
        _hptr(o["cu_seqlens"]), _hptr(o["n_survivors"]), _hptr(o["total_tokens"]),
        _hptr(o["max_seqlen"]), int(max_attn_seqs), _hptr(q_h), _hptr(k_h), _hptr(v_h), T_cap, Hq,
        Hkv, D, float(softmax_scale), _hptr(o["o"]), _hptr(o["lse"]), _dptr(arena), arena.numel(),
        _stream(stream))
    _check("mosaic_stage_host", st)
    return o
