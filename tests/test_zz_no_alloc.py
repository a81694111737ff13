"""mosaic_compact_static: the compaction (G4-G5) with its scan state in the library's own static
device array, for callers that cannot allocate device memory.  Checked against the existing path
(mosaic_compact with a caller workspace) -- integer / index work, so bit for bit, the bar every
compaction test here uses -- on two calls in a row that share the array, and against the oracle.
This file is collected last on purpose (pytest -x: a failure here hides nothing after it); it
passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from paper_2606_03014_b200 import mosaic

pytestmark = pytest.mark.gpu


def _inputs(Q, p_bypass, seed):
    g = np.random.default_rng(seed)
    bypass = (g.random(Q) < p_bypass).astype(np.uint8)
    ctx_len = g.integers(0, 40000, size=Q).astype(np.int32)
    return bypass, ctx_len


def _outputs(Q, fill):
    dev = "cuda"
    # pre-filled, so that an entry the call should have written and did not shows up
    return dict(survivor_idx=torch.full((max(Q, 1),), fill, dtype=torch.int32, device=dev),
                cu_seqlens=torch.full((Q + 1,), fill, dtype=torch.int64, device=dev),
                n_survivors=torch.full((1,), fill, dtype=torch.int32, device=dev),
                total_tokens=torch.full((1,), fill, dtype=torch.int64, device=dev),
                max_seqlen=torch.full((1,), fill, dtype=torch.int32, device=dev))


def _same(a, b, S):
    assert int(a["n_survivors"]) == int(b["n_survivors"]) == S
    assert int(a["total_tokens"]) == int(b["total_tokens"])
    assert int(a["max_seqlen"]) == int(b["max_seqlen"])
    assert torch.equal(a["survivor_idx"][:S], b["survivor_idx"][:S])
    assert torch.equal(a["cu_seqlens"][:S + 1], b["cu_seqlens"][:S + 1])


def test_two_calls_in_a_row_match_the_workspace_path():
    # two different problems back to back on one stream: the second call finds the first one's
    # scan state (ticket, tile prefixes of a LARGER problem) in the shared array and must clear it
    cases = [(777_777, 0.3, 1), (100_001, 0.9, 2)]
    dev_in, got = [], []
    for Q, pb, seed in cases:
        bypass, ctx_len = _inputs(Q, pb, seed)
        b, c = torch.from_numpy(bypass).cuda(), torch.from_numpy(ctx_len).cuda()
        dev_in.append((bypass, ctx_len, b, c))
    for (Q, _, _), (_, _, b, c) in zip(cases, dev_in):        # the two static calls, nothing between
        got.append(mosaic.compact_static(b, c, out=_outputs(Q, -7)))
    torch.cuda.synchronize()
    for (Q, _, _), (bypass, ctx_len, b, c), g in zip(cases, dev_in, got):
        want = oracle.compact(bypass, ctx_len)
        S = want["n_survivors"]
        ref = mosaic.compact(b, c)                             # the existing path
        torch.cuda.synchronize()
        _same(g, ref, S)
        assert np.array_equal(g["survivor_idx"][:S].cpu().numpy(), want["survivor_idx"])
        assert np.array_equal(g["cu_seqlens"][:S + 1].cpu().numpy(), want["cu_seqlens"])
        assert int(g["total_tokens"]) == want["total_tokens"]
        assert int(g["max_seqlen"]) == want["max_seqlen"]
        # nothing past the survivors was written
        assert bool((g["survivor_idx"][S:] == -7).all()) and bool((g["cu_seqlens"][S + 1:] == -7).all())


def test_same_problem_twice_and_edges():
    Q = 50_000
    bypass, ctx_len = _inputs(Q, 0.5, 3)
    b, c = torch.from_numpy(bypass).cuda(), torch.from_numpy(ctx_len).cuda()
    first = mosaic.compact_static(b, c, out=_outputs(Q, -1))
    second = mosaic.compact_static(b, c, out=_outputs(Q, -1))
    ref = mosaic.compact(b, c)
    torch.cuda.synchronize()
    S = int(ref["n_survivors"])
    _same(first, ref, S)
    _same(second, ref, S)
    # all bypassed, none bypassed, one question, no question
    for Qe, pb in ((4097, 1.1), (4097, -1.0), (1, -1.0), (0, 0.5)):
        bypass, ctx_len = _inputs(Qe, pb, 4)
        b, c = torch.from_numpy(bypass).cuda(), torch.from_numpy(ctx_len).cuda()
        g = mosaic.compact_static(b, c, out=_outputs(Qe, -1))
        torch.cuda.synchronize()
        want = oracle.compact(bypass, ctx_len)
        S = want["n_survivors"]
        assert int(g["n_survivors"]) == S and int(g["total_tokens"]) == want["total_tokens"]
        assert int(g["max_seqlen"]) == want["max_seqlen"]
        assert np.array_equal(g["survivor_idx"][:S].cpu().numpy(), want["survivor_idx"])
        assert np.array_equal(g["cu_seqlens"][:S + 1].cpu().numpy(), want["cu_seqlens"])


def test_maximum_size_and_beyond():
    Qmax = mosaic.COMPACT_STATIC_MAX_Q
    bypass, ctx_len = _inputs(Qmax, 0.4, 5)
    b, c = torch.from_numpy(bypass).cuda(), torch.from_numpy(ctx_len).cuda()
    g = mosaic.compact_static(b, c, out=_outputs(Qmax, -1))
    ref = mosaic.compact(b, c)
    torch.cuda.synchronize()
    _same(g, ref, int(ref["n_survivors"]))
    assert int(g["total_tokens"]) > 2 ** 31                    # int64 totals, as in the plain path
    # one question more is refused, with the status that says why, before anything is launched
    b1 = torch.zeros(Qmax + 1, dtype=torch.uint8, device="cuda")
    c1 = torch.zeros(Qmax + 1, dtype=torch.int32, device="cuda")
    out = _outputs(Qmax + 1, -5)
    with pytest.raises(mosaic.MosaicError) as e:
        mosaic.compact_static(b1, c1, out=out)
    assert e.value.status == mosaic.ERR_WORKSPACE_TOO_SMALL
    torch.cuda.synchronize()
    assert int(out["n_survivors"]) == -5


def test_replays_inside_a_cuda_graph():
    """What the entry point is for: after one ordinary call (which asks for the array's address), the
    call is captured into a CUDA graph -- where allocating is not allowed -- and replayed."""
    Q = 300_000
    bypass, ctx_len = _inputs(Q, 0.6, 6)
    b, c = torch.from_numpy(bypass).cuda(), torch.from_numpy(ctx_len).cuda()
    out = _outputs(Q, -1)
    mosaic.compact_static(b, c, out=out)                       # warm-up, outside the capture
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            mosaic.compact_static(b, c, out=out, stream=side)
    torch.cuda.current_stream().wait_stream(side)
    ref = mosaic.compact(b, c)
    torch.cuda.synchronize()
    S = int(ref["n_survivors"])
    for _ in range(2):
        for t in out.values():
            t.fill_(-1)
        graph.replay()
        torch.cuda.synchronize()
        _same(out, ref, S)
