"""The N > 1 path of bench.py on CPU: two gloo ranks, each with its own seeded batch (weak
scaling, no data-path collective); the only communication is the whole-job aggregation
(max over ranks of the time, sum over ranks of the work).  DESIGN.md section 8."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from conftest import ROOT

sys.path.insert(0, str(ROOT))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import oracle
    from paper_2606_03014_b200 import workloads as wl
    cfg = wl.C1
    gi = wl.gate_inputs(cfg, bench.rank_seed(rank))      # each rank: its own batch
    oc = oracle.compact(oracle.gate(gi.answers, gi.tau)["bypass"], gi.ctx_len)
    flops = bench.attn_flops(np.diff(oc["cu_seqlens"]), cfg.Hq, cfg.D)
    secs = 1.0 + rank                                     # rank 1 is the slow one
    secs_max, flops_all = bench.whole_job(secs, flops, world)
    out[rank] = (secs_max, flops_all, flops, int(oc["n_survivors"]))
    dist.destroy_process_group()


def test_two_ranks_whole_job_aggregate():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        r0, r1 = out[0], out[1]
    assert r0[0] == r1[0] == 2.0                          # max over ranks
    assert r0[1] == r1[1] == r0[2] + r1[2]                # sum over ranks
    assert r0[2] != r1[2] or r0[3] != r1[3]               # different batches per rank


def test_single_rank_is_identity():
    import bench
    assert bench.whole_job(0.5, 7.0, 1) == (0.5, 7.0)


def _spawned(out):
    """What bench.py --gpus N runs in every rank it starts itself, on gloo: the environment that
    spawn_ranks sets up is the one torchrun would have set."""
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    assert int(os.environ["LOCAL_RANK"]) == rank and os.environ["MASTER_ADDR"] == "127.0.0.1"
    dist.init_process_group("gloo")
    import bench
    out[rank] = bench.whole_job(1.0 + rank, 10.0 * (rank + 1), world)
    dist.destroy_process_group()


def test_bench_spawns_its_own_ranks():
    """`bench.py --gpus N` without a launcher starts N ranks itself (bench.spawn_ranks)."""
    import bench
    with mp.Manager() as m:
        out = m.dict()
        bench.spawn_ranks(2, _spawned, (out,))
        assert out[0] == out[1] == (2.0, 30.0)


def test_gpus_flag_must_match_the_world_size():
    """A rank whose --gpus differs from WORLD_SIZE refuses to run (no N-labelled single-GPU line)."""
    import subprocess
    env = dict(os.environ, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--gpus", "2", "--steps", "1"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode != 0 and "WORLD_SIZE" in (r.stderr + r.stdout)
