"""Host logic of bench.py that needs no GPU: the replica (N > 1) reduction over ranks, with gloo, world_size 2."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_1901_08088_b200 import workloads as W
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world)           # rank 1 is the slow one
    w = W.lj_uniform(N=512, seed=rank)                             # replicas: each rank its own seeded input
    out.put((rank, ms, bench.whole_job_value(ms, w.N, world), float(w.pos.sum())))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_max_over_ranks_gloo():
    world, port = 2, 29731
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [15.0, 15.0]                     # every rank reports the slowest rank's time
    assert res[0][2] == pytest.approx(1e6 * 15.0 / (512 * 2))      # whole-job ns/particle: all ranks' particles
    assert res[0][3] != res[1][3]                                  # different seeds per rank


def test_single_rank_is_identity():
    import bench
    assert bench.max_over_ranks(3.25, 1) == 3.25
    assert bench.whole_job_value(1.0, 1000, 1) == pytest.approx(1000.0)
