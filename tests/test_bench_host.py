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


def test_both_arms_print_the_same_config_keys():
    import bench
    from paper_1901_08088_b200 import workloads as W
    w = W.make_config(1)
    a, b = bench.config_keys(1, w), bench.config_keys(1, W.make_config(1))
    assert a == b and set(a) == {"workload", "N", "types", "r_list", "max_neigh"}


def test_stored_ncu_counters_belong_to_the_current_traversal_kernel():
    """bench.py quotes counters of one ncu capture (profiles/traverse_ncu_counters.txt: DRAM bytes, instructions, pipe
    utilisation).  They describe the kernel as of their `commit=` stamp: that commit must contain the last change to
    traverse_kernels.cu, and the file must not be modified beyond it — otherwise re-capture before quoting."""
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    if not os.path.isdir(os.path.join(root, ".git")):
        pytest.skip("no git history here")
    kern = "paper_1901_08088_b200/csrc/traverse_kernels.cu"
    git = lambda *a: subprocess.run(["git", "-C", root, *a], capture_output=True, text=True)
    fields = dict(tok.split("=", 1) for tok in open(os.path.join(root, "profiles", "traverse_ncu_counters.txt")).read().split())
    last = git("log", "-1", "--format=%H", "--", kern).stdout.strip()
    assert last and fields.get("commit")
    assert git("merge-base", "--is-ancestor", last, fields["commit"]).returncode == 0, (last, fields["commit"])
    assert git("diff", "--quiet", "HEAD", "--", kern).returncode == 0, "traverse_kernels.cu has uncommitted changes"
    for k in ("dram_bytes", "inst_executed", "issue_active_pct", "lsu_data_pipe_pct", "shared_wavefronts", "shared_bank_conflicts"):
        assert float(fields[k]) > 0
