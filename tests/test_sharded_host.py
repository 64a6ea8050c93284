"""Host logic of the query-sharded multi-GPU path (paper_1901_08088_b200/sharded.py) on CPU:
world_size 2 and 3 over gloo.  The CUDA backend is replaced by a stand-in that answers from the CPU oracle, so what is
tested is the plumbing: the all-gather of unequal blocks, the Z-order slices, and that the slices merge into exactly the
single-process list."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


class OracleBackend:
    """CPU stand-in for sharded.CudaBackend: same interface, lists from the oracle, Z-order from the oracle's tree."""

    def __init__(self):
        pass

    def build(self, pos, type, box):
        from oracle import tree as OT
        self.pos = pos.numpy().astype(np.float32)
        self.type = None if type is None else type.numpy().astype(np.int32)
        self.box = np.asarray(box, np.float32)
        T = 1 if self.type is None else int(self.type.max()) + 1
        self.perm = OT.build(self.pos, self.type, self.box, T=T).perm
        return 0

    def neighbors_range(self, r_list, first, count):
        from oracle import neighbors as ON
        rp, nb, _ = ON.neighbor_list(self.pos, self.type, self.box, r_list, method="brute")
        cnt = np.diff(rp)
        rows = self.perm[first:first + count]
        cap = max(int(cnt.max()), 1)
        nlist = np.full((count, cap), -1, np.int32)
        for k, i in enumerate(rows):
            nlist[k, : cnt[i]] = nb[rp[i]:rp[i + 1]]
        M = int(cnt[rows].max()) if count else 0
        return torch.from_numpy(rows.astype(np.int64)), torch.from_numpy(cnt[rows].astype(np.int32)), torch.from_numpy(nlist), M


def _workload(N=1501):
    from paper_1901_08088_b200 import workloads as W
    w = W.colloid_solvent(N=N, n_colloid=7, seed=3)                 # two types, three cutoffs; 1501: an N no world size divides
    return w


def _worker(rank, world, port, out, N=1501):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1901_08088_b200 import sharded
    w = _workload(N)
    snl = sharded.ShardedNeighborList(w.N, T=w.T, max_neigh=8, device="cpu", backend=OracleBackend())
    lo, cnt = snl.own_first, snl.own_count
    snl.build(torch.from_numpy(w.pos[lo:lo + cnt] + 1.0), torch.from_numpy(w.type[lo:lo + cnt]), w.box)   # a first step ...
    first_pos = snl.pos
    snl.build(torch.from_numpy(w.pos[lo:lo + cnt]), torch.from_numpy(w.type[lo:lo + cnt]), w.box)         # ... and the next
    assert snl.pos is first_pos                                      # gathered into the same persistent tensor, no new one per step
    gathered_ok = bool(np.array_equal(snl.pos.numpy(), w.pos) and np.array_equal(snl.type.numpy(), w.type))
    rows, n_neigh, nlist, M = snl.neighbors(w.r_list)
    out.put((rank, gathered_ok, snl.first, snl.count, rows.numpy(), n_neigh.numpy(), nlist.numpy(), M))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,port,N", [(2, 29741, 1501), (3, 29743, 1501), (2, 29745, 1500)])   # 1500 / 2: equal blocks, gathered in place
def test_sharded_slices_merge_to_the_full_list_gloo(world, port, N):
    from oracle import neighbors as ON
    from paper_1901_08088_b200 import sharded
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out, N)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((out.get(timeout=180) for _ in range(world)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = _workload(N)
    assert all(r[1] for r in res)                                               # the all-gather rebuilt pos and type
    assert [r[2] for r in res] == [sharded.slice_bounds(w.N, world, g)[0] for g in range(world)]
    assert sum(r[3] for r in res) == w.N and max(r[3] for r in res) - min(r[3] for r in res) <= 1
    n_all, l_all = sharded.merge_slices(w.N, [(r[4], r[5], r[6]) for r in res])
    rp, nb, _ = ON.neighbor_list(w.pos, w.type, w.box, w.r_list, method="brute")
    assert np.array_equal(n_all, np.diff(rp))
    for i in range(w.N):
        assert np.array_equal(np.sort(l_all[i, : n_all[i]]), nb[rp[i]:rp[i + 1]])
    assert len({r[7] for r in res}) == 1 and res[0][7] == int(np.diff(rp).max())   # every rank knows the global maximum


def test_slice_arithmetic_and_merge_errors():
    from paper_1901_08088_b200 import sharded
    for N in (0, 1, 7, 1000, 1 << 20):
        for world in (1, 2, 3, 8):
            b = [sharded.slice_bounds(N, world, g) for g in range(world)]
            assert b[0][0] == 0 and sum(c for _, c in b) == N
            assert all(b[g][0] + b[g][1] == b[g + 1][0] for g in range(world - 1))
    with pytest.raises(ValueError):
        sharded.merge_slices(3, [(np.array([0, 1]), np.zeros(2, np.int32), np.zeros((2, 1), np.int32))])   # particle 2 missing
