"""Slab domain decomposition with halos (paper_1901_08088_b200/sharded.py: SlabNeighborList; SURVEY §8e/§8f NEXT-4 second
half) on CPU: world_size 2 and 3 over gloo with a stand-in backend that answers from the CPU oracle.
Tested: the neighbor exchange (P2P, unequal counts, both faces to one peer at world 2), that every rank's local set is
exactly own + the particles within the halo of its faces, that the merged lists are the single-process oracle's — with
particles placed exactly on slab faces and pairs across the periodic edge of the cut axis — and the refusal of slabs
thinner than the halo."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


class OracleSlabBackend:
    """CPU stand-in for sharded.CudaSlabBackend: lists of the first n_rows particles of the local set, from the oracle."""

    def build(self, pos, type, box, n_global):
        self.pos = pos.numpy().astype(np.float32)
        self.type = None if type is None else type.numpy().astype(np.int32)
        self.box = np.asarray(box, np.float32)
        return 0

    def neighbors_rows(self, r_list, n_rows):
        from oracle import neighbors as ON
        rp, nb, _ = ON.neighbor_list(self.pos, self.type, self.box, r_list, method="brute")
        cnt = np.diff(rp)[:n_rows]
        cap = max(int(cnt.max()) if n_rows else 0, 1) + 3
        nlist = np.full((n_rows, cap), 12345678, np.int32)             # garbage beyond the count, as the CUDA path leaves it
        for i in range(n_rows):
            nlist[i, : cnt[i]] = nb[rp[i]:rp[i + 1]]
        return torch.from_numpy(cnt.astype(np.int32)), torch.from_numpy(nlist), int(cnt.max()) if n_rows else 0


def _workload():
    """Two types in a box whose longest edge is y; particles exactly on the slab faces of world 2 and 3 and on the box faces."""
    from paper_1901_08088_b200 import workloads as W
    rng = np.random.default_rng(17)
    L = np.array([9.0, 18.0, 10.0])
    N = 1400
    p = rng.random((N, 3)) * L
    for k, y in enumerate([0.0, 6.0, 9.0, 12.0, 18.0 - 2.0 ** -18, 5.999999, 9.000001]):
        p[k, 1] = y                                                    # on / next to the faces at L/3, L/2, 2L/3 and the box edge
        p[k + 10] = p[k] + np.array([0.3, -0.9, 0.2])                  # a partner across that face
    p = np.mod(p, L)
    pos, box = W._finish(p, L)
    typ = (rng.random(N) < 0.2).astype(np.int32)
    r = np.array([[1.3, 1.7], [1.7, 2.2]], np.float32)
    return pos, typ, box, r


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1901_08088_b200 import sharded
    pos, typ, box, r = _workload()
    snl = sharded.SlabNeighborList(box, r, T=2, device="cpu", backend=OracleSlabBackend())
    mine = np.nonzero(sharded.slab_index(pos, box, world, snl.axis) == rank)[0]
    snl.build(torch.from_numpy(pos[mine]), torch.from_numpy(typ[mine]), torch.from_numpy(mine.astype(np.int64)), len(pos))
    own, ghosts = sharded.local_set_indices(pos, box, world, rank, snl.h)
    local_ok = bool(np.array_equal(snl.gid[: snl.n_own].numpy(), own) and
                    np.array_equal(np.sort(snl.gid[snl.n_own:].numpy()), np.sort(ghosts)) and
                    np.array_equal(snl.pos.numpy(), pos[snl.gid.numpy()]) and np.array_equal(snl.type.numpy(), typ[snl.gid.numpy()]))
    gid, n_neigh, nlist, M = snl.neighbors()
    out.put((rank, local_ok, gid.numpy(), n_neigh.numpy(), nlist.numpy(), M, snl.n_ghost, snl.halo_bytes, snl.axis))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,port", [(2, 29751), (3, 29753)])
def test_slab_lists_merge_to_the_single_process_oracle_gloo(world, port):
    from oracle import neighbors as ON
    from paper_1901_08088_b200 import sharded
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((out.get(timeout=240) for _ in range(world)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    pos, typ, box, r = _workload()
    N = len(pos)
    assert all(x[1] for x in res)                                      # every rank holds exactly own + halo, unshifted
    assert all(x[8] == 1 for x in res)                                 # cut along y, the longest edge
    assert all(0 < x[6] < N for x in res) and all(x[7] > 0 for x in res)
    n_all, l_all = sharded.merge_slices(N, [(x[2], x[3], x[4]) for x in res])     # raises unless every particle has one owner
    rp, nb, _ = ON.neighbor_list(pos, typ, box, r, method="brute")
    assert np.array_equal(n_all, np.diff(rp))
    for i in range(N):
        assert np.array_equal(np.sort(l_all[i, : n_all[i]]), nb[rp[i]:rp[i + 1]]), i
    assert len({x[5] for x in res}) == 1 and res[0][5] == int(np.diff(rp).max())
    # the halo is a fraction of the system, not all of it (world 3: two faces of 18/3 = 6 wide slabs, h ~ 2.2)
    assert sum(x[6] for x in res) < (1.0 if world == 2 else 0.9) * N * 2 * 2.3 / (18.0 / world) + 50


def test_slab_geometry_and_refusals():
    from paper_1901_08088_b200 import sharded
    box = np.array([0, 0, 0, 9, 18, 10], np.float32)
    h = sharded.halo_width(np.array([[2.2]]))
    assert 2.2 < h < 2.21
    assert sharded.slab_geometry(box, 3, h) == (1, 6.0)
    with pytest.raises(ValueError):
        sharded.slab_geometry(box, 9, h)                               # 2-wide slabs, 2.2 halo: ghosts from second neighbors
    assert sharded.slab_geometry(box, 1, 100.0)[0] == 1                # a single rank has no halo to worry about
    pos = np.array([[1, 0.0, 1], [1, 5.9999, 1], [1, 6.0, 1], [1, 17.99, 1], [1, 18.0, 1]], np.float32)
    assert sharded.slab_index(pos, box, 3, 1).tolist() == [0, 0, 1, 2, 2]          # a face belongs to the upper slab; the box edge clamps
    for world in (1, 2, 3, 4):
        pts = np.random.default_rng(world).random((500, 3)).astype(np.float32) * box[3:]
        seen = np.zeros(500, int)
        for g in range(world):
            own, ghosts = sharded.local_set_indices(pts, box, world, g, h)
            seen[own] += 1
            assert len(np.intersect1d(own, ghosts)) == 0 and len(np.unique(ghosts)) == len(ghosts)
        assert np.all(seen == 1)
