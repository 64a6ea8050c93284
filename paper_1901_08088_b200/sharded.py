"""Multi-GPU query sharding ("straightforwardly generalized to execute on
multiple GPUs", PAPER.md:186-188 strong scaling).

One process per GPU (torch.distributed).  Every rank owns a contiguous block of the particles (by original index).
Per neighbor-list build:

  1. ONE collective: all-gather of the positions (12 bytes per particle; plus the types once) — over NCCL / NVLink on
     GPUs, gloo in the CPU tests.  There is no other exchange on the path.
  2. every rank builds the identical tree over all particles (qbvh_build; the build is about a fifth of the work);
  3. rank g traverses only the queries of Z-order slice g (qbvh_neighbors_range): sorted positions
     [g N / W, (g+1) N / W).  Its lists stay on the rank: row k belongs to the particle whose original index is
     perm[first + k]; entries are global original indices.

`ShardedNeighborList` holds the plumbing only (collective, slicing, merging for checks); the arithmetic is in the
CUDA kernels behind `backend` (default: the C-ABI binding).  Tests plug in a CPU stand-in for `backend` to check the
slicing and merging over gloo without a GPU.
"""
from __future__ import annotations

import numpy as np


def slice_bounds(N: int, world: int, rank: int) -> tuple[int, int]:
    """Z-order slice of rank `rank`: sorted positions [first, first + count); slices tile [0, N) and differ by <= 1."""
    first = (N * rank) // world
    return first, (N * (rank + 1)) // world - first


def owned_block(N: int, world: int, rank: int) -> tuple[int, int]:
    """Block of original indices a rank contributes to the all-gather (same arithmetic as the slices)."""
    return slice_bounds(N, world, rank)


def merge_slices(N: int, parts) -> tuple[np.ndarray, np.ndarray]:
    """Assemble global lists from per-rank results.  parts: iterable of (row_particle, n_neigh, nlist) with
    row_particle[k] = original index of row k.  Returns (n_neigh[N], nlist[N, cap]) with cap = the widest part; every
    particle must appear in exactly one part."""
    parts = list(parts)
    cap = max([p[2].shape[1] for p in parts] + [1])
    n_all = np.full(N, -1, np.int64)
    l_all = np.full((N, cap), -1, np.int64)
    seen = np.zeros(N, np.int64)
    for row_particle, n_neigh, nlist in parts:
        row_particle = np.asarray(row_particle, np.int64)
        np.add.at(seen, row_particle, 1)
        n_all[row_particle] = n_neigh
        l_all[row_particle, : nlist.shape[1]] = nlist
    if not np.all(seen == 1):
        raise ValueError("the slices do not tile the particles exactly once")
    return n_all, l_all


class CudaBackend:
    """The C-ABI binding on this rank's GPU."""

    def __init__(self, N: int, T: int, max_neigh: int, device):
        import torch
        from . import qbvh
        self.torch, self.qbvh, self.device = torch, qbvh, torch.device(device)
        self.N, self.T, self.max_neigh = N, T, max_neigh
        self.inner = qbvh.NeighborList(N, T=T, max_neigh=1, device=device)     # owns the workspace; lists are per slice
        self.perm = torch.empty(max(N, 1), dtype=torch.int32, device=self.device)   # Z-order permutation, kept on the GPU
        self.perm_valid = False

    def build(self, pos, type, box):
        self.perm_valid = False
        return self.inner.build(pos, type, box)

    def neighbors_range(self, r_list, first: int, count: int):
        torch, qbvh = self.torch, self.qbvh
        nlist = torch.empty((max(count, 1), max(self.max_neigh, 1)), dtype=torch.int32, device=self.device)
        n_neigh = torch.zeros(max(count, 1), dtype=torch.int32, device=self.device)
        M = qbvh.qbvh_neighbors_range(r_list, nlist, n_neigh, self.max_neigh, first, count)
        while M > self.max_neigh:                                              # overflow: retry with capacity >= M
            self.max_neigh = int((M + 7) // 8 * 8)
            nlist = torch.empty((max(count, 1), self.max_neigh), dtype=torch.int32, device=self.device)
            M = qbvh.qbvh_neighbors_range(r_list, nlist, n_neigh, self.max_neigh, first, count)
        if not self.perm_valid:                                                # once per build, device to device
            qbvh.qbvh_debug_export_into(qbvh.EXPORT_PERM, self.perm)
            self.perm_valid = True
        return self.perm[first:first + count].to(torch.int64), n_neigh[:count], nlist[:count], M


class ShardedNeighborList:
    """Query-sharded neighbor lists over the ranks of a torch.distributed process group."""

    def __init__(self, N: int, T: int = 1, max_neigh: int = 128, device="cuda:0", group=None, backend=None):
        import torch
        import torch.distributed as dist
        self.torch, self.dist, self.group = torch, dist, group
        self.world = dist.get_world_size(group) if dist.is_initialized() else 1
        self.rank = dist.get_rank(group) if dist.is_initialized() else 0
        self.N, self.T = int(N), int(T)
        self.device = torch.device(device)
        self.own_first, self.own_count = owned_block(self.N, self.world, self.rank)
        self.first, self.count = slice_bounds(self.N, self.world, self.rank)
        self.backend = backend if backend is not None else CudaBackend(self.N, self.T, max_neigh, device)
        self._gather_bufs = {}

    def all_gather_rows(self, local, name="rows"):
        """All-gather of the ranks' row blocks into ONE persistent tensor per `name` (the build's input: nothing is
        allocated per step).  Equal blocks (world divides N): the collective writes straight into it.  Unequal blocks
        (they differ by one row): the collective needs equal pieces, so it lands in a padded persistent buffer and the
        blocks are copied into place."""
        torch, dist = self.torch, self.dist
        if self.world == 1:
            return local
        key = (name, local.dtype, tuple(local.shape[1:]))
        bufs = self._gather_bufs.get(key)
        if bufs is None:
            full = torch.empty((self.N,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
            longest = max(owned_block(self.N, self.world, r)[1] for r in range(self.world))
            padded = None
            if self.N % self.world:
                padded = (torch.zeros((longest,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device),
                          torch.empty((self.world * longest,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device))
            bufs = self._gather_bufs[key] = (full, longest, padded)
        full, longest, padded = bufs
        if padded is None:
            dist.all_gather_into_tensor(full, local, group=self.group)
            return full
        mine, everyone = padded
        mine[: local.shape[0]] = local
        dist.all_gather_into_tensor(everyone, mine, group=self.group)
        for r in range(self.world):
            first, count = owned_block(self.N, self.world, r)
            full[first:first + count] = everyone[r * longest: r * longest + count]
        return full

    def build(self, pos_local, type_local, box):
        """pos_local: this rank's (own_count, 3) block.  All-gathers, then builds the full tree on every rank."""
        assert tuple(pos_local.shape) == (self.own_count, 3)
        self.pos = self.all_gather_rows(pos_local.contiguous(), "pos")
        self.type = None if type_local is None else self.all_gather_rows(type_local.contiguous(), "type")
        return self.backend.build(self.pos, self.type, box)

    def neighbors(self, r_list):
        """Lists of this rank's Z-order slice: (row_particle, n_neigh, nlist, M_global)."""
        perm, n_neigh, nlist, M = self.backend.neighbors_range(r_list, self.first, self.count)
        if self.world > 1:
            m = self.torch.tensor([M], dtype=self.torch.int64, device=n_neigh.device)
            self.dist.all_reduce(m, op=self.dist.ReduceOp.MAX, group=self.group)
            M = int(m.item())
        return perm, n_neigh, nlist, M
