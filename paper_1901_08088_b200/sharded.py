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


# ---------------------------------------------------------------------------------------------------------------------
# Slab domain decomposition with halos (SURVEY §8e bullet 2, §8f NEXT-4 second half; "a domain decomposition
# strategy", PAPER.md:186 strong scaling).  Unlike query sharding nothing is redundant: rank g owns the particles of slab
# g of W equal slabs along the longest box axis, receives from its two neighbor ranks the particles within a halo width
# h >= r of the shared faces (one neighbor exchange per build), builds the tree over own + ghost particles and keeps the
# rows of its own particles.  Ghosts keep their ORIGINAL coordinates and the tree is built in the ORIGINAL periodic box,
# so a pair across the box edge is found by the library's own minimum image and every distance is computed from exactly
# the numbers the single-GPU run uses: the lists are identical, not merely close.  Build and traversal both divide by W
# (plus the halo fraction 2h / slab width).
# ---------------------------------------------------------------------------------------------------------------------
def slab_axis(box) -> int:
    """The cut axis: the longest box edge (first one on ties)."""
    return int(np.argmax(np.asarray(box, np.float64)[3:6]))


def halo_width(r_list) -> float:
    """Halo width h: a little more than the largest cutoff (a neighbor differs by at most r along the cut axis; the slack
    covers the fp32 rounding of the pair predicate)."""
    r = float(np.max(np.asarray(r_list, np.float64)))
    return r * (1.0 + 2.0 ** -10)


def slab_geometry(box, world: int, h: float):
    """(axis, slab width); refuses slabs thinner than the halo (ghosts would have to come from second neighbors)."""
    box = np.asarray(box, np.float64)
    axis = slab_axis(box)
    width = box[3 + axis] / world
    if world > 1 and width < h:
        raise ValueError(f"slab width {width:.6g} along axis {axis} is below the halo width {h:.6g}: use fewer ranks")
    return axis, width


def _is_torch(x) -> bool:
    return type(x).__module__.startswith("torch")


def slab_index(pos, box, world: int, axis: int):
    """Slab of every particle: floor((x - lo) / width) clamped to [0, W-1], in fp64.  numpy in, numpy out; a torch tensor
    (any device) in, a tensor on that device out — the same fp64 operations either way."""
    scale = world / float(box[3 + axis])
    if _is_torch(pos):
        x = pos[:, axis].double() - float(box[axis])
        return (x * scale).floor().long().clamp_(0, world - 1)
    x = np.asarray(pos, np.float64)[:, axis] - float(box[axis])
    return np.clip(np.floor(x * scale).astype(np.int64), 0, world - 1)


def halo_masks(pos, box, world: int, axis: int, g: int, h: float):
    """Which of rank g's OWN particles its left (g-1) and right (g+1) neighbors need: within h of the respective face.
    numpy or torch in, the same kind out."""
    x = (pos[:, axis].double() if _is_torch(pos) else np.asarray(pos, np.float64)[:, axis]) - float(box[axis])
    width = float(box[3 + axis]) / world
    return (x - g * width) < h, ((g + 1) * width - x) <= h


def local_set_indices(pos, box, world: int, g: int, h: float):
    """What rank g ends up with, computed from ALL particles (for tests and single-process emulation; the distributed path
    never sees other ranks' particles): (indices of its own particles, indices of its ghosts)."""
    axis, _ = slab_geometry(box, world, h)
    slab = slab_index(pos, box, world, axis)
    own = np.nonzero(slab == g)[0]
    if world == 1:
        return own, own[:0]
    ghosts = []
    peers = {(g - 1) % world, (g + 1) % world}
    for peer in sorted(peers):
        idx = np.nonzero(slab == peer)[0]
        to_left, to_right = halo_masks(pos[idx], box, world, axis, peer, h)
        want = np.zeros(len(idx), bool)
        if (peer + 1) % world == g:
            want |= to_right                      # I am its right neighbor
        if (peer - 1) % world == g:
            want |= to_left                       # I am its left neighbor
        ghosts.append(idx[want])
    return own, np.concatenate(ghosts)


class SlabNeighborList:
    """Neighbor lists of the particles this rank owns (slab `rank` of `world`), from own + halo particles.

    backend: object with  build(pos, type, box, n_expected_global)  and  neighbors_rows(r_list, n_rows) ->
    (n_neigh[n_rows], nlist[n_rows, cap], M)  — rows are the first n_rows particles given to build, entries are indices
    into the array given to build.  Default: CudaSlabBackend.  Tests plug in a CPU stand-in (the oracle)."""

    def __init__(self, box, r_list, T: int = 1, max_neigh: int = 128, device="cuda:0", group=None, backend=None):
        import torch
        import torch.distributed as dist
        self.torch, self.dist, self.group = torch, dist, group
        self.world = dist.get_world_size(group) if dist.is_initialized() else 1
        self.rank = dist.get_rank(group) if dist.is_initialized() else 0
        self.box = np.asarray(box, np.float32)
        self.r_list = np.asarray(r_list, np.float32)
        self.h = halo_width(self.r_list)
        self.axis, self.width = slab_geometry(self.box, self.world, self.h)
        self.device = torch.device(device)
        self.backend = backend if backend is not None else CudaSlabBackend(T, max_neigh, device)
        self.halo_bytes = 0

    def exchange(self, pos, type, gid):
        """One neighbor exchange: sends the particles within h of each face to the rank across it, returns the ghosts
        received (pos, type, gid).  With two ranks both faces lead to the same peer: one message with the union."""
        torch, dist = self.torch, self.dist
        W, g = self.world, self.rank
        if W == 1:
            return pos[:0], (None if type is None else type[:0]), gid[:0]
        to_left, to_right = halo_masks(pos, self.box, W, self.axis, g, self.h)        # on the device the positions live on
        left, right = (g - 1) % W, (g + 1) % W
        sends = {left: to_left | to_right} if left == right else {left: to_left, right: to_right}
        counts = torch.zeros(2, dtype=torch.int64, device=pos.device)          # what I send to my left / right neighbor
        for k, peer in enumerate((left, right)):
            counts[k] = int(sends[peer].sum())
        allc = torch.empty(2 * W, dtype=torch.int64, device=pos.device)
        dist.all_gather_into_tensor(allc, counts, group=self.group)
        allc = allc.cpu().numpy().reshape(W, 2)
        recv_n = {left: int(allc[left, 1])} if left == right else {left: int(allc[left, 1]), right: int(allc[right, 0])}
        ops, bufs = [], []
        self.halo_bytes = 0                                                      # bytes this rank sends per build
        for peer, mask in sends.items():
            idx = torch.nonzero(mask).flatten()
            payload = [pos[idx].contiguous(), gid[idx].contiguous()] + ([] if type is None else [type[idx].contiguous()])
            self.halo_bytes += sum(p.numel() * p.element_size() for p in payload)
            if len(idx):                                                         # (an empty halo is not sent: the peer knows the count)
                ops += [dist.P2POp(dist.isend, p, peer, group=self.group) for p in payload]
        for peer, n in recv_n.items():
            rb = [torch.empty((n, 3), dtype=pos.dtype, device=pos.device), torch.empty(n, dtype=gid.dtype, device=pos.device)]
            if type is not None:
                rb.append(torch.empty(n, dtype=type.dtype, device=pos.device))
            bufs.append(rb)
            if n:
                ops += [dist.P2POp(dist.irecv, b, peer, group=self.group) for b in rb]
        if ops:
            for req in dist.batch_isend_irecv(ops):
                req.wait()
        gpos = torch.cat([b[0] for b in bufs])
        ggid = torch.cat([b[1] for b in bufs])
        gtyp = None if type is None else torch.cat([b[2] for b in bufs])
        return gpos, gtyp, ggid

    def build(self, pos_own, type_own, gid_own, n_global: int):
        """pos_own (n, 3), type_own (n) or None, gid_own (n) int64: this rank's particles, all inside slab `rank`."""
        torch = self.torch
        if not bool((slab_index(pos_own, self.box, self.world, self.axis) == self.rank).all()):
            raise ValueError("a particle handed to this rank lies outside its slab")
        gpos, gtyp, ggid = self.exchange(pos_own, type_own, gid_own)
        return self.build_from_local_set(torch.cat([pos_own, gpos]).contiguous(),
                                         None if type_own is None else torch.cat([type_own, gtyp]).contiguous(),
                                         torch.cat([gid_own, ggid]).contiguous(), int(pos_own.shape[0]), n_global)

    def build_from_local_set(self, pos, type, gid, n_own: int, n_global: int):
        """The build half after the exchange: own particles first, ghosts behind them (also the entry for a single-process
        emulation of the ranks, which forms the local sets itself)."""
        self.pos, self.type, self.gid = pos, type, gid
        self.n_own, self.n_ghost = n_own, int(pos.shape[0]) - n_own
        return self.backend.build(self.pos, self.type, self.box, n_global)

    def neighbors(self):
        """(gid_own, n_neigh, nlist with GLOBAL particle ids, M over all ranks) for this rank's own particles."""
        torch, dist = self.torch, self.dist
        n_neigh, nlist, M = self.backend.neighbors_rows(self.r_list, self.n_own)
        # local indices -> global ids, in the entries' own width (int32: N < 2^30).  Entries beyond a row's count are
        # unspecified by the C-ABI and stay so (clamped into range for the gather, nothing more).
        gid32 = self.gid.to(device=nlist.device, dtype=torch.int32)
        nlist_g = gid32[nlist.clamp_(0, max(int(gid32.shape[0]) - 1, 0))] if gid32.shape[0] else nlist
        if self.world > 1:
            m = torch.tensor([M], dtype=torch.int64, device=n_neigh.device)
            dist.all_reduce(m, op=dist.ReduceOp.MAX, group=self.group)
            M = int(m.item())
        return self.gid[: self.n_own], n_neigh, nlist_g, M


class CudaSlabBackend:
    """The C-ABI binding for a particle count that changes from build to build (own + ghosts): one workspace sized
    with headroom, re-allocated only when it is outgrown."""

    def __init__(self, T: int, max_neigh: int, device):
        import torch
        from . import qbvh
        self.torch, self.qbvh, self.device = torch, qbvh, torch.device(device)
        self.T, self.max_neigh = T, max_neigh
        self.cap_n, self.workspace, self.nlist, self.n_neigh = 0, None, None, None

    def build(self, pos, type, box, n_global: int):
        torch, qbvh = self.torch, self.qbvh
        n = int(pos.shape[0])
        self.n = n
        if n > self.cap_n or self.workspace is None:
            self.cap_n = int(1.25 * n) + 1024
            self.workspace = torch.empty(qbvh.qbvh_workspace_bytes(self.cap_n, self.T), dtype=torch.uint8, device=self.device)
            self.nlist = None
            qbvh.qbvh_set_workspace(self.workspace)
        qbvh.qbvh_set_stream(torch.cuda.current_stream(self.device).cuda_stream)
        qbvh.qbvh_set_num_types(self.T)
        # the Morton cells are a grid over the whole box and this rank's particles fill 1/W of it: pick the grid the
        # whole system would get (density independence)
        lvl = 2
        while lvl < 6 and n_global > (48 << (3 * lvl)):
            lvl += 1
        qbvh.qbvh_set_option(qbvh.OPT_CELL_LEVEL, lvl)
        try:
            return qbvh.qbvh_build(pos, type, n, box)
        finally:
            qbvh.qbvh_set_option(qbvh.OPT_CELL_LEVEL, 0)

    def neighbors_rows(self, r_list, n_rows: int):
        torch, qbvh = self.torch, self.qbvh
        while True:
            if self.nlist is None or self.nlist.shape[0] < self.n or self.nlist.shape[1] != self.max_neigh:
                self.nlist = torch.empty((max(self.cap_n, 1), max(self.max_neigh, 1)), dtype=torch.int32, device=self.device)
                self.n_neigh = torch.zeros(max(self.cap_n, 1), dtype=torch.int32, device=self.device)
            M = qbvh.qbvh_neighbors(r_list, self.nlist, self.n_neigh, self.max_neigh)      # rows of ghosts are computed and dropped
            own_max = int(self.n_neigh[:n_rows].max().item()) if n_rows else 0
            if own_max <= self.max_neigh:
                return self.n_neigh[:n_rows], self.nlist[:n_rows], own_max
            self.max_neigh = int((own_max + 7) // 8 * 8)
            self.nlist = None
