"""Seeded synthetic input generators for the five BASELINE.json configs.

This module is the ONLY code shared by the CUDA path's tests/bench and the CPU
oracle's tests.  It holds none of the method's arithmetic (no Morton codes, no
tree, no quantizer, no neighbor predicate): it only draws particle positions,
types and cutoff tables.  Recipes follow SURVEY.md §8(d) and are restated in
DESIGN.md §"Input recipe".

The paper measured on MD-equilibrated HOOMD-blue configurations that are not
available; these seeded inputs take the paper's workload
*shapes* (liquid-like LJ fluid PAPER.md:172, short cutoff :204, inhomogeneous
large system :212, size-disparate mixture :45) and stand in for them.

Conventions common to all generators
  * RNG  = numpy.random.default_rng([config_id, seed]); all draws in fp64.
  * Coordinates are formed in [0, L), shifted by -L/2, cast to fp32, then
    re-wrapped *in fp32* into [-L/2, L/2) (a cast can land exactly on +L/2).
  * box  = float32 [lo_x, lo_y, lo_z, L_x, L_y, L_z] with lo = -0.5f * L (exact).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np


@dataclass
class Workload:
    name: str
    pos: np.ndarray            # (N,3) float32, wrapped into [lo, lo+L)
    type: Optional[np.ndarray]  # (N,) int32 in [0,T) or None (T = 1)
    box: np.ndarray            # (6,) float32 {lo_xyz, L_xyz}
    r_list: np.ndarray         # (T,T) float32, symmetric
    max_neigh: int
    meta: dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return int(self.pos.shape[0])

    @property
    def T(self) -> int:
        return int(self.r_list.shape[0])


def _finish(pos64: np.ndarray, L) -> tuple[np.ndarray, np.ndarray]:
    """[0,L) fp64 coordinates -> centred, wrapped fp32 coordinates + box."""
    L = np.broadcast_to(np.asarray(L, dtype=np.float64), (3,))
    L32 = L.astype(np.float32)
    lo32 = (np.float32(-0.5) * L32).astype(np.float32)
    hi32 = (np.float32(0.5) * L32).astype(np.float32)
    p = (pos64 - 0.5 * L).astype(np.float32)
    for d in range(3):
        c = p[:, d]
        c = np.where(c >= hi32[d], (c - L32[d]).astype(np.float32), c)
        c = np.where(c < lo32[d], (c + L32[d]).astype(np.float32), c)
        # a second pass is never needed for inputs in [0,L); clamp guards the
        # one-ulp case (c + L) == hi
        c = np.where(c >= hi32[d], np.nextafter(hi32[d], np.float32(-np.inf)), c)
        p[:, d] = c
    assert np.all(p >= lo32) and np.all(p < hi32)
    box = np.concatenate([lo32, L32]).astype(np.float32)
    return np.ascontiguousarray(p, dtype=np.float32), box


def place(pos64: np.ndarray, L, lo) -> tuple[np.ndarray, np.ndarray]:
    """[0,L) fp64 coordinates -> fp32 coordinates in a box whose origin is `lo` (any place, not centred), wrapped
    *in fp32* into [lo, lo + L): every coordinate p satisfies lo <= p and p - lo < L exactly."""
    L = np.broadcast_to(np.asarray(L, dtype=np.float64), (3,))
    L32 = L.astype(np.float32)
    lo32 = np.broadcast_to(np.asarray(lo, dtype=np.float64), (3,)).astype(np.float32)
    p = (pos64 + lo32.astype(np.float64)).astype(np.float32)
    for d in range(3):
        c = p[:, d]
        hi = lo32[d].astype(np.float64) + L32[d].astype(np.float64)      # exact upper face
        c = np.where(c.astype(np.float64) >= hi, (c - L32[d]).astype(np.float32), c)
        c = np.where(c < lo32[d], (c + L32[d]).astype(np.float32), c)
        c = np.maximum(c, lo32[d])
        top = np.float32(hi)
        if np.float64(top) >= hi:
            top = np.nextafter(top, np.float32(-np.inf))                # largest fp32 strictly below the face
        c = np.minimum(c, top)
        p[:, d] = c
    box = np.concatenate([lo32, L32]).astype(np.float32)
    return np.ascontiguousarray(p, dtype=np.float32), box


def shifted(w: "Workload", lo) -> "Workload":
    """The same configuration in a box with origin `lo` instead of -L/2 (positions re-rounded to fp32 there)."""
    L = w.box[3:6].astype(np.float64)
    p64 = w.pos.astype(np.float64) - w.box[:3].astype(np.float64)       # back to [0, L)
    pos, box = place(p64, L, lo)
    return Workload(f"{w.name}_lo{tuple(float(x) for x in np.atleast_1d(lo))}", pos, w.type, box, w.r_list,
                    w.max_neigh, dict(w.meta))


def as_f64(w: "Workload", seed: int = 0) -> tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Double-precision stand-in for a workload: every coordinate moved inside its own fp32 rounding interval by a
    seeded uniform fraction of the spacing (so it is no longer an fp32 number but still rounds to the fp32 input), kept
    inside the box.  Returns (pos64, box64, r_list64)."""
    rng = np.random.default_rng([9064, seed])
    p32 = w.pos
    sp = np.spacing(np.abs(p32)).astype(np.float64)
    pos = p32.astype(np.float64) + (rng.random(p32.shape) - 0.5) * 0.9 * sp
    box = w.box.astype(np.float64)
    pos = np.maximum(pos, box[:3])
    pos = np.minimum(pos, np.nextafter(box[:3] + box[3:], -np.inf))
    r = w.r_list.astype(np.float64) * (1.0 + 1e-9)      # a cutoff that is not an fp32 number either
    return np.ascontiguousarray(pos), box, r


def _rng(config_id: int, seed: int) -> np.random.Generator:
    return np.random.default_rng([config_id, seed])


# ----------------------------------------------------------------------------
# config 1: LJ fluid, uniform random (ideal-gas positions)
# ----------------------------------------------------------------------------
def lj_uniform(N: int = 4096, rho: float = 0.85, r_list: float = 2.9,
               max_neigh: int = 256, seed: int = 0, config_id: int = 1) -> Workload:
    rng = _rng(config_id, seed)
    L = (N / rho) ** (1.0 / 3.0)
    pos, box = _finish(rng.random((N, 3)) * L, L)
    return Workload(f"lj_uniform_N{N}", pos, None, box,
                    np.array([[r_list]], dtype=np.float32), max_neigh,
                    {"rho": rho, "L": L, "config": config_id})


# ----------------------------------------------------------------------------
# config 2: LJ fluid, jittered simple-cubic lattice, permuted
# ----------------------------------------------------------------------------
def lj_lattice(N: int = 1 << 20, n_lat: int = 102, rho: float = 0.85,
               jitter: float = 0.15, r_list: float = 2.9, max_neigh: int = 128,
               seed: int = 0, config_id: int = 2) -> Workload:
    assert N <= n_lat ** 3
    rng = _rng(config_id, seed)
    L = (N / rho) ** (1.0 / 3.0)
    sites = rng.choice(n_lat ** 3, size=N, replace=False)
    ijk = np.stack(np.unravel_index(sites, (n_lat, n_lat, n_lat)), axis=1).astype(np.float64)
    p = (ijk + 0.5) * (L / n_lat) + rng.normal(0.0, jitter, size=(N, 3))
    p = np.mod(p, L)
    p[p >= L] = 0.0
    p = p[rng.permutation(N)]
    pos, box = _finish(p, L)
    return Workload(f"lj_lattice_N{N}", pos, None, box,
                    np.array([[r_list]], dtype=np.float32), max_neigh,
                    {"rho": rho, "L": L, "config": config_id})


# ----------------------------------------------------------------------------
# config 3: colloid-solvent mixture (two types, three cutoffs)
# ----------------------------------------------------------------------------
def colloid_solvent(N: int = 500_000, n_colloid: int = 2000, d_colloid: float = 10.0,
                    d_solvent: float = 1.0, phi: float = 0.3, max_neigh: int = 128,
                    seed: int = 0, config_id: int = 3) -> Workload:
    from scipy.spatial import cKDTree

    rng = _rng(config_id, seed)
    n_solvent = N - n_colloid
    V = (n_colloid * (np.pi / 6.0) * d_colloid ** 3 + n_solvent * (np.pi / 6.0) * d_solvent ** 3) / phi
    L = V ** (1.0 / 3.0)
    # colloids: random sequential addition, one candidate at a time
    col = np.empty((n_colloid, 3))
    n_acc = 0
    n_cand = 0
    while n_acc < n_colloid:
        c = rng.random(3) * L
        n_cand += 1
        if n_acc:
            d = col[:n_acc] - c
            d -= L * np.round(d / L)
            if np.min(np.einsum("ij,ij->i", d, d)) < d_colloid ** 2:
                continue
        col[n_acc] = c
        n_acc += 1
    # solvent: uniform candidates in fixed batches, kept if outside every colloid
    excl = 0.5 * (d_colloid + d_solvent)
    tree = cKDTree(col, boxsize=L)
    sol = np.empty((n_solvent, 3))
    n_acc = 0
    batch = 1 << 16
    while n_acc < n_solvent:
        c = rng.random((batch, 3)) * L
        c[c >= L] = 0.0
        dist, _ = tree.query(c, k=1)
        keep = c[dist >= excl]
        take = min(len(keep), n_solvent - n_acc)
        sol[n_acc:n_acc + take] = keep[:take]
        n_acc += take
    p = np.concatenate([col, sol], axis=0)
    t = np.concatenate([np.zeros(n_colloid, np.int32), np.ones(n_solvent, np.int32)])
    perm = rng.permutation(N)
    p, t = p[perm], t[perm]
    pos, box = _finish(p, L)
    dia = np.array([d_colloid, d_solvent])
    r = 0.5 * (dia[:, None] + dia[None, :]) * 2.0 ** (1.0 / 6.0) + 0.4
    return Workload(f"colloid_solvent_N{N}", pos, np.ascontiguousarray(t), box,
                    r.astype(np.float32), max_neigh,
                    {"L": L, "n_colloid": n_colloid, "rsa_candidates": n_cand, "config": config_id})


# ----------------------------------------------------------------------------
# config 4: Kremer-Grest bead-spring melt (lock-step chain growth)
# ----------------------------------------------------------------------------
def polymer_melt(n_chains: int = 10_000, chain_len: int = 100, rho: float = 0.85,
                 bond: float = 0.97, r_reject: float = 0.8, max_rounds: int = 50,
                 r_list: float = 2.0 ** (1.0 / 6.0) + 0.4, max_neigh: int = 64,
                 seed: int = 0, config_id: int = 4) -> Workload:
    """Lock-step growth: bead k of every chain is placed before bead k+1 of any.

    A proposal is rejected if any bead placed in an EARLIER growth step (any
    chain) lies within r_reject (minimum image); rejected chains redraw, up to
    max_rounds rounds, then the last proposal is accepted.  The rejection test
    uses a hash grid of cell width >= r_reject holding at most CAP beads per
    cell (beads beyond CAP in one cell are not seen by the test; deterministic).
    """
    N = n_chains * chain_len
    L = (N / rho) ** (1.0 / 3.0)
    # the full-size generator takes about a minute: keep its output in the temp directory (pure function of the args)
    import os
    import tempfile
    tag = f"{n_chains}_{chain_len}_{rho}_{bond}_{r_reject}_{max_rounds}_{seed}_{config_id}"
    cache = os.path.join(tempfile.gettempdir(), f"qbvh_polymer_melt_{tag}.npz")
    if N >= 200_000 and os.path.exists(cache):
        try:
            z = np.load(cache)
            return Workload(f"polymer_melt_N{N}", z["pos"], None, z["box"], np.array([[r_list]], dtype=np.float32),
                            max_neigh, {"rho": rho, "L": L, "forced_accepts": int(z["forced"]), "config": config_id})
        except Exception:
            pass
    rng = _rng(config_id, seed)
    nc = int(np.floor(L / r_reject))
    assert nc >= 3, "box too small for the rejection grid"
    w = L / nc
    CAP = 8
    cell_cnt = np.zeros(nc ** 3, np.int32)
    cell_pts = np.zeros((nc ** 3, CAP, 3))
    offs = np.array([(i, j, k) for i in (-1, 0, 1) for j in (-1, 0, 1) for k in (-1, 0, 1)])

    def cell_of(p):
        c = np.floor(p / w).astype(np.int64)
        return np.clip(c, 0, nc - 1)

    def insert(p):
        c = cell_of(p)
        cid = (c[:, 0] * nc + c[:, 1]) * nc + c[:, 2]
        order = np.argsort(cid, kind="stable")
        cid_s, p_s = cid[order], p[order]
        # slot = running count inside equal cid groups
        first = np.r_[True, cid_s[1:] != cid_s[:-1]]
        grp_start = np.maximum.accumulate(np.where(first, np.arange(len(cid_s)), 0))
        slot = cell_cnt[cid_s] + (np.arange(len(cid_s)) - grp_start)
        ok = slot < CAP
        cell_pts[cid_s[ok], slot[ok]] = p_s[ok]
        np.add.at(cell_cnt, cid_s, 1)
        np.minimum(cell_cnt, CAP, out=cell_cnt)

    def too_close(p):
        c = cell_of(p)
        nb = (c[:, None, :] + offs[None, :, :]) % nc           # (m,27,3)
        cid = (nb[..., 0] * nc + nb[..., 1]) * nc + nb[..., 2]  # (m,27)
        q = cell_pts[cid]                                       # (m,27,CAP,3)
        d = q - p[:, None, None, :]
        d -= L * np.round(d / L)
        d2 = np.einsum("...k,...k->...", d, d)
        valid = np.arange(CAP)[None, None, :] < cell_cnt[cid][..., None]
        d2 = np.where(valid, d2, np.inf)
        return np.any(d2 < r_reject ** 2, axis=(1, 2))

    beads = np.empty((n_chains, chain_len, 3))
    prev = rng.random((n_chains, 3)) * L
    prev[prev >= L] = 0.0
    beads[:, 0] = prev
    insert(prev)
    forced = 0
    for k in range(1, chain_len):
        new = np.empty_like(prev)
        todo = np.arange(n_chains)
        for rnd in range(max_rounds):
            u = rng.normal(size=(len(todo), 3))
            u /= np.linalg.norm(u, axis=1, keepdims=True)
            cand = np.mod(prev[todo] + bond * u, L)
            cand[cand >= L] = 0.0
            new[todo] = cand
            bad = too_close(cand)
            todo = todo[bad]
            if len(todo) == 0:
                break
        forced += len(todo)
        beads[:, k] = new
        insert(new)
        prev = new
    pos, box = _finish(beads.reshape(N, 3), L)
    if N >= 200_000:
        try:
            np.savez(cache + f".{os.getpid()}.tmp.npz", pos=pos, box=box, forced=forced)
            os.replace(cache + f".{os.getpid()}.tmp.npz", cache)
        except Exception:
            pass
    return Workload(f"polymer_melt_N{N}", pos, None, box,
                    np.array([[r_list]], dtype=np.float32), max_neigh,
                    {"rho": rho, "L": L, "forced_accepts": int(forced), "config": config_id})


# ----------------------------------------------------------------------------
# config 5: vapor-liquid slab, orthorhombic box Lz = 3 Lx
# ----------------------------------------------------------------------------
def vapor_liquid_slab(N: int = 1 << 21, rho_liq: float = 0.75, rho_vap: float = 0.02,
                      r_list: float = 3.3, max_neigh: int = 256, seed: int = 0,
                      config_id: int = 5) -> Workload:
    rng = _rng(config_id, seed)
    Lx = (N / (rho_liq + 2.0 * rho_vap)) ** (1.0 / 3.0)
    Lz = 3.0 * Lx
    n_liq = int(round(rho_liq * Lx ** 3))
    n_vap = N - n_liq
    liq = rng.random((n_liq, 3)) * Lx
    liq[:, 2] += Lx
    vap = rng.random((n_vap, 3)) * np.array([Lx, Lx, 2.0 * Lx])
    vap[:, 2] = np.where(vap[:, 2] < Lx, vap[:, 2], vap[:, 2] + Lx)
    p = np.concatenate([liq, vap], axis=0)[rng.permutation(N)]
    Lvec = np.array([Lx, Lx, Lz])
    p = np.minimum(p, np.nextafter(Lvec, 0.0))
    pos, box = _finish(p, Lvec)
    return Workload(f"vapor_liquid_N{N}", pos, None, box,
                    np.array([[r_list]], dtype=np.float32), max_neigh,
                    {"Lx": Lx, "Lz": Lz, "n_liq": n_liq, "n_vap": n_vap, "config": config_id})


# ----------------------------------------------------------------------------
# lattices for the oracle pins (closed-form coordination shells)
# ----------------------------------------------------------------------------
def simple_cubic(n: int, a: float = 1.0) -> tuple[np.ndarray, np.ndarray]:
    """n^3 sites, spacing a, periodic box L = n*a; sites at cell centres."""
    g = (np.arange(n) + 0.5) * a
    p = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)
    return _finish(p, n * a)


def fcc(n: int, a: float = 1.0) -> tuple[np.ndarray, np.ndarray]:
    """4 n^3 sites of the conventional FCC cell of edge a; nearest-neighbor distance a/sqrt(2)."""
    basis = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]]) + 0.25
    g = np.arange(n)
    cells = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 1, 3)
    p = ((cells + basis[None]) * a).reshape(-1, 3)
    return _finish(p, n * a)


# ----------------------------------------------------------------------------
# registry: the five configs at full size and at reduced ("small") size
# ----------------------------------------------------------------------------
def make_config(cid: int, small: bool = False, seed: int = 0) -> Workload:
    if cid == 1:
        return lj_uniform(seed=seed)
    if cid == 2:
        if small:
            return lj_lattice(N=40_000, n_lat=35, seed=seed)
        return lj_lattice(seed=seed)
    if cid == 3:
        if small:
            return colloid_solvent(N=30_000, n_colloid=120, seed=seed)
        return colloid_solvent(seed=seed)
    if cid == 4:
        if small:
            return polymer_melt(n_chains=400, chain_len=100, seed=seed)
        return polymer_melt(seed=seed)
    if cid == 5:
        if small:
            return vapor_liquid_slab(N=50_003, seed=seed)
        return vapor_liquid_slab(seed=seed)
    raise ValueError(f"unknown config {cid}")
