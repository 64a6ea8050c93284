"""Pins for the neighbor-list oracle (oracle/neighbors.c) — CPU only.

Each test pins the oracle to something other than itself: lattice coordination
shells (closed form), exact pair symmetry (invariant), brute force on tiny
inputs, the ideal-gas mean count (closed form), hand-placed pairs, and an fp64
restatement with the north_star's 1e-5 sigma band.  A dropped term, a wrong
sign, a swapped axis or box length fails at least one of them.
"""
import numpy as np
import pytest

from oracle import neighbors as ON
from paper_1901_08088_b200 import workloads as W

from conftest import read_golden


def rows(row_ptr, nbr):
    return [nbr[row_ptr[i]:row_ptr[i + 1]] for i in range(len(row_ptr) - 1)]


# --------------------------------------------------------------------------- lattices
@pytest.mark.parametrize("method", ["brute", "cell"])
def test_simple_cubic_shells(method):
    shells = [(int(s), int(c)) for s, _, c in read_golden("sc_shells.txt")]
    n = 9  # n >= 2*ceil(r/a)+1 for r up to 3.1 a, so no pair is seen through two images
    a = 1.3
    pos, box = W.simple_cubic(n, a)
    # a radius strictly between consecutive shells: sqrt(s + 0.4) lattice units
    for s, cum in shells:
        r = a * np.sqrt(s + 0.4)
        cnt = ON.counts(pos, None, box, np.array([[r]], np.float32), method=method)
        assert np.all(cnt == cum), (s, cum, np.unique(cnt))
    # below the first shell: nobody has neighbors
    assert np.all(ON.counts(pos, None, box, np.array([[0.9 * a]], np.float32), method=method) == 0)


@pytest.mark.parametrize("method", ["brute", "cell"])
def test_fcc_shells(method):
    shells = [(int(s), int(c)) for s, _, c in read_golden("fcc_shells.txt")]
    a = 1.7
    pos, box = W.fcc(5, a)  # L = 5a = 7.07 d  >  2 * sqrt(5.4) d
    d = a / np.sqrt(2.0)
    for s, cum in shells:
        r = d * np.sqrt(s + 0.4)
        cnt = ON.counts(pos, None, box, np.array([[r]], np.float32), method=method)
        assert np.all(cnt == cum), (s, cum, np.unique(cnt))


def test_orthorhombic_lattice_axis_mixup():
    """A stretched lattice (spacing a, 2a, 3a): swapping axes or box lengths changes the counts."""
    n = 8
    g = np.arange(n) + 0.5
    p = np.stack(np.meshgrid(g * 1.0, g * 2.0, g * 3.0, indexing="ij"), -1).reshape(-1, 3)
    pos, box = W._finish(p, np.array([n * 1.0, n * 2.0, n * 3.0]))
    # neighbors within r: integer (i,j,k) != 0 with i^2 + 4 j^2 + 9 k^2 <= r^2
    for r in (1.1, 2.05, 2.3, 3.05, 3.2, 3.7):
        rng_ = range(-4, 5)
        expect = sum(1 for i in rng_ for j in rng_ for k in rng_
                     if (i, j, k) != (0, 0, 0) and i * i + 4 * j * j + 9 * k * k <= r * r)
        for m in ("brute", "cell"):
            cnt = ON.counts(pos, None, box, np.array([[r]], np.float32), method=m)
            assert np.all(cnt == expect), (r, expect, np.unique(cnt))


# --------------------------------------------------------------------------- hand-placed pairs
def test_hand_placed_pairs():
    box = np.array([-5, -5, -15, 10, 10, 30], np.float32)
    # (0) and (1) are 0.5 apart through the periodic x face; (2) is 0.75 from (0) through the z face (Lz = 30)
    pos = np.array([[-4.75, 0, 0], [4.75, 0, 0], [-4.75, 0, 14.75 + 14.5 - 30 + 0.0]], np.float32)
    pos[2] = [-4.75, 0.0, -14.5]
    pos = np.vstack([pos, [[-4.75, 0.0, 14.75]]]).astype(np.float32)  # (3): 0.75 from (2) through z
    r = np.array([[0.8]], np.float32)
    for m in ("brute", "cell"):
        rp, nb, _ = ON.neighbor_list(pos, None, box, r, method=m)
        got = [list(x) for x in rows(rp, nb)]
        assert got == [[1], [0], [3], [2]], got
    # inclusive cutoff ("<= r_c"): a pair at exactly r is a neighbor, one ulp below r it is not
    pos = np.array([[0, 0, 0], [3, 0, 0]], np.float32)
    assert ON.counts(pos, None, box, np.array([[3.0]], np.float32)).tolist() == [1, 1]
    below = np.nextafter(np.float32(3.0), np.float32(0))
    assert ON.counts(pos, None, box, np.array([[below]], np.float32)).tolist() == [0, 0]
    # coincident particles are neighbors of each other; self is excluded by index
    pos = np.array([[1, 2, 3], [1, 2, 3]], np.float32)
    assert ON.counts(pos, None, box, np.array([[0.1]], np.float32)).tolist() == [1, 1]
    # N = 1 and N = 0
    assert ON.counts(pos[:1], None, box, np.array([[4.0]], np.float32)).tolist() == [0]
    assert ON.counts(pos[:0], None, box, np.array([[4.0]], np.float32)).tolist() == []


def test_pair_predicate_arithmetic():
    """O1 by hand in numpy fp32 for one awkward pair (wrap in y only)."""
    box = np.array([-8, -6, -4, 16, 12, 8], np.float32)
    pi = np.array([1.25, -5.5, 0.3], np.float32)
    pj = np.array([2.0, 5.75, -0.2], np.float32)
    dx = np.float32(pj[0] - pi[0])
    dy = np.float32(np.float32(pj[1] - pi[1]) - box[4])  # 11.25 > 6 -> minus Ly
    dz = np.float32(pj[2] - pi[2])
    d2 = np.float32(np.float64(dz) * np.float64(dz) +
                    np.float64(np.float32(np.float64(dy) * np.float64(dy) + np.float64(np.float32(dx * dx)))))
    ok, d2_c, d64 = ON.pair(pi, pj, box, 1.2)
    assert d2_c == d2 and ok == (d2 <= np.float32(1.2) * np.float32(1.2))
    assert abs(d64 - np.sqrt(0.75 ** 2 + 0.75 ** 2 + 0.5 ** 2)) < 1e-6
    # antisymmetry of the arguments leaves d2 unchanged
    assert ON.pair(pj, pi, box, 1.2)[1] == d2_c


# --------------------------------------------------------------------------- invariants
def sym_check(row_ptr, nbr):
    N = len(row_ptr) - 1
    i = np.repeat(np.arange(N), np.diff(row_ptr))
    fwd = i.astype(np.int64) * N + nbr
    bwd = nbr.astype(np.int64) * N + i
    return np.array_equal(np.sort(fwd), np.sort(bwd))


def test_pair_symmetry_zero_exceptions():
    w = W.lj_uniform()
    rp, nb, _ = ON.neighbor_list(w.pos, None, w.box, w.r_list, method="brute")
    assert sym_check(rp, nb)
    w = W.make_config(3, small=True)
    rp, nb, _ = ON.neighbor_list(w.pos, w.type, w.box, w.r_list, method="cell")
    assert sym_check(rp, nb)
    for r in rows(rp, nb)[:2000]:
        assert np.all(np.diff(r) > 0)  # ascending, no duplicates


def test_ideal_gas_mean_count():
    """E[n] = (4/3) pi r^3 rho (N-1)/N for uniform random positions (86.8 at config 1)."""
    w = W.lj_uniform()
    cnt = ON.counts(w.pos, None, w.box, w.r_list, method="brute")
    expect = 4.0 / 3.0 * np.pi * 2.9 ** 3 * 0.85 * (w.N - 1) / w.N
    # Poisson-like: std of the mean ~ sqrt(expect / N) * (pair correlation factor ~ sqrt(2))
    assert abs(cnt.mean() - expect) < 5 * np.sqrt(2 * expect / w.N), (cnt.mean(), expect)


# --------------------------------------------------------------------------- brute force == cell list
def _tiny_cases():
    rng = np.random.default_rng(7)
    cases = []
    for N in (1, 2, 100, 4096):
        L = np.array([7.0, 7.0, 7.0])
        cases.append((f"cubic{N}", *W._finish(rng.random((N, 3)) * L, L), None, np.array([[2.0]], np.float32)))
    L = np.array([6.0, 6.0, 18.0])
    cases.append(("slab", *W._finish(rng.random((3000, 3)) * L, L), None, np.array([[2.2]], np.float32)))
    # two types, unequal cutoffs, one pair type switched off (r <= 0)
    L = np.array([9.0, 9.0, 9.0])
    t = (rng.random(2500) < 0.2).astype(np.int32)
    cases.append(("two_types", *W._finish(rng.random((2500, 3)) * L, L), t,
                  np.array([[3.5, 1.7], [1.7, 0.0]], np.float32)))
    # r just under L/2 -> two cells per axis -> stencil de-duplication path
    L = np.array([5.0, 5.0, 5.0])
    cases.append(("half_box", *W._finish(rng.random((600, 3)) * L, L), None, np.array([[2.49]], np.float32)))
    # particles exactly on box faces, duplicated coordinates
    p = rng.random((500, 3)) * L
    p[:50, 0] = 0.0
    p[50:100, 1] = 0.0
    p[100:120] = p[120:140]
    cases.append(("faces_dups", *W._finish(p, L), None, np.array([[1.3]], np.float32)))
    return cases


@pytest.mark.parametrize("case", _tiny_cases(), ids=lambda c: c[0])
def test_brute_equals_cell_list(case):
    _, pos, box, t, r = case
    a = ON.neighbor_list(pos, t, box, r, method="brute")
    b = ON.neighbor_list(pos, t, box, r, method="cell")
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])


# --------------------------------------------------------------------------- fp64 restatement with the tolerance band
def test_against_fp64_definition_with_band():
    """numpy fp64 minimum-image brute force: sets agree except pairs within 1e-5 of r, all of which are band-tagged."""
    w = W.make_config(5, small=True)
    sel = np.arange(3000)
    pos, box = w.pos[sel], w.box
    r = 3.3
    p = pos.astype(np.float64)
    L = box[3:].astype(np.float64)
    d = p[None, :, :] - p[:, None, :]
    d -= L * np.round(d / L)
    dist = np.sqrt((d ** 2).sum(-1))
    np.fill_diagonal(dist, np.inf)
    rp, nb, band = ON.neighbor_list(pos, None, box, np.array([[r]], np.float32), method="brute")
    got = np.zeros_like(dist, dtype=bool)
    i = np.repeat(np.arange(len(sel)), np.diff(rp))
    got[i, nb] = True
    r32 = float(np.float32(r))
    diff = got != (dist <= r32)
    assert np.all(np.abs(dist[diff] - r32) < 1e-5)
    in_band = np.zeros_like(got)
    in_band[i, nb] = band.astype(bool)
    assert np.array_equal(in_band, got & (np.abs(dist - r32) < 1e-5))
    # the band is narrow: about 2e-5 of all pairs at r ~ 3 sigma (3 * 2e-5 / r), far fewer here
    assert band.mean() < 1e-3


def test_paper_sanity_constants():
    c = {k: float(v) for k, v, _ in read_golden("paper_constants.txt")}
    assert abs(50.0 / 1023 - c["bin_width_box50"]) < 0.005
    assert abs((4 * np.pi / 3) / 8 - c["sphere_over_cube"]) < 0.05
    assert abs((4 * np.pi / 3) / 27 - c["sphere_over_27cells"]) < 0.01
