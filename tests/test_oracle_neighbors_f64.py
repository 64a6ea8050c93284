"""Pins for the double-precision neighbor-list oracle (oracle/neighbors_f64.c) — CPU only.

The fp64 oracle is pinned to things other than itself: lattice coordination shells (closed form), exact pair symmetry,
brute force = cell list on tiny inputs, decisions from exact rational arithmetic, pairs at exactly r_c through face and
corner images, the fp32 oracle on fp32-representable inputs (outside the 1e-5 sigma band), and a pair that only
double precision resolves.
"""
from fractions import Fraction

import numpy as np
import pytest

from oracle import neighbors as ON
from paper_1901_08088_b200 import workloads as W

from adversarial_inputs import boundary_pairs
from conftest import read_golden


def counts64(pos, typ, box, r, method):
    rp, _ = ON.neighbor_list_f64(pos, typ, box, r, method=method)
    return np.diff(rp)


def lattice64(kind, n, a):
    """fp64 lattice in a box [lo, lo + n a) with an origin and a spacing that are not fp32 numbers."""
    pos32, box32 = (W.simple_cubic if kind == "sc" else W.fcc)(n, 1.0)
    frac = (pos32.astype(np.float64) - box32[:3].astype(np.float64))          # lattice sites in units of a, exact
    lo = np.array([0.1234567890123, -7.7654321098765, 1e-3])
    box = np.concatenate([lo, np.full(3, n * a)])
    return frac * a + lo, box


@pytest.mark.parametrize("method", ["brute", "cell"])
def test_simple_cubic_shells_f64(method):
    shells = [(int(s), int(c)) for s, _, c in read_golden("sc_shells.txt")]
    a = 1.3 * (1 + 1e-9)
    pos, box = lattice64("sc", 9, a)
    for s, cum in shells:
        cnt = counts64(pos, None, box, np.array([[a * np.sqrt(s + 0.4)]]), method)
        assert np.all(cnt == cum), (s, cum, np.unique(cnt))
    assert np.all(counts64(pos, None, box, np.array([[0.9 * a]]), method) == 0)


@pytest.mark.parametrize("method", ["brute", "cell"])
def test_fcc_shells_f64(method):
    shells = [(int(s), int(c)) for s, _, c in read_golden("fcc_shells.txt")]
    a = 1.7 / 3.0 * 3.0000001
    pos, box = lattice64("fcc", 5, a)
    d = a / np.sqrt(2.0)
    for s, cum in shells:
        cnt = counts64(pos, None, box, np.array([[d * np.sqrt(s + 0.4)]]), method)
        assert np.all(cnt == cum), (s, cum, np.unique(cnt))


def test_symmetry_and_brute_equals_cell_f64():
    rng = np.random.default_rng(64)
    cases = []
    L = np.array([7.3, 7.3, 7.3])
    cases.append((rng.random((900, 3)) * L, None, L, np.array([[1.6]])))
    L = np.array([5.0, 5.0, 15.0])
    typ = rng.integers(0, 2, 700).astype(np.int32)
    cases.append((rng.random((700, 3)) * L, typ, L, np.array([[1.1, 2.3], [2.3, 0.0]])))
    L = np.array([4.0, 4.0, 4.0])
    p = rng.random((300, 3)) * L
    p[:30, 0] = 0.0                                  # on a face
    p[40] = p[41]                                    # coincident particles are neighbors of each other
    cases.append((p, None, L, np.array([[1.99]])))   # r just under L/2: the de-duplicated stencil
    for p, typ, L, r in cases:
        lo = np.array([3.25, -100.0, 0.0])
        box = np.concatenate([lo, L])
        pos = p + lo
        rb, nb = ON.neighbor_list_f64(pos, typ, box, r, method="brute")
        rc, nc = ON.neighbor_list_f64(pos, typ, box, r, method="cell")
        assert np.array_equal(rb, rc) and np.array_equal(nb, nc)
        pairs = set()
        for i in range(len(pos)):
            for j in nb[rb[i]:rb[i + 1]]:
                pairs.add((i, int(j)))
        assert all((j, i) in pairs for (i, j) in pairs)            # j in list(i) <=> i in list(j), no exception
        assert all(i != j for (i, j) in pairs)


def test_predicate_against_exact_rationals_f64():
    """Decisions of O1-64 equal the decisions of exact rational arithmetic on the same fp64 inputs, for every pair whose
    exact squared distance is not within 1e-12 (relative) of r^2 — a wrong sign, axis or box length fails at once."""
    rng = np.random.default_rng(5)
    L = np.array([6.0, 9.0, 4.5])
    lo = np.array([-3.0, 100.0, 0.25])
    box = np.concatenate([lo, L])
    pos = rng.random((60, 3)) * L + lo
    r = 2.2
    checked = 0
    for i in range(0, 60, 3):
        for j in range(60):
            if i == j:
                continue
            ok, d2 = ON.pair_f64(pos[i], pos[j], box, r)
            ex = Fraction(0)
            for d in range(3):
                x = Fraction(pos[j][d]) - Fraction(pos[i][d])
                Ld = Fraction(L[d])
                if x > Ld / 2:
                    x -= Ld
                elif x < -Ld / 2:
                    x += Ld
                ex += x * x
            r2 = Fraction(r) ** 2
            if abs(ex - r2) > r2 * Fraction(1, 10 ** 12):
                assert ok == (ex <= r2), (i, j)
                checked += 1
            assert abs(Fraction(d2) - ex) <= ex * Fraction(1, 10 ** 14) + Fraction(1, 10 ** 28)
    assert checked > 1000


@pytest.mark.parametrize("lo", [(0.0, 0.0, 0.0), (1000.0, -3000.0, 17.0)])
def test_boundary_pairs_f64(lo):
    """Pairs at exactly r_c, one grid step inside and one outside, through face and corner images (all coordinates on a
    binary grid: every operation of the predicate is exact): inclusive at r_c, exclusive beyond."""
    L, r, grid = 24.0, 3.0, 2.0 ** -6
    p, lo64 = boundary_pairs(lo, L, r, grid)
    pos = np.mod(p, L) + lo64
    box = np.concatenate([lo64, np.full(3, L)])
    rp, nb = ON.neighbor_list_f64(pos, None, box, np.array([[r]]), method="brute")
    # exact distances of everybody from particle 0 by integer arithmetic on the grid
    q = np.rint(np.mod(p, L) / grid).astype(np.int64)
    n_l = int(round(L / grid))
    d = q - q[0]
    d = (d + n_l // 2) % n_l - n_l // 2
    d2 = (d * d).sum(1)
    r2 = int(round(r / grid)) ** 2
    expect = np.nonzero((d2 <= r2) & (np.arange(len(q)) != 0))[0]
    assert np.array_equal(nb[rp[0]:rp[1]], expect)
    assert np.sum(d2 == r2) >= 10                                   # the construction really has pairs at exactly r_c


def test_agrees_with_the_fp32_oracle_outside_the_band():
    w = W.make_config(1)
    sel = slice(0, 2000)
    p32 = w.pos[sel]
    r64, n64 = ON.neighbor_list_f64(p32.astype(np.float64), None, w.box.astype(np.float64), w.r_list.astype(np.float64))
    r32, n32, band = ON.neighbor_list(p32, None, w.box, w.r_list)
    a = set(zip(np.repeat(np.arange(len(p32)), np.diff(r64)).tolist(), n64.tolist()))
    b = set(zip(np.repeat(np.arange(len(p32)), np.diff(r32)).tolist(), n32.tolist()))
    inband = set((i, j) for (i, j), f in zip(zip(np.repeat(np.arange(len(p32)), np.diff(r32)).tolist(), n32.tolist()), band.tolist()) if f)
    assert (b - a) <= inband                      # whatever fp32 accepts and fp64 rejects lies within 1e-5 sigma of r
    for (i, j) in a - b:                          # and the other way round
        assert abs(ON.pair(p32[i], p32[j], w.box, float(w.r_list[0, 0]))[2] - float(w.r_list[0, 0])) < 1e-5


def test_only_double_precision_resolves_this_pair():
    """Two particles r (1 + 1e-10) apart at coordinates near 1000: fp64 says 'not a neighbor'; their fp32 roundings
    coincide with a pair exactly r apart, which fp32 accepts.  The fp64 oracle must not be a cast of fp32 work."""
    r = 2.5
    box = np.array([990.0, 990.0, 990.0, 32.0, 32.0, 32.0])
    pi = np.array([1000.0, 1001.0, 1002.0])
    pj = pi + np.array([r * (1 + 1e-10), 0.0, 0.0])
    assert not ON.pair_f64(pi, pj, box, r)[0]
    assert ON.pair_f64(pi, pi + np.array([r, 0.0, 0.0]), box, r)[0]
    assert ON.pair(pi.astype(np.float32), pj.astype(np.float32), box.astype(np.float32), r)[0]
