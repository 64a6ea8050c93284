"""Hand-constructed inputs shared by the oracle pins and the GPU parity tests (no method arithmetic)."""
import numpy as np


def boundary_pairs(lo, L, r, grid):
    """Particles on a coarse binary grid (every subtraction below is exact in fp32) with partners at distance
    EXACTLY r, one grid step inside and one outside, straight through each face and diagonally through a corner
    image: integer vectors (1,2,2)*r/3 have length exactly r."""
    lo = np.asarray(lo, np.float64)
    pts = []
    base = [np.array([grid, grid, grid]), np.array([L / 2, grid, L - grid]), np.array([L - grid, L - grid, L - grid]),
            np.array([2 * grid, L / 2, L / 2])]
    u = r / 3.0
    vecs = []
    for s in (-1, 1):
        for d in range(3):
            e = np.zeros(3)
            e[d] = s * r
            vecs.append(e)
        for perm in ((1, 2, 2), (2, 1, 2), (2, 2, 1)):
            for sy in (-1, 1):
                for sz in (-1, 1):
                    vecs.append(np.array([s * perm[0], sy * perm[1], sz * perm[2]]) * u)
    for b in base:
        pts.append(b)
        for v in vecs:
            for shrink in (0.0, grid, -grid):          # exactly r, inside, outside (along the vector's first nonzero axis)
                w = v.copy()
                k = int(np.nonzero(w)[0][0])
                w[k] -= np.sign(w[k]) * shrink
                pts.append(np.mod(b + w, L))
    p = np.array(pts)
    return p, lo
