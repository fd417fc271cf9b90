"""Conservative remap of a grid PDF onto a grid of another spacing (TEST INFRASTRUCTURE ONLY).

Needed by the spatial-convergence test of the paper (runs with cell width eta * h* for
eta = 1.25, 1, 0.8, 0.6 are compared with the eta = 0.5 reference through E(t) and BC(t)). The paper does
not say how distributions on DIFFERENT grids are compared; reading A19: the reference is
piecewise constant (density P_c / vol over the cell c), and the mass it puts into cell d of the other
grid is the integral of that density over d, i.e. P_c times the overlap volume fraction, a product of
1-D overlap fractions. Mass is preserved exactly; E and BC are then formed on the common (coarser) grid.

Plain definition, python loops: cell c of grid (origin, h) covers origin + (c -/+ 1/2) h per dimension."""
import itertools
import math

import numpy as np


def overlaps_1d(c, o, h, o2, h2):
    """Cells d of the grid (o2, h2) that the cell c of the grid (o, h) overlaps, with the fraction of c's
    length inside each: [(d, frac), ...]."""
    lo, hi = o + (c - 0.5) * h, o + (c + 0.5) * h
    d_lo = math.floor((lo - o2) / h2 + 0.5)
    d_hi = math.floor((hi - o2) / h2 + 0.5)
    out = []
    for d in range(d_lo, d_hi + 1):
        a, b = max(lo, o2 + (d - 0.5) * h2), min(hi, o2 + (d + 0.5) * h2)
        if b - a > 1e-12 * h:            # (two grid lines that coincide up to rounding make no sliver cell)
            out.append((d, (b - a) / h))
    return out


def resample(keys, p, origin, h, origin2, h2):
    """(keys2 int32 [M, n] sorted lexicographically, p2 float64 [M]) on the grid (origin2, h2)."""
    n = keys.shape[1]
    acc = {}
    for c, pc in zip(keys.tolist(), p.tolist()):
        per_dim = [overlaps_1d(c[j], origin[j], h[j], origin2[j], h2[j]) for j in range(n)]
        for combo in itertools.product(*per_dim):
            d = tuple(x[0] for x in combo)
            w = 1.0
            for x in combo:
                w *= x[1]
            acc[d] = acc.get(d, 0.0) + pc * w
    ks = sorted(acc)
    return np.array(ks, dtype=np.int32).reshape(-1, n), np.array([acc[k] for k in ks])
