"""Independent numpy/scipy restatements used to PIN the oracle (never the other way round)."""
import itertools

import numpy as np
from numpy.polynomial import chebyshev as npcheb


def np_neighbors(pos, cell, rc, wide=4):
    """All (i, j, shift) with 0 < |r_j + shift.cell - r_i| < rc; shift range fixed and wide."""
    pos = np.asarray(pos, float); cell = np.asarray(cell, float).reshape(3, 3)
    out = []
    rng = range(-wide, wide + 1)
    for i in range(len(pos)):
        for j in range(len(pos)):
            for s in itertools.product(rng, rng, rng):
                if i == j and s == (0, 0, 0):
                    continue
                d = pos[j] - pos[i] + np.array(s, float) @ cell
                if d @ d < rc * rc:
                    out.append((i, j, s, d))
    return out


def np_fk(r, rc, basis_size):
    """Eq. 17-18 with numpy's Chebyshev evaluator: f_k = 1/2 (T_k(x) + 1) fc, k = 0..basis_size."""
    r = np.asarray(r, float)
    x = 2.0 * (r / rc - 1.0) ** 2 - 1.0
    fc = np.where(r < rc, 0.5 * (np.cos(np.pi * r / rc) + 1.0), 0.0)
    out = []
    for k in range(basis_size + 1):
        c = np.zeros(k + 1); c[k] = 1.0
        out.append(0.5 * (npcheb.chebval(x, c) + 1.0) * fc)
    return np.array(out)
