"""The paper's z-grid and Algorithm 1 on an explicit step grid.

TEST INFRASTRUCTURE (see oracle/__init__.py).  New module: oracle/propagate.py (uniform grid, amb. A13) is unchanged.

PAPER.md L67: "the z-grid is constructed according to zgrid[i] = z_min (z_max / z_min)^(i / n_z), zgrid[0] = 0 and
zgrid[-i] = -zgrid[i], with i ranging from 1 to n_z" -- 2 n_z + 1 points, dense near closest approach; typical
z_min = 1e-3, n_z = 500, z_max = 100.  Algorithm 1 (L69-104) advances X from z = zgrid[i] to z_new = zgrid[i+1] with
h = z_new - z and z_mid = z + h/2; M is evaluated 4 n_z + 1 times (L106): once per grid point and once per midpoint.
"""
import numpy as np

from .assemble import S_and_H
from .propagate import rhs


def paper_zgrid(z_min: float, z_max: float, n_z: int) -> np.ndarray:
    """The 2 n_z + 1 points -z_max .. 0 .. +z_max of PAPER.md L67, ascending."""
    pos = np.array([z_min * (z_max / z_min) ** (i / n_z) for i in range(1, n_z + 1)])
    return np.concatenate([-pos[::-1], [0.0], pos])


def propagate_grid(prob, b: float, v: float, zgrid, init_state: int = 0, matrices=None, track_norm: bool = False):
    """Algorithm 1 on the step grid zgrid[0] < ... < zgrid[n].  Returns c(zgrid[n]) (and max |c^H S c - 1|).

    matrices: optional callable z -> (S, H); default oracle.assemble.S_and_H at (b, z, v).
    `count` attribute of the returned evaluations is exposed through matrices wrappers in the tests."""
    zgrid = np.asarray(zgrid, dtype=np.float64)
    one = len(prob.centres) == 1
    if matrices is None:
        def matrices(z):
            return S_and_H(prob, b, float(z), v)
    c = np.zeros(prob.n_tot, dtype=np.complex128)          # lines 1-2
    c[init_state] = 1.0
    S_new, H_new = matrices(zgrid[0])                        # lines 3-4
    drift = 0.0
    for i in range(len(zgrid) - 1):
        z, z_new = zgrid[i], zgrid[i + 1]
        h = z_new - z
        z_mid = z + 0.5 * h                                  # line 13
        S_z, H_z = S_new, H_new                              # line 12: M(z_new) of the previous step is reused
        S_mid, H_mid = matrices(z_mid)
        S_new, H_new = matrices(z_new)
        k1 = rhs(S_z, H_z, c, v, one)
        k2 = rhs(S_mid, H_mid, c + 0.5 * h * k1, v, one)
        k3 = rhs(S_mid, H_mid, c + 0.5 * h * k2, v, one)
        k4 = rhs(S_new, H_new, c + h * k3, v, one)
        c = c + (h / 6.0) * (k1 + 2.0 * k2 + 2.0 * k3 + k4)
        if track_norm:
            drift = max(drift, abs(np.vdot(c, S_new @ c).real - 1.0))
    return (c, drift) if track_norm else c
