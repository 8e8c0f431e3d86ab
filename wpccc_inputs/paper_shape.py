"""The paper's own benchmark workload, as far as the text fixes it: p + H(1s) at 100 keV (v = 2),
the z-grid from -300 to 300 with 6001 points, eight impact parameters per job, and the basis grown through l_max:
one-centre N = 42 (l_max = 0) ... 4257 (l_max = 10), two-centre N = 60 ... 1910 (l_max = 5), i.e. N_l = N_0 - l radial
functions per l with all m kept (N_0 = 42, and 30 per centre) -- SURVEY.md section 4.  The composition of the N_0 - l
functions is not stated; here: bound states n = l+1 .. n_max and N_0 - n_max wave-packet bins in k in [0, 4] for every l
(n_max = 11 and 31 bins for one centre, n_max = 6 and 24 bins for two), which reproduces the printed sizes exactly.
Input generation only (no method arithmetic); SURVEY.md 8(f) NEXT-3.
"""
from __future__ import annotations

import numpy as np

from .basis import make_centre, make_problem
from .configs import log_spaced

V_100KEV = 2.0
SIZES_1C = {l: sum((2 * j + 1) * (42 - j) for j in range(l + 1)) for l in range(11)}       # 42 .. 4257
SIZES_2C = {l: 2 * sum((2 * j + 1) * (30 - j) for j in range(l + 1)) for l in range(6)}    # 60 .. 1910


def paper_zgrid_points(z_min: float = 1e-3, z_max: float = 300.0, n_z: int = 3000) -> np.ndarray:
    """The 2 n_z + 1 = 6001 points of P:L154 on the geometric grid of P:L67 (zgrid[+-i] = +-z_min (z_max/z_min)^(i/n_z), zgrid[0] = 0)."""
    pos = z_min * (z_max / z_min) ** (np.arange(1, n_z + 1) / n_z)
    return np.concatenate([-pos[::-1], [0.0], pos])


def paper_problem(two_centre: bool, l_max: int, Nr: int = 2000, h: float = 0.05, quad: dict | None = None, nk: int = 16, sub: int = 4):
    """(Problem, run) of the paper-shaped workload at this l_max; run = dict(b[8], v[8], zgrid[6001])."""
    if two_centre:
        n_max, bins, k_max = 6, 24, 4.0
        quad = quad or dict(n_rho=64, n_phi=16, n_z=128, rho_max=40.0, z_pad=40.0, phi_rule=0)
    else:
        n_max, bins, k_max = 11, 31, 4.0
    centres = [make_centre(1.0, l_max, n_max, bins, k_max, Nr, h, nk=nk, sub=sub) for _ in range(2 if two_centre else 1)]
    prob = make_problem(centres, 1.0, Nr, h, 2 * l_max, quad=quad if two_centre else None, meta=dict(config="paper-shape", l_max=l_max))
    want = (SIZES_2C if two_centre else SIZES_1C)[l_max]
    assert prob.n_tot == want, (prob.n_tot, want)
    b = log_spaced(0.2, 12.0, 8)
    return prob, dict(b=b, v=np.full(8, V_100KEV), zgrid=paper_zgrid_points())


def exponential_grid(Nr: int, r_max: float = 100.0, a: float = 4.0) -> np.ndarray:
    """r_k = r_max (e^{a k / Nr} - 1)/(e^a - 1), k = 0..Nr: "denser around the origin"; a = 4: first spacing
    ~ r_max a / (Nr (e^a - 1)), last spacing ~ r_max a / Nr."""
    k = np.arange(Nr + 1, dtype=np.float64)
    r = r_max * np.expm1(a * k / Nr) / np.expm1(a)
    r[0] = 0.0
    return r


def trapezoid_weights(r: np.ndarray) -> np.ndarray:
    """w_0 = 0 (the integrand r^2 f f' V vanishes at the origin), w_k = (r_{k+1} - r_{k-1})/2, w_Nr = (r_Nr - r_{Nr-1})/2."""
    w = np.zeros_like(r)
    w[1:-1] = 0.5 * (r[2:] - r[:-2])
    w[-1] = 0.5 * (r[-1] - r[-2])
    return w


def resample_problem(prob, rgrid: np.ndarray):
    """The basis of `prob` (tabulated on a fine uniform grid) sampled on the non-uniform grid `rgrid` (cubic splines),
    trapezoid weights of that grid, every function renormalised by its grid norm (reading A6).  The returned Problem carries
    the grid as the attribute `rgrid`; its `h` is only nominal."""
    from scipy.interpolate import CubicSpline
    from .basis import Centre
    rf = prob.h * np.arange(prob.Nr + 1)
    assert rgrid[-1] <= rf[-1] + 1e-12
    w = trapezoid_weights(rgrid)
    centres = []
    for c in prob.centres:
        U = CubicSpline(rf, c.u, axis=1)(rgrid)
        G = CubicSpline(rf, c.g, axis=1)(rgrid)
        U[:, 0] = 0.0; G[:, 0] = 0.0
        nrm = np.sqrt((w[None, :] * U * U).sum(1))
        centres.append(Centre(Z=c.Z, l=c.l.copy(), eps=c.eps.copy(), kind=c.kind.copy(), nq=c.nq.copy(),
                              u=np.ascontiguousarray(U / nrm[:, None]), g=np.ascontiguousarray(G / nrm[:, None])))
    Nr = len(rgrid) - 1
    out = make_problem(centres, prob.Z_proj, Nr, float(rgrid[-1] / Nr), prob.lambda_max, quad=prob.quad, meta=dict(prob.meta, grid="non-uniform"))
    out.w = w
    out.rgrid = np.ascontiguousarray(rgrid, dtype=np.float64)
    return out
