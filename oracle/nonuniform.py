"""The hot path on a NON-UNIFORM radial grid ("The grid is denser around the origin to capture finer
details in that region.  The same grid is also used in the computation of the integral in Eq. (7)"; five-point
polynomial interpolation off the grid).  SURVEY.md 8(f) NEXT-3.

TEST INFRASTRUCTURE (see oracle/__init__.py).  New module: the uniform-grid oracle (transfer.interp5, assemble.S_and_H)
is unchanged.  Eq. (7) needs nothing new: direct.radial_F / direct_block already take the grid points r_k and weights
w_k as arrays.  What changes is the interpolation of the tabulated u, g at the quadrature nodes:

    stencil centre j = the grid point nearest to r (the lower one on a tie), clamped to [2, Nr - 2];
    value = sum_{a = j-2 .. j+2} table[a] prod_{c != a} (r - r_c)/(r_a - r_c)     (Lagrange on the actual abscissae);
    zero for r > r_Nr.
"""
import math

import numpy as np

from .angular import theta_tilde
from .direct import direct_block
from .transfer import azimuthal_phi, quadrature_nodes, rotation_matrix


def interp5_grid(table: np.ndarray, rgrid: np.ndarray, r):
    """Five-point Lagrange interpolation of table[k] = u(rgrid[k]) at the points r."""
    r = np.asarray(r, dtype=np.float64)
    Nr = len(rgrid) - 1
    i = np.searchsorted(rgrid, r, side="right")                  # number of grid points <= r
    lo = np.clip(i - 1, 0, Nr - 1)
    hi = lo + 1
    j = np.where((r - rgrid[lo]) <= (rgrid[hi] - r), lo, hi)
    j = np.clip(j, 2, Nr - 2)
    out = np.zeros_like(r)
    for a in range(-2, 3):
        La = np.ones_like(r)
        for c in range(-2, 3):
            if c != a:
                La = La * (r - rgrid[j + c]) / (rgrid[j + a] - rgrid[j + c])
        out = out + La * table[j + a]
    return np.where(r > rgrid[Nr], 0.0, out)


def two_centre_blocks_grid(prob, rgrid, b: float, z: float, v: float):
    """transfer.two_centre_blocks (cylindrical rule, discrete or Bessel azimuth) with the tables interpolated on `rgrid`."""
    T, P = prob.centres
    R = math.hypot(b, z)
    cT, sT = z / R, b / R
    rho, wrho, phi, wphi, zp, wz = quadrature_nodes(prob.quad, R)
    RH, ZZ = np.meshgrid(rho, zp, indexing="ij")
    W = wrho[:, None] * wz[None, :]
    rT = np.sqrt(RH ** 2 + ZZ ** 2)
    rP = np.sqrt(RH ** 2 + (ZZ - R) ** 2)
    cTb, cPb = ZZ / rT, (ZZ - R) / rP
    nn = W.size

    def tabs(C, rr, cc):
        A, Ag = [], []
        for ir in range(C.n_rad):
            l = int(C.l[ir])
            fu = interp5_grid(C.u[ir], rgrid, rr) / rr
            fg = interp5_grid(C.g[ir], rgrid, rr) / rr
            for q in range(-l, l + 1):
                th = theta_tilde(l, q, cc)
                A.append((fu * th).reshape(nn)); Ag.append((fg * th).reshape(nn))
        return np.array(A), np.array(Ag)

    A, Ag = tabs(T, rT, cTb)
    B, Bg = tabs(P, rP, cPb)
    Ah = -P.Z / rP.reshape(nn) * A + Ag
    Bh = -T.Z / rT.reshape(nn) * B + Bg
    x = v * sT * RH
    phase_m = np.exp(-1j * v * cT * (ZZ - 0.5 * R))
    phase_p = np.exp(+1j * v * cT * (ZZ - 0.5 * R))
    rule = prob.quad.get("phi_rule", 0)
    qT = np.array([q for (_, l, q) in T.states()])
    qP = np.array([q for (_, l, q) in P.states()])
    NT, NP = len(qT), len(qP)
    Sb = np.zeros((NP, NT), np.complex128); Hpt = np.zeros((NP, NT), np.complex128); Htp = np.zeros((NT, NP), np.complex128)
    dmax = int(np.max(np.abs(qT)) + np.max(np.abs(qP)))
    for d in range(-dmax, dmax + 1):
        mask = (qT[None, :] - qP[:, None]) == d
        if not mask.any():
            continue
        wm = (W * phase_m * azimuthal_phi(d, x, phi, wphi, -1, rule)).reshape(nn)
        wp = (W * phase_p * azimuthal_phi(-d, x, phi, wphi, +1, rule)).reshape(nn)
        Sb += mask * ((B * wm) @ A.T)
        Hpt += mask * ((B * wm) @ Ah.T)
        Htp += mask.T * ((A * wp) @ Bh.T)
    Theta = math.acos(z / R)
    DT, DP = rotation_matrix(T, Theta), rotation_matrix(P, Theta)
    return DP @ Sb @ DT.T, DP @ Hpt @ DT.T, DT @ Htp @ DP.T


def S_and_H_grid(prob, rgrid, b: float, z: float, v: float, time_phase: bool = True):
    """(S, H) at R = (b, 0, z) for a basis tabulated on `rgrid` with weights prob.w; assembly as oracle/assemble.py."""
    T = prob.centres[0]
    NT = T.n_states
    DT = direct_block(T, prob.w, rgrid, prob.lambda_max, b, z, v, charge=prob.Z_proj, projectile_centre=False, time_phase=False)
    if len(prob.centres) == 1:
        S, H = np.eye(NT, dtype=np.complex128), DT.astype(np.complex128)
    else:
        P = prob.centres[1]
        NP = P.n_states
        DP = direct_block(P, prob.w, rgrid, prob.lambda_max, b, z, v, charge=T.Z, projectile_centre=True, time_phase=False)
        S_PT, H_PT, H_TP = two_centre_blocks_grid(prob, rgrid, b, z, v)
        N = NT + NP
        S = np.eye(N, dtype=np.complex128)
        S[NT:, :NT] = S_PT; S[:NT, NT:] = S_PT.conj().T
        H = np.zeros((N, N), dtype=np.complex128)
        H[:NT, :NT] = DT; H[NT:, NT:] = DP; H[NT:, :NT] = H_PT; H[:NT, NT:] = H_TP
    if time_phase:
        e = np.concatenate([[c.eps[ir] for (ir, _, _) in c.states()] for c in prob.centres])
        ph = np.exp(1j * (e[:, None] - e[None, :]) * z / v)
        S, H = S * ph, H * ph
    return S, H
