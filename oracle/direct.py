"""Direct (one-centre) coupling matrix elements: eq. (6)-(7) of the paper.

TEST INFRASTRUCTURE (see oracle/__init__.py).

  F^c_lambda(a', a; R) = sum_{k=1}^{Nr} w_k u_{a'}(r_k) u_a(r_k) min(r_k,R)^lambda / max(r_k,R)^{lambda+1}
      -- eq. (7) on the r-grid "also used in the computation of the integral in Eq. (7)" (L148),
         evaluated at the exact R (amb. A9), trapezoid weights (amb. A8), u = r f.
  D^T_{alpha' alpha} = -Z_P e^{i(eps'-eps) z/v} sum_lambda G^lambda P_lambda^mu(cos Theta) F^T_lambda
  D^P_{beta' beta}  = -Z_T e^{i(eps'-eps) z/v} sum_lambda (-1)^lambda G^lambda P_lambda^mu(cos Theta) F^P_lambda
      -- eq. (6) with factorials restored (amb. A3), interaction-picture phase (amb. A2),
         projectile-centre sign (amb. A15); mu = m' - m; cos Theta = z/R; b along +x.
"""
import math

import numpy as np

from .angular import assoc_legendre, direct_angular_coefficient


def radial_F(u_ap, u_a, w, r, R: float, lam: int) -> float:
    """Eq. (7) as the plain grid sum (k = 1..Nr; the r = 0 term vanishes because u(0) = 0)."""
    total = 0.0
    terms = np.empty(len(r) - 1)
    for k in range(1, len(r)):
        rk = r[k]
        lo, hi = (rk, R) if rk < R else (R, rk)
        terms[k - 1] = w[k] * u_ap[k] * u_a[k] * lo ** lam / hi ** (lam + 1)
    total = math.fsum(terms)
    return total


def radial_F_all(centre, w, r, R: float, lambda_max: int) -> np.ndarray:
    """F[lam, a', a] for all radial pairs of one centre (vectorised form of radial_F; same sum)."""
    lo = np.minimum(r[1:], R)
    hi = np.maximum(r[1:], R)
    U = centre.u[:, 1:]
    F = np.zeros((lambda_max + 1, centre.n_rad, centre.n_rad))
    for lam in range(lambda_max + 1):
        V = lo ** lam / hi ** (lam + 1)
        F[lam] = (U * (w[1:] * V)) @ U.T
    return F


def direct_block_loops(centre, w, r, lambda_max: int, b: float, z: float, v: float, charge: float,
                       projectile_centre: bool, time_phase: bool = True) -> np.ndarray:
    """N x N complex block D^T (projectile_centre=False, charge=Z_P) or D^P (True, charge=Z_T).
    Eq. (6) written out element by element (the definition; slow)."""
    R = math.hypot(b, z)
    cosT = z / R
    F = radial_F_all(centre, w, r, R, lambda_max)
    st = centre.states()
    N = len(st)
    D = np.zeros((N, N), dtype=np.complex128)
    for i, (ap, lp, mp) in enumerate(st):
        for j, (a, l, m) in enumerate(st):
            mu = mp - m
            acc = 0.0
            for lam in range(abs(lp - l), min(lp + l, lambda_max) + 1):
                G = direct_angular_coefficient(lp, mp, l, m, lam)
                if G == 0.0:
                    continue
                sgn = (-1) ** lam if projectile_centre else 1
                acc += sgn * G * float(assoc_legendre(lam, mu, cosT)) * F[lam, ap, a]
            ph = np.exp(1j * (centre.eps[ap] - centre.eps[a]) * z / v) if time_phase else 1.0
            D[i, j] = -charge * ph * acc
    return D


_G_MEMO = {}


def angular_table(ls, lambda_max: int):
    """G[lam, i, j] = G^lam_{alpha' alpha} and MU[i, j] = m' - m for the states of a centre with radial
    orbital momenta `ls` (position independent; memoised on (ls, lambda_max))."""
    key = (tuple(int(x) for x in ls), lambda_max)
    if key not in _G_MEMO:
        st = [(ir, l, m) for ir, l in enumerate(key[0]) for m in range(-l, l + 1)]
        N = len(st)
        G = np.zeros((lambda_max + 1, N, N))
        MU = np.zeros((N, N), dtype=np.int64)
        for i, (_, lp, mp) in enumerate(st):
            for j, (_, l, m) in enumerate(st):
                MU[i, j] = mp - m
                for lam in range(abs(lp - l), min(lp + l, lambda_max) + 1):
                    G[lam, i, j] = direct_angular_coefficient(lp, mp, l, m, lam)
        IR = np.array([s_[0] for s_ in st])
        _G_MEMO[key] = (G, MU, IR)
    return _G_MEMO[key]


def direct_block(centre, w, r, lambda_max: int, b: float, z: float, v: float, charge: float,
                 projectile_centre: bool, time_phase: bool = True) -> np.ndarray:
    """Same sums as direct_block_loops with the position-independent G^lam tabulated once:
    D = -charge * phase * sum_lam (+-1)^lam G^lam[i,j] P_lam^{mu_ij}(cos Theta) F_lam[a'_i, a_j]."""
    R = math.hypot(b, z)
    cosT = z / R
    F = radial_F_all(centre, w, r, R, lambda_max)
    G, MU, IR = angular_table(centre.l, lambda_max)
    N = len(IR)
    acc = np.zeros((N, N))
    for lam in range(lambda_max + 1):
        Pl = np.array([float(assoc_legendre(lam, mu, cosT)) if abs(mu) <= lam else 0.0
                       for mu in range(-lambda_max, lambda_max + 1)])
        sgn = (-1) ** lam if projectile_centre else 1
        acc += sgn * G[lam] * Pl[np.clip(MU, -lambda_max, lambda_max) + lambda_max] * (np.abs(MU) <= lam) \
            * F[lam][np.ix_(IR, IR)]
    D = (-charge * acc).astype(np.complex128)
    if time_phase:
        e = centre.eps[IR]
        D = D * np.exp(1j * (e[:, None] - e[None, :]) * z / v)
    return D
