"""Two-centre matrix elements by the paper's own quadrature: eq. (9) in prolate spheroidal
coordinates, Gauss-Laguerre in eta and Gauss-Legendre in tau, analytic azimuthal integral (Bessel
function J_{q-q'}, L139), rotated to the collision frame by eq. (8) (L122-127).  SURVEY.md 8(f) NEXT-2.

TEST INFRASTRUCTURE (see oracle/__init__.py).  New module: nothing in oracle/transfer.py changes; the rotation,
the interpolation and the angular functions are the ones pinned there.

Coordinates: foci T (origin) and P (z' = R) of the body frame,
    r_T = R (eta + tau)/2,  r_P = R (eta - tau)/2,   eta in [1, inf),  tau in [-1, 1],
    cos th'_T = (eta tau + 1)/(eta + tau),  cos th'_P = (eta tau - 1)/(eta - tau),
    z' - R/2 = (R/2) eta tau,   rho' = (R/2) sqrt((eta^2 - 1)(1 - tau^2)),   d^3r = (R/2)^3 (eta^2 - tau^2) d eta d tau d phi.
Body-frame integrals (Galerkin reading A1, residual tables A5, conventions of oracle/transfer.py):
    Sb   [(b,q'),(a,q)] = sum_{i,k} W_ik B_{bq'} A_{aq}                    e^{-i v cosTh (R/2) eta_i tau_k} Phi^-_{q-q'}(x_ik)
    Hb_PT[(b,q'),(a,q)] = sum_{i,k} W_ik B_{bq'} (-(Z_P/r_P) A + Ag)_{aq}  (same weight)
    Hb_TP[(a,q),(b,q')] = sum_{i,k} W_ik A_{aq} (-(Z_T/r_T) B + Bg)_{bq'}  e^{+i v cosTh (R/2) eta_i tau_k} Phi^+_{q'-q}(x_ik)
    W_ik = w^eta_i w^tau_k (R/2)^3 (eta_i^2 - tau_k^2),   x_ik = v sinTh (R/2) sqrt((eta_i^2 - 1)(1 - tau_k^2)),
    Phi^{+-}_D(x) = (-+i)^D J_D(x)   (the continuum azimuthal integral of eq. (9); there is no phi' rule here).
Gauss-Laguerre in eta: with x = lam (R/2)(eta - 1),  Int_1^inf f d eta = (2/(lam R)) Int_0^inf f dx
    ~ (2/(lam R)) sum_i w_i e^{x_i} f(1 + 2 x_i/(lam R));  lam = quad["eta_scale"] (1: the weight e^{-(r_T + r_P - R)/2}).
Radial functions: five-point interpolation of the tabulated u, g on the r-grid (transfer.interp5), zero
beyond r_max.
"""
import math

import numpy as np

from .angular import theta_tilde
from .direct import direct_block
from .transfer import interp5, rotation_matrix


def gauss_laguerre_scaled(n: int):
    """Nodes x_i and SCALED weights w_i e^{x_i} of the n-point Gauss-Laguerre rule (library primitive for the nodes;
    the scaled weights from the closed form w_i e^{x_i} = x_i e^{x_i} / ((n + 1) L_{n+1}(x_i))^2, evaluated with
    e^{-x/2}-scaled Laguerre polynomials so that nothing over- or underflows)."""
    from scipy.special import roots_laguerre
    x, _ = roots_laguerre(n)
    # s_k = L_k(x) e^{-x/2}: (k + 1) s_{k+1} = (2k + 1 - x) s_k - k s_{k-1}
    s0 = np.exp(-0.5 * x)
    s1 = (1.0 - x) * s0
    for k in range(1, n + 1):
        s0, s1 = s1, ((2 * k + 1 - x) * s1 - k * s0) / (k + 1)
    return x, x / ((n + 1) * s1) ** 2


def spheroidal_nodes(quad: dict, R: float):
    """(eta_i, w^eta_i, tau_k, w^tau_k) of the rule quad = dict(kind=1, n_rho=n_eta, n_z=n_tau, eta_scale=lam)."""
    lam = float(quad.get("eta_scale", 1.0))
    x, wx = gauss_laguerre_scaled(int(quad["n_rho"]))
    s = 0.5 * lam * R
    tau, wt = np.polynomial.legendre.leggauss(int(quad["n_z"]))
    return 1.0 + x / s, wx / s, tau, wt


def bessel_phi(delta: int, x, sign: int):
    """Phi^{sign}_Delta(x) = (-i sign)^Delta J_Delta(x): the azimuthal integral of eq. (9)."""
    from scipy.special import jv
    return (-1j * sign) ** delta * jv(delta, np.asarray(x, dtype=np.float64))


def body_frame_blocks_spheroidal(prob, b: float, z: float, v: float):
    """(Sb, Hb_PT, Hb_TP) as in transfer.body_frame_blocks, on the spheroidal product nodes; one matrix product per
    Delta = q - q' (library primitive)."""
    T, P = prob.centres
    R = math.hypot(b, z)
    cT, sT = z / R, b / R
    eta, weta, tau, wtau = spheroidal_nodes(prob.quad, R)
    E, Tt = np.meshgrid(eta, tau, indexing="ij")
    W = weta[:, None] * wtau[None, :] * (0.5 * R) ** 3 * (E * E - Tt * Tt)
    rT, rP = 0.5 * R * (E + Tt), 0.5 * R * (E - Tt)
    cTb, cPb = (E * Tt + 1.0) / (E + Tt), (E * Tt - 1.0) / (E - Tt)
    x = v * sT * 0.5 * R * np.sqrt((E * E - 1.0) * (1.0 - Tt * Tt))
    ax = v * cT * 0.5 * R * E * Tt
    phase_m, phase_p = np.exp(-1j * ax), np.exp(+1j * ax)
    h = prob.h

    def tabs(C, rr, cc):
        A, Ag = [], []
        for ir in range(C.n_rad):
            l = int(C.l[ir])
            fu = interp5(C.u[ir], h, rr) / rr
            fg = interp5(C.g[ir], h, rr) / rr
            for q in range(-l, l + 1):
                th = theta_tilde(l, q, cc)
                A.append(fu * th); Ag.append(fg * th)
        return np.array(A), np.array(Ag)

    nn = W.size
    A, Ag = tabs(T, rT, cTb)
    B, Bg = tabs(P, rP, cPb)
    NT, NP = len(A), len(B)
    A = A.reshape(NT, nn); Ag = Ag.reshape(NT, nn); B = B.reshape(NP, nn); Bg = Bg.reshape(NP, nn)
    Ah = -P.Z / rP.reshape(nn) * A + Ag
    Bh = -T.Z / rT.reshape(nn) * B + Bg
    qT = np.array([q for (_, l, q) in T.states()])
    qP = np.array([q for (_, l, q) in P.states()])
    Sb = np.zeros((NP, NT), np.complex128); Hpt = np.zeros((NP, NT), np.complex128); Htp = np.zeros((NT, NP), np.complex128)
    dmax = int(np.max(np.abs(qT)) + np.max(np.abs(qP)))
    for d in range(-dmax, dmax + 1):
        mask = (qT[None, :] - qP[:, None]) == d
        if not mask.any():
            continue
        wm = (W * phase_m * bessel_phi(d, x, -1)).reshape(nn)
        wp = (W * phase_p * bessel_phi(-d, x, +1)).reshape(nn)
        Sb += mask * ((B * wm) @ A.T)
        Hpt += mask * ((B * wm) @ Ah.T)
        Htp += mask.T * ((A * wp) @ Bh.T)
    return Sb, Hpt, Htp


def body_frame_element_loops(prob, beta, alpha, b: float, z: float, v: float, kind: str) -> complex:
    """One body-frame integral of eq. (9) as a plain double loop over the (eta, tau) nodes (the definition; pins the
    matrix-product form above).  beta = (irad, l, q') on P, alpha = (irad, l, q) on T; kind 'S' | 'HPT' | 'HTP'."""
    T, P = prob.centres
    R = math.hypot(b, z)
    cT, sT = z / R, b / R
    eta, weta, tau, wtau = spheroidal_nodes(prob.quad, R)
    (ib, lb, qp), (ia, la, q) = beta, alpha
    sign = +1 if kind == "HTP" else -1
    d = (qp - q) if kind == "HTP" else (q - qp)
    tot = 0.0 + 0.0j
    for e, we in zip(eta, weta):
        for t, wt in zip(tau, wtau):
            rT, rP = 0.5 * R * (e + t), 0.5 * R * (e - t)
            cTb, cPb = (e * t + 1.0) / (e + t), (e * t - 1.0) / (e - t)
            fa = float(interp5(T.u[ia], prob.h, np.array([rT]))[0]) / rT * float(theta_tilde(la, q, np.array([cTb]))[0])
            fb = float(interp5(P.u[ib], prob.h, np.array([rP]))[0]) / rP * float(theta_tilde(lb, qp, np.array([cPb]))[0])
            if kind == "S":
                f = fb * fa
            elif kind == "HPT":
                ga = float(interp5(T.g[ia], prob.h, np.array([rT]))[0]) / rT * float(theta_tilde(la, q, np.array([cTb]))[0])
                f = fb * (-P.Z / rP * fa + ga)
            else:
                gb = float(interp5(P.g[ib], prob.h, np.array([rP]))[0]) / rP * float(theta_tilde(lb, qp, np.array([cPb]))[0])
                f = fa * (-T.Z / rT * fb + gb)
            xx = v * sT * 0.5 * R * math.sqrt(max(0.0, (e * e - 1.0) * (1.0 - t * t)))
            tot += we * wt * (0.5 * R) ** 3 * (e * e - t * t) * f * np.exp(1j * sign * v * cT * 0.5 * R * e * t) * complex(bessel_phi(d, xx, sign))
    return complex(tot)


def two_centre_blocks_spheroidal(prob, b: float, z: float, v: float):
    """Lab-frame S_PT, H_PT [N_P x N_T], H_TP [N_T x N_P] (no time phases): eq. (8) rotation of the eq. (9) integrals."""
    T, P = prob.centres
    R = math.hypot(b, z)
    Theta = math.acos(z / R)
    Sb, Hpt, Htp = body_frame_blocks_spheroidal(prob, b, z, v)
    DT, DP = rotation_matrix(T, Theta), rotation_matrix(P, Theta)
    return DP @ Sb @ DT.T, DP @ Hpt @ DT.T, DT @ Htp @ DP.T


def S_and_H_spheroidal(prob, b: float, z: float, v: float, time_phase: bool = True):
    """(S, H) at R = (b, 0, z) with the two-centre blocks from the spheroidal rule; direct blocks and the assembly exactly
    as oracle/assemble.py (S = [[I, S_PT^H], [S_PT, I]], H = [[D^T, H_TP], [H_PT, D^P]], interaction-picture phases)."""
    T, P = prob.centres
    NT, NP = T.n_states, P.n_states
    r = prob.h * np.arange(prob.Nr + 1)
    DT = direct_block(T, prob.w, r, prob.lambda_max, b, z, v, charge=prob.Z_proj, projectile_centre=False, time_phase=False)
    DP = direct_block(P, prob.w, r, prob.lambda_max, b, z, v, charge=T.Z, projectile_centre=True, time_phase=False)
    S_PT, H_PT, H_TP = two_centre_blocks_spheroidal(prob, b, z, v)
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
