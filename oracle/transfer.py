"""Two-centre (overlap / electron-transfer) matrix elements: eq. (8)-(9) structure,
in the cylindrical Gauss-Legendre form BASELINE.json configs[1], [3] fix (amb. A10), Galerkin reading (amb. A1).

TEST INFRASTRUCTURE (see oracle/__init__.py).

Geometry: target at origin, projectile at R = (b, 0, z), v = v z^.
Body frame: z'^ = (sin Th, 0, cos Th), x'^ = (cos Th, 0, -sin Th), y'^ = y^, origin at T.
Cylindrical body coordinates (rho', phi', z'):
    r_T = sqrt(rho'^2 + z'^2),  r_P = sqrt(rho'^2 + (z'-R)^2),
    cos th'_T = z'/r_T,  cos th'_P = (z'-R)/r_P,
    z_m = (z' - R/2) cos Th - rho' cos phi' sin Th      (lab z of the electron from the midpoint).

Integrals (no time phases here; they are applied in assemble.py):
    S_PT [beta,alpha] = Int conj psi_beta(r_P) e^{-i v z_m} psi_alpha(r_T) d^3r
    H_PT [beta,alpha] = Int conj psi_beta(r_P) e^{-i v z_m} [ -(Z_P/r_P) psi_alpha + psi^g_alpha ](r_T) d^3r
    H_TP [alpha,beta] = Int conj psi_alpha(r_T) e^{+i v z_m} [ -(Z_T/r_T) psi_beta + psi^g_beta ](r_P) d^3r
with psi = (u/r) Y_lm, psi^g = (g/r) Y_lm, g = (H_c - eps) u (amb. A5).

Two implementations of the same discrete sums:
  L0  lab-frame triple loop over the product nodes with lab-frame spherical harmonics (the definition);
  L1  factorised: body-frame (rho', z') sums with the discrete azimuthal sum Phi_Delta, then the
      Wigner rotation of eq. (8).  L0 == L1 algebraically for the same nodes.
"""
import math

import numpy as np

from .angular import sph_harm, theta_tilde, wigner_small_d


def gauss_legendre(n: int, a: float, b: float):
    """n-point Gauss-Legendre nodes/weights mapped to [a, b] (library primitive: numpy leggauss)."""
    x, w = np.polynomial.legendre.leggauss(n)
    return 0.5 * (b - a) * x + 0.5 * (b + a), 0.5 * (b - a) * w


def quadrature_nodes(quad: dict, R: float):
    """Node layout of amb. A10: rho' one panel on [0, rho_max]; phi' one panel on [0, 2 pi];
    z' three panels [-z_pad, 0], [0, R], [R, R + z_pad] with n_z/4, n_z/2, n_z/4 nodes.
    Returns (rho, w_rho [already times rho], phi, w_phi, zp, w_z)."""
    rho, wr = gauss_legendre(quad["n_rho"], 0.0, quad["rho_max"])
    phi, wp = gauss_legendre(quad["n_phi"], 0.0, 2.0 * math.pi)
    nz = quad["n_z"]
    zs, wz = [], []
    for n_, (a, c) in zip((nz // 4, nz // 2, nz // 4), ((-quad["z_pad"], 0.0), (0.0, R), (R, R + quad["z_pad"]))):
        x, w = gauss_legendre(n_, a, c)
        zs.append(x); wz.append(w)
    return rho, wr * rho, phi, wp, np.concatenate(zs), np.concatenate(wz)


def interp5(table: np.ndarray, h: float, r):
    """Five-point Lagrange interpolation of a reduced radial table at r (amb. A12).

    table[k] = u(k h), k = 0..Nr.  Stencil k = j-2..j+2 with j = clamp(round(r/h), 2, Nr-2);
    returns 0 for r > r_max = Nr h."""
    r = np.asarray(r, dtype=np.float64)
    Nr = len(table) - 1
    j = np.clip(np.floor(r / h + 0.5).astype(np.int64), 2, Nr - 2)
    t = r / h - j                      # position in units of h relative to the stencil centre
    out = np.zeros_like(r)
    offs = (-2, -1, 0, 1, 2)
    for a in offs:
        La = np.ones_like(r)
        for c in offs:
            if c != a:
                La = La * (t - c) / (a - c)
        out = out + La * table[j + a]
    return np.where(r > Nr * h, 0.0, out)


def azimuthal_phi(delta: int, x, phi, w_phi, sign: int, phi_rule: int = 0):
    """Phi^{sign}_Delta(x) = (1/2 pi) sum_j w_j e^{i Delta phi_j} e^{-i sign x cos phi_j}
    for the factor e^{i sign v z_m}  (z_m contains -rho' cos phi' sin Th, x = v rho' sin Th).
    phi_rule = 1 replaces the discrete sum by its continuum limit (-i sign)^Delta J_Delta(x) (eq. (9))."""
    x = np.asarray(x, dtype=np.float64)
    if phi_rule == 1:
        from scipy.special import jv
        return (-1j * sign) ** delta * jv(delta, x)
    out = np.zeros(x.shape, dtype=np.complex128)
    for pj, wj in zip(phi, w_phi):
        out = out + wj * np.exp(1j * delta * pj) * np.exp(-1j * sign * x * math.cos(pj))
    return out / (2.0 * math.pi)


def lab_frame_element(prob, beta, alpha, b: float, z: float, v: float, kind: str) -> complex:
    """L0: the definition.  beta = (irad, l, m) on the projectile centre, alpha on the target centre.

    kind: 'S'    -> Int conj psi_beta(r_P) e^{-i v z_m} psi_alpha(r_T)
          'HPT'  -> Int conj psi_beta(r_P) e^{-i v z_m} [-(Z_P/r_P) psi_alpha + psi^g_alpha](r_T)
          'HTP'  -> Int conj psi_alpha(r_T) e^{+i v z_m} [-(Z_T/r_T) psi_beta + psi^g_beta](r_P)
    Triple loop over (rho', phi', z') product nodes, lab-frame Y_lm at every node."""
    T, P = prob.centres
    R = math.hypot(b, z)
    cT, sT = z / R, b / R
    rho, wrho, phi, wphi, zp, wz = quadrature_nodes(prob.quad, R)
    ib, lb, mb = beta
    ia, la, ma = alpha
    h = prob.h
    total = 0.0 + 0.0j
    for i, (rh, wr_) in enumerate(zip(rho, wrho)):
        for pj, wp_ in zip(phi, wphi):
            xb, yb = rh * math.cos(pj), rh * math.sin(pj)
            # lab coordinates of body point (xb, yb, zb): zb z'^ + xb x'^ + yb y^
            zb = zp
            XT, YT, ZT = zb * sT + xb * cT, yb * np.ones_like(zb), zb * cT - xb * sT
            zbP = zp - R
            XP, YP, ZP = zbP * sT + xb * cT, yb * np.ones_like(zb), zbP * cT - xb * sT
            zm = (zp - 0.5 * R) * cT - xb * sT
            rT = np.sqrt(rh * rh + zp * zp)
            rP = np.sqrt(rh * rh + (zp - R) ** 2)
            YlmT = sph_harm(la, ma, ZT / rT, np.arctan2(YT, XT))
            YlmP = sph_harm(lb, mb, ZP / rP, np.arctan2(YP, XP))
            uT = interp5(T.u[ia], h, rT); uP = interp5(P.u[ib], h, rP)
            if kind == "S":
                f = np.conj(uP / rP * YlmP) * np.exp(-1j * v * zm) * (uT / rT * YlmT)
            elif kind == "HPT":
                gT = interp5(T.g[ia], h, rT)
                f = np.conj(uP / rP * YlmP) * np.exp(-1j * v * zm) * ((-P.Z / rP * uT + gT) / rT * YlmT)
            elif kind == "HTP":
                gP = interp5(P.g[ib], h, rP)
                f = np.conj(uT / rT * YlmT) * np.exp(+1j * v * zm) * ((-T.Z / rT * uP + gP) / rP * YlmP)
            else:
                raise ValueError(kind)
            total += wr_ * wp_ * np.sum(wz * f)
    return complex(total)


def body_frame_tables(prob, R: float):
    """Node tables on the (rho', z') product grid (the "component kernels" of PAPER.md L148).

    Returns dict with W[i,k] (weights incl. rho'), rT, rP, and per centre the lists
      A [(a,q)] = u_a(r_T)/r_T Theta~_{l_a q}(cos th'_T),        Ag = g_a(r_T)/r_T Theta~ ...
      B [(b,q')] = u_b(r_P)/r_P Theta~_{l_b q'}(cos th'_P),      Bg likewise,
    indexed in state order (irad, then q = -l..l)."""
    T, P = prob.centres
    rho, wrho, phi, wphi, zp, wz = quadrature_nodes(prob.quad, R)
    RH, ZZ = np.meshgrid(rho, zp, indexing="ij")
    W = wrho[:, None] * wz[None, :]
    rT = np.sqrt(RH ** 2 + ZZ ** 2)
    rP = np.sqrt(RH ** 2 + (ZZ - R) ** 2)
    cTb, cPb = ZZ / rT, (ZZ - R) / rP
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

    A, Ag = tabs(T, rT, cTb)
    B, Bg = tabs(P, rP, cPb)
    return dict(W=W, rT=rT, rP=rP, RH=RH, ZZ=ZZ, A=A, Ag=Ag, B=B, Bg=Bg, phi=phi, wphi=wphi)


def body_frame_blocks_loops(prob, b: float, z: float, v: float):
    """L1 step 1 (element-by-element loops; the definition): body-frame integrals I[(b,q'),(a,q)] of SURVEY.md App. A.3 (eq. (9) structure).

    Returns (Sb, Hb_PT, Hb_TP) where
      Sb   [(b,q'),(a,q)] = sum_nodes W B A                          e^{-i v cosTh (z'-R/2)} Phi^-_{q-q'}
      Hb_PT[(b,q'),(a,q)] = sum_nodes W B (-(Z_P/r_P) A + Ag)       e^{-i v cosTh (z'-R/2)} Phi^-_{q-q'}
      Hb_TP[(a,q),(b,q')] = sum_nodes W A (-(Z_T/r_T) B + Bg)       e^{+i v cosTh (z'-R/2)} Phi^+_{q'-q}
    (conj Y_{l_b q'} Y_{l_a q} gives e^{i(q-q')phi}/(2 pi), hence Delta = q - q' for <P|..|T>;
     conj Y_{l_a q} Y_{l_b q'} gives Delta = q' - q for <T|..|P>.)"""
    T, P = prob.centres
    R = math.hypot(b, z)
    cT, sT = z / R, b / R
    tb = body_frame_tables(prob, R)
    W, RH, ZZ = tb["W"], tb["RH"], tb["ZZ"]
    x = v * sT * RH
    phase_m = np.exp(-1j * v * cT * (ZZ - 0.5 * R))
    phase_p = np.exp(+1j * v * cT * (ZZ - 0.5 * R))
    rule = prob.quad.get("phi_rule", 0)
    qT = [q for (_, l, q) in T.states()]
    qP = [q for (_, l, q) in P.states()]
    dmax = max(abs(q) for q in qT) + max(abs(q) for q in qP)
    Phi_m = {d: azimuthal_phi(d, x, tb["phi"], tb["wphi"], -1, rule) for d in range(-dmax, dmax + 1)}
    Phi_p = {d: azimuthal_phi(d, x, tb["phi"], tb["wphi"], +1, rule) for d in range(-dmax, dmax + 1)}
    NT, NP = len(qT), len(qP)
    Sb = np.zeros((NP, NT), np.complex128)
    Hpt = np.zeros((NP, NT), np.complex128)
    Htp = np.zeros((NT, NP), np.complex128)
    A, Ag, B, Bg = tb["A"], tb["Ag"], tb["B"], tb["Bg"]
    Ah = -P.Z / tb["rP"] * A + Ag          # [-(Z_P/r_P) psi_alpha + psi^g_alpha]
    Bh = -T.Z / tb["rT"] * B + Bg          # [-(Z_T/r_T) psi_beta + psi^g_beta]
    for ib in range(NP):
        for ia in range(NT):
            d = qT[ia] - qP[ib]
            wm = W * phase_m * Phi_m[d]
            Sb[ib, ia] = np.sum(wm * B[ib] * A[ia])
            Hpt[ib, ia] = np.sum(wm * B[ib] * Ah[ia])
            Htp[ia, ib] = np.sum(W * phase_p * Phi_p[-d] * A[ia] * Bh[ib])
    return Sb, Hpt, Htp


def body_frame_blocks(prob, b: float, z: float, v: float):
    """Same sums as body_frame_blocks_loops, with the node sum of every (q', q) group done by one
    matrix product (library primitive): for each Delta = q - q',
        Sb|_Delta = B (W phase_- Phi^-_Delta) A^T,  Hb_PT|_Delta = B (..) Ah^T,  Hb_TP|_Delta = A (W phase_+ Phi^+_{-Delta}) Bh^T."""
    T, P = prob.centres
    R = math.hypot(b, z)
    cT, sT = z / R, b / R
    tb = body_frame_tables(prob, R)
    W, RH, ZZ = tb["W"], tb["RH"], tb["ZZ"]
    x = v * sT * RH
    phase_m = np.exp(-1j * v * cT * (ZZ - 0.5 * R))
    phase_p = np.exp(+1j * v * cT * (ZZ - 0.5 * R))
    rule = prob.quad.get("phi_rule", 0)
    qT = np.array([q for (_, l, q) in T.states()])
    qP = np.array([q for (_, l, q) in P.states()])
    NT, NP = len(qT), len(qP)
    nn = W.size
    A = tb["A"].reshape(NT, nn); Ag = tb["Ag"].reshape(NT, nn)
    B = tb["B"].reshape(NP, nn); Bg = tb["Bg"].reshape(NP, nn)
    Ah = -P.Z / tb["rP"].reshape(nn) * A + Ag
    Bh = -T.Z / tb["rT"].reshape(nn) * B + Bg
    Sb = np.zeros((NP, NT), np.complex128)
    Hpt = np.zeros((NP, NT), np.complex128)
    Htp = np.zeros((NT, NP), np.complex128)
    dmax = int(np.max(np.abs(qT)) + np.max(np.abs(qP)))
    for d in range(-dmax, dmax + 1):
        mask = (qT[None, :] - qP[:, None]) == d          # [NP, NT]
        if not mask.any():
            continue
        wm = (W * phase_m * azimuthal_phi(d, x, tb["phi"], tb["wphi"], -1, rule)).reshape(nn)
        wp = (W * phase_p * azimuthal_phi(-d, x, tb["phi"], tb["wphi"], +1, rule)).reshape(nn)
        Sb += mask * ((B * wm) @ A.T)
        Hpt += mask * ((B * wm) @ Ah.T)
        Htp += mask.T * ((A * wp) @ Bh.T)
    return Sb, Hpt, Htp


def rotation_matrix(centre, Theta: float) -> np.ndarray:
    """Block-diagonal matrix Dm[(irad,m),(irad,q)] = d^{l}_{m q}(Theta) (eq. (8))."""
    st = centre.states()
    N = len(st)
    Dm = np.zeros((N, N))
    for i, (ir, l, m) in enumerate(st):
        for j, (jr, l2, q) in enumerate(st):
            if ir == jr:
                Dm[i, j] = wigner_small_d(l, m, q, Theta)
    return Dm


def two_centre_blocks(prob, b: float, z: float, v: float):
    """L1: lab-frame S_PT [N_P x N_T], H_PT [N_P x N_T], H_TP [N_T x N_P], no time phases.

    Eq. (8): K_{beta alpha} = sum_{q' q} d^{l_beta}_{m_beta q'}(Th) d^{l_alpha}_{m_alpha q}(Th) S^body_{(b q'),(a q)}."""
    T, P = prob.centres
    R = math.hypot(b, z)
    Theta = math.acos(z / R)
    Sb, Hpt, Htp = body_frame_blocks(prob, b, z, v)
    DT = rotation_matrix(T, Theta)
    DP = rotation_matrix(P, Theta)
    return DP @ Sb @ DT.T, DP @ Hpt @ DT.T, DT @ Htp @ DP.T
