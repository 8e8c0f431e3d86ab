"""Pins for oracle/direct.py: closed forms (hydrogen), brute-force 3-D quadrature, symmetries."""
import math

import numpy as np
import pytest

from oracle import angular as ang
from oracle.direct import radial_F, radial_F_all, direct_block, direct_block_loops
from wpccc_inputs import make_problem, radial_grid
from wpccc_inputs.configs import bound_only_centre

RAD = [(1, 0), (2, 0), (3, 0), (2, 1), (3, 1), (3, 2)]     # 1s 2s 3s 2p 3p 3d


def closed_F(name, R):
    """Continuum values of eq. (7) for hydrogen (sympy-derived closed forms)."""
    e = math.exp
    if name == "1s1s0":
        return (e(2 * R) - R - 1) * e(-2 * R) / R
    if name == "1s2s0":
        return 2 * math.sqrt(2) * (3 * R + 2) * e(-1.5 * R) / 27
    if name == "1s2p1":
        return 2 * math.sqrt(6) * (64 * e(1.5 * R) - 27 * R**3 - 72 * R**2 - 96 * R - 64) * e(-1.5 * R) / (243 * R**2)
    if name == "2p2p2":
        return 5 * (144 * e(R) - R**5 - 6 * R**4 - 24 * R**3 - 72 * R**2 - 144 * R - 144) * e(-R) / (24 * R**3)
    if name == "1s3d2":
        return (math.sqrt(30) * (2187 * e(4 * R / 3) - 64 * R**5 - 288 * R**4 - 864 * R**3 - 1944 * R**2 - 2916 * R - 2187)
                * e(-4 * R / 3) / (6912 * R**3))
    raise KeyError(name)


def test_closed_forms_match_numerical_integration():
    """The closed forms themselves, against scipy.integrate.quad of eq. (7) with analytic R_nl."""
    from scipy.integrate import quad
    from wpccc_inputs import hydrogenic_bound_u
    R = 1.5
    for name, (n1, l1), (n0, l0), lam in [("1s1s0", (1, 0), (1, 0), 0), ("1s2s0", (1, 0), (2, 0), 0),
                                          ("1s2p1", (1, 0), (2, 1), 1), ("2p2p2", (2, 1), (2, 1), 2),
                                          ("1s3d2", (1, 0), (3, 2), 2)]:
        f = lambda r: float(hydrogenic_bound_u(n1, l1, 1.0, np.array([r]))[0] * hydrogenic_bound_u(n0, l0, 1.0, np.array([r]))[0]
                            * min(r, R) ** lam / max(r, R) ** (lam + 1))
        val = quad(f, 0, R, epsabs=1e-13, epsrel=1e-13)[0] + quad(f, R, 80, epsabs=1e-13, epsrel=1e-13)[0]
        assert val == pytest.approx(closed_F(name, R), abs=1e-11)


@pytest.mark.parametrize("name,ia,ib,lam", [("1s1s0", 0, 0, 0), ("1s2s0", 0, 1, 0), ("1s2p1", 0, 3, 1),
                                            ("2p2p2", 3, 3, 2), ("1s3d2", 0, 5, 2)])
def test_radial_F_converges_to_closed_form(name, ia, ib, lam):
    """Grid sum of eq. (7): error vs the continuum closed form is O(h^2) (kink of V_lambda at r=R, amb. A9)."""
    R = 1.5 + 0.013          # off-grid for every h below
    errs = []
    for Nr, h in ((1000, 0.1), (2000, 0.05), (4000, 0.025)):
        C = bound_only_centre(1.0, RAD, Nr, h)
        r, w = radial_grid(Nr, h)
        errs.append(abs(radial_F(C.u[ia], C.u[ib], w, r, R, lam) - closed_F(name, R)))
    assert errs[1] < 2e-4 and errs[2] < errs[1] < errs[0]
    # second-order: halving h twice reduces the error by ~16 (allow 6..40: the kink term oscillates with (R/h mod 1))
    assert 6.0 < errs[0] / errs[2] < 60.0


def test_radial_F_all_equals_loop_and_is_symmetric():
    C = bound_only_centre(1.0, RAD, 600, 0.1)
    r, w = radial_grid(600, 0.1)
    F = radial_F_all(C, w, r, 2.37, 4)
    for lam in (0, 1, 3):
        for a, b in ((0, 0), (0, 3), (4, 5), (2, 1)):
            assert F[lam, a, b] == pytest.approx(radial_F(C.u[a], C.u[b], w, r, 2.37, lam), rel=1e-13, abs=1e-16)
    np.testing.assert_allclose(F, np.transpose(F, (0, 2, 1)), atol=1e-17)


def test_radial_F_separable_form():
    """V_lam = r^lam/R^(lam+1) below R and R^lam/r^(lam+1) above: prefix/suffix sums give the same number."""
    C = bound_only_centre(1.0, RAD, 800, 0.05)
    r, w = radial_grid(800, 0.05)
    R, lam = 3.3333, 2
    p = w * C.u[1] * C.u[4]
    below = r < R
    alt = np.sum(p[below] * r[below] ** lam) / R ** (lam + 1) + R ** lam * np.sum(p[~below][1:] / r[~below][1:] ** (lam + 1)) \
        + R ** lam * p[~below][0] / r[~below][0] ** (lam + 1)
    assert radial_F(C.u[1], C.u[4], w, r, R, lam) == pytest.approx(alt, rel=1e-13)


def _problem(Nr=2000, h=0.05, lam=4):
    C = bound_only_centre(1.0, RAD, Nr, h)
    return C, make_problem([C], 1.0, Nr, h, lam)


def test_direct_1s1s_closed_form():
    """<1s| -1/|r-R| |1s> = -(1/R)(1 - (1+R) e^{-2R})  (textbook); grid error O(h^2)."""
    C, prob = _problem(4000, 0.0125)
    r = prob.h * np.arange(prob.Nr + 1)
    for b, z in ((0.7, 1.1), (2.0, -3.0)):
        R = math.hypot(b, z)
        D = direct_block(C, prob.w, r, 4, b, z, 2.0, 1.0, False, time_phase=False)
        assert D[0, 0].real == pytest.approx(-(1 / R) * (1 - (1 + R) * math.exp(-2 * R)), abs=3e-5)
        assert D[0, 0].imag == 0.0


def test_direct_block_table_equals_loops_and_symmetries():
    C, prob = _problem(500, 0.1)
    r = prob.h * np.arange(prob.Nr + 1)
    for proj in (False, True):
        D1 = direct_block(C, prob.w, r, 4, 0.9, -0.4, 1.3, 1.0, proj)
        D2 = direct_block_loops(C, prob.w, r, 4, 0.9, -0.4, 1.3, 1.0, proj)
        np.testing.assert_allclose(D1, D2, rtol=0, atol=1e-16)
        np.testing.assert_allclose(D1, D1.conj().T, rtol=0, atol=1e-16)          # Hermitian
        D0 = direct_block(C, prob.w, r, 4, 0.9, -0.4, 1.3, 1.0, proj, time_phase=False)
        assert np.abs(D0.imag).max() == 0.0                                       # real symmetric without phase
    # D^P(R) is D^T evaluated with the perturbing charge at -R: (-1)^lam  <=>  (b,z) -> (-b,-z); with b>=0 convention
    # this equals cos Theta -> -cos Theta and mu -> sign (-1)^mu; check through parity: P_lam^mu(-x) = (-1)^(lam+mu) P_lam^mu(x)
    DT = direct_block(C, prob.w, r, 4, 0.9, 0.4, 1.3, 1.0, False, time_phase=False).real
    DP = direct_block(C, prob.w, r, 4, 0.9, -0.4, 1.3, 1.0, True, time_phase=False).real
    st = C.states()
    sign = np.array([[(-1) ** (mp - m) for (_, _, m) in st] for (_, _, mp) in st])
    np.testing.assert_allclose(DP, sign * DT, atol=1e-16)


def _brute_force_direct(state_p, state, b, z, n_eta=70, n_tau=70, n_phi=48):
    """<psi'| -1/|r - R| |psi> by 3-D quadrature in prolate spheroidal coordinates with foci at the target
    nucleus and the projectile (removes the Coulomb singularity), lab-frame Y_lm at every node, analytic R_nl."""
    from scipy.special import roots_laguerre, roots_legendre
    from wpccc_inputs import hydrogenic_bound_u
    (n1, l1, m1), (n0, l0, m0) = state_p, state
    R = math.hypot(b, z)
    cT, sT = z / R, b / R
    xe, we = roots_laguerre(n_eta)
    xt, wt = roots_legendre(n_tau)
    s = 1.2 * R / 2                                   # exponential scale ~ e^{-(r_T)(1/n1+1/n0)}
    eta = 1 + xe / s
    weta = we * np.exp(xe) / s
    E, T = np.meshgrid(eta, xt, indexing="ij")
    rT = R * (E + T) / 2
    rP = R * (E - T) / 2
    vol = (R / 2) ** 3 * (E**2 - T**2)
    zb = R * (E * T + 1) / 2                          # along the T->P axis, origin at T
    rho = (R / 2) * np.sqrt(np.maximum(0, (E**2 - 1) * (1 - T**2)))
    phis = 2 * math.pi * (np.arange(n_phi) + 0.5) / n_phi
    tot = 0.0 + 0.0j
    u1 = hydrogenic_bound_u(n1, l1, 1.0, rT.ravel()).reshape(rT.shape) / rT
    u0 = hydrogenic_bound_u(n0, l0, 1.0, rT.ravel()).reshape(rT.shape) / rT
    for ph in phis:
        xb, yb = rho * math.cos(ph), rho * math.sin(ph)
        X, Y, Z = zb * sT + xb * cT, yb, zb * cT - xb * sT        # body -> lab (App. A.1 frame)
        Y1 = ang.sph_harm(l1, m1, Z / rT, np.arctan2(Y, X))
        Y0 = ang.sph_harm(l0, m0, Z / rT, np.arctan2(Y, X))
        tot += np.sum(weta[:, None] * wt[None, :] * vol * np.conj(u1 * Y1) * (-1.0 / rP) * (u0 * Y0)) * (2 * math.pi / n_phi)
    return tot


@pytest.mark.parametrize("sp,s0", [((1, 0, 0), (1, 0, 0)), ((1, 0, 0), (2, 1, 0)), ((1, 0, 0), (2, 1, 1)),
                                   ((2, 1, -1), (2, 1, 1)), ((2, 1, 0), (3, 2, 1)), ((3, 2, 0), (2, 1, 1))])
def test_direct_vs_brute_force_3d(sp, s0):
    """eq. (6)-(7) (factorials restored, amb. A3) against brute-force 3-D quadrature of the definition."""
    b, z = 0.7, 1.1
    C, prob = _problem(8000, 0.005)                    # fine grid: O(h^2) kink error ~ 4e-7
    r = prob.h * np.arange(prob.Nr + 1)
    D = direct_block(C, prob.w, r, 4, b, z, 1.0, 1.0, False, time_phase=False)
    st = C.states()
    nl = {(n, l): i for i, (n, l) in enumerate(RAD)}
    i = st.index((nl[(sp[0], sp[1])], sp[1], sp[2]))
    j = st.index((nl[(s0[0], s0[1])], s0[1], s0[2]))
    ref = _brute_force_direct(sp, s0, b, z)
    assert abs(ref.imag) < 1e-12
    assert D[i, j].real == pytest.approx(ref.real, abs=2e-6)


def test_direct_golden_values_survey_B2():
    """SURVEY.md App. B.2 (independent prototype, converged spheroidal brute force): values at b=0.7, z=1.1."""
    vals = {((1, 0, 0), (1, 0, 0)): -0.63673035542, ((1, 0, 0), (2, 1, 0)): -0.066202384599,
            ((1, 0, 0), (2, 1, 1)): +0.029789553233, ((2, 1, -1), (2, 1, 1)): +0.0043115592951,
            ((3, 2, -2), (3, 2, 2)): -7.45399234e-06}
    for (sp, s0), ref in vals.items():
        assert _brute_force_direct(sp, s0, 0.7, 1.1).real == pytest.approx(ref, abs=2e-9)
