"""Pins for oracle/spheroidal.py (eq. (9) of the paper in its own prolate-spheroidal form,
Gauss-Laguerre x Gauss-Legendre + analytic Bessel azimuth): quadrature exactness, the loop
definition, SURVEY.md App. B.1 closed forms and App. B.2 printed values, the converged cylindrical rule of
oracle/transfer.py (a different coordinate system, node set and azimuthal treatment), and the Galerkin identity."""
import math

import numpy as np
import pytest

from oracle import spheroidal as sph
from oracle import transfer as tr
from wpccc_inputs import make_problem, tiny_problem
from wpccc_inputs.configs import bound_only_centre

RAD = [(1, 0), (2, 0), (2, 1)]
SPH = dict(kind=1, n_rho=64, n_phi=1, n_z=64, rho_max=40.0, z_pad=40.0, phi_rule=1, eta_scale=1.0)
CYL = dict(n_rho=160, n_phi=16, n_z=320, rho_max=40.0, z_pad=40.0, phi_rule=1)


def _bound_problem(quad, Nr=4000, h=0.0125, ZP=1.0):
    T = bound_only_centre(1.0, RAD, Nr, h)
    P = bound_only_centre(ZP, RAD, Nr, h)
    return make_problem([T, P], ZP, Nr, h, 2, quad=quad)


def test_scaled_gauss_laguerre_is_exact_for_polynomials():
    for n in (5, 24, 64, 96):
        x, wx = sph.gauss_laguerre_scaled(n)
        assert np.all(np.diff(x) > 0) and np.all(wx > 0)
        for m in (0, 1, 2, 7, min(2 * n - 1, 30)):
            # Int_0^inf x^m e^-x dx = m!; the rule with weights (w e^x) e^-x must be exact for m <= 2n - 1
            assert np.sum(wx * np.exp(-x) * x**m) == pytest.approx(math.factorial(m), rel=2e-12)
    x, wx = sph.gauss_laguerre_scaled(12)
    x2, w2 = np.polynomial.laguerre.laggauss(12)                        # independent library rule
    np.testing.assert_allclose(x, x2, rtol=1e-12)
    np.testing.assert_allclose(wx * np.exp(-x), w2, rtol=1e-11)


def test_nodes_integrate_a_spheroid_volume():
    """sum W over the nodes with the weight e^{-lam (R/2)(eta - 1)}: Int (R/2)^3 (eta^2 - tau^2) e^{-s(eta-1)} d eta d tau
    = (R/2)^3 [2 (1/s + 2/s^2 + 2/s^3) - (2/3)/s],  s = lam R/2."""
    for R, lam in ((1.7, 1.0), (0.4, 2.5)):
        eta, weta, tau, wtau = sph.spheroidal_nodes(dict(n_rho=20, n_z=16, eta_scale=lam), R)
        s = 0.5 * lam * R
        E, T = np.meshgrid(eta, tau, indexing="ij")
        got = np.sum(weta[:, None] * wtau[None, :] * (0.5 * R) ** 3 * (E * E - T * T) * np.exp(-s * (E - 1.0)))
        ref = (0.5 * R) ** 3 * (2.0 * (1 / s + 2 / s**2 + 2 / s**3) - (2.0 / 3.0) / s)
        assert got == pytest.approx(ref, rel=1e-12)


def test_matrix_product_form_equals_the_loop_definition():
    q = dict(kind=1, n_rho=10, n_phi=1, n_z=16, rho_max=30.0, z_pad=30.0, phi_rule=1, eta_scale=1.3)
    prob = tiny_problem(True, l_max=1, n_max=2, bins=1, k_max=1.5, Nr=300, h=0.1, Z_P=2.0, quad=q, seed=5)
    b, z, v = 0.8, -0.5, 1.1
    Sb, Hpt, Htp = sph.body_frame_blocks_spheroidal(prob, b, z, v)
    Ts, Ps = prob.centres[0].states(), prob.centres[1].states()
    for i, j in [(0, 0), (1, 3), (len(Ps) - 1, len(Ts) - 2), (3, 1)]:
        assert abs(sph.body_frame_element_loops(prob, Ps[i], Ts[j], b, z, v, "S") - Sb[i, j]) < 1e-14
        assert abs(sph.body_frame_element_loops(prob, Ps[i], Ts[j], b, z, v, "HPT") - Hpt[i, j]) < 1e-14
        assert abs(sph.body_frame_element_loops(prob, Ps[i], Ts[j], b, z, v, "HTP") - Htp[j, i]) < 1e-14


@pytest.mark.parametrize("R", [0.8, 2.0, 5.0])
def test_static_overlaps_closed_forms(R):
    """v = 0: textbook two-centre hydrogen integrals; the spheroidal rule has no cusp problem."""
    prob = _bound_problem(SPH)
    S, HPT, HTP = sph.two_centre_blocks_spheroidal(prob, 1e-9, R, 0.0)
    e = math.exp
    assert S[0, 0].real == pytest.approx((1 + R + R * R / 3) * e(-R), abs=5e-10)
    ref_1s2s = (16 * math.sqrt(2) / (27 * R)) * (e(-R / 2) * (-3 * R * R + 22 * R - 64) + e(-R) * (10 * R + 64))
    ref_1s2p0 = (16 * math.sqrt(2) / (27 * R * R)) * (e(-R / 2) * (3 * R**3 - 16 * R * R + 32 * R + 64) - e(-R) * (8 * R * R + 64 * R + 64))
    assert S[0, 1].real == pytest.approx(ref_1s2s, abs=5e-10)
    assert S[0, 3].real == pytest.approx(ref_1s2p0, abs=5e-10)
    assert HPT[0, 0].real == pytest.approx(-(1 + R) * e(-R), abs=5e-10)
    assert HTP[0, 0].real == pytest.approx(-(1 + R) * e(-R), abs=5e-10)


def test_printed_values_of_survey_B2():
    """Int conj psi_beta(r_P) e^{+i v z_m} psi_alpha(r_T) d^3r at b = 0.9, z = -1.3, v = 1
    (e^{+i v z_m} = the S_PT integrand at velocity -v)."""
    prob = _bound_problem(SPH)
    S, _, _ = sph.two_centre_blocks_spheroidal(prob, 0.9, -1.3, -1.0)
    stT, stP = prob.centres[0].states(), prob.centres[1].states()
    nl = {(n, l): i for i, (n, l) in enumerate(RAD)}
    printed = {((1, 0, 0), (1, 0, 0)): 0.403240479255, ((1, 0, 0), (2, 1, 0)): -0.082163614445 + 0.243694370036j,
               ((2, 1, 1), (1, 0, 0)): 0.062932251848 + 0.022323617770j}
    for (beta, alpha), val in printed.items():
        i = stP.index((nl[beta[:2]], beta[1], beta[2])); j = stT.index((nl[alpha[:2]], alpha[1], alpha[2]))
        assert abs(S[i, j] - val) < 2e-9, (beta, alpha, S[i, j], val)


def test_agrees_with_the_converged_cylindrical_rule():
    """The same integrals by the cylindrical Gauss-Legendre rule of oracle/transfer.py at high resolution."""
    b, z, v = 1.3, 0.7, 0.9
    Ss, Hs, Ts = sph.two_centre_blocks_spheroidal(_bound_problem(SPH), b, z, v)
    Sc, Hc, Tc = tr.two_centre_blocks(_bound_problem(CYL), b, z, v)
    assert np.abs(Ss - Sc).max() < 2e-8
    assert np.abs(Hs - Hc).max() < 1e-6 and np.abs(Ts - Tc).max() < 1e-6        # cylinders: cusp-limited (1/r on the axis)


def test_galerkin_identity_and_hermiticity():
    prob = _bound_problem(SPH)
    b, z, v, dz = 1.0, 0.4, 1.0, 1e-3
    S0, H0 = sph.S_and_H_spheroidal(prob, b, z, v)
    Sp, _ = sph.S_and_H_spheroidal(prob, b, z + dz, v)
    Sm, _ = sph.S_and_H_spheroidal(prob, b, z - dz, v)
    n = prob.centres[0].n_states
    lhs = H0[n:, :n] - H0[:n, n:].conj().T
    rhs = -1j * v * (Sp[n:, :n] - Sm[n:, :n]) / (2 * dz)
    assert np.abs(lhs - rhs).max() < 5e-7
    assert np.abs(S0 - S0.conj().T).max() < 1e-15
    assert abs(S0[5, 0] - 0.5182285778229) < 1e-9                        # SURVEY.md App. B.4 printed element
    assert abs(H0[5, 0] - (-0.5380476899624 + 0.03993524629055j)) < 1e-9  # (cusp-limited to 5e-7 with cylinders)
