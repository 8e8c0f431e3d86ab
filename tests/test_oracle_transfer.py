"""Pins for oracle/transfer.py: closed forms (static overlaps), independent spheroidal/Bessel brute force with
the translation factor, L0 (lab-frame definition) == L1 (factorised), Galerkin identity, interpolation."""
import math

import numpy as np
import pytest

from oracle import angular as ang
from oracle import transfer as tr
from oracle.assemble import S_and_H
from wpccc_inputs import make_problem, tiny_problem
from wpccc_inputs.configs import bound_only_centre

RAD = [(1, 0), (2, 0), (2, 1)]
HI = dict(n_rho=160, n_phi=16, n_z=320, rho_max=40.0, z_pad=40.0, phi_rule=1)


def _bound_problem(quad, Nr=4000, h=0.0125, ZP=1.0):
    T = bound_only_centre(1.0, RAD, Nr, h)
    P = bound_only_centre(ZP, RAD, Nr, h)
    return make_problem([T, P], ZP, Nr, h, 2, quad=quad)


def test_interp5_exact_for_quartics_and_zero_beyond_rmax():
    h, Nr = 0.1, 50
    k = np.arange(Nr + 1) * h
    poly = lambda x: 0.3 * x**4 - 1.1 * x**3 + 0.2 * x**2 + 2 * x
    r = np.array([0.003, 0.149, 0.151, 2.5, 4.87, 4.999, 5.0])
    np.testing.assert_allclose(tr.interp5(poly(k), h, r), poly(r), rtol=1e-12)
    assert tr.interp5(poly(k), h, np.array([5.0001, 77.0])).tolist() == [0.0, 0.0]
    # on a grid point the table value comes back exactly (Lagrange basis)
    np.testing.assert_allclose(tr.interp5(np.sin(k), h, k[3:10]), np.sin(k[3:10]), rtol=0, atol=1e-15)


def test_quadrature_nodes_integrate_volume_and_layout():
    q = dict(n_rho=8, n_phi=6, n_z=16, rho_max=3.0, z_pad=2.0)
    rho, wrho, phi, wphi, zp, wz = tr.quadrature_nodes(q, 1.5)
    assert (len(rho), len(phi), len(zp)) == (8, 6, 16)
    assert np.sum(wrho) * np.sum(wphi) * np.sum(wz) == pytest.approx(math.pi * 9.0 * 5.5, rel=1e-13)   # cylinder volume
    assert zp[:4].max() < 0 < zp[4:12].min() and zp[4:12].max() < 1.5 < zp[12:].min()                  # panels 4/8/4


def test_azimuthal_phi_discrete_vs_bessel():
    from scipy.special import jv
    x = np.array([0.0, 0.05, 0.2, 0.4])
    phi, w = tr.gauss_legendre(40, 0.0, 2 * math.pi)
    for d in range(-3, 4):
        for sign in (+1, -1):
            disc = tr.azimuthal_phi(d, x, phi, w, sign, 0)
            np.testing.assert_allclose(disc, (-1j * sign) ** d * jv(d, x), rtol=0, atol=1e-12)   # converged GL rule
            assert np.allclose(tr.azimuthal_phi(d, x, phi, w, sign, 1), (-1j * sign) ** d * jv(d, x), atol=0)


@pytest.mark.parametrize("R", [0.8, 2.0, 5.0])
def test_static_overlaps_closed_forms(R):
    """v = 0, b -> body frame = lab frame (b tiny): textbook two-centre hydrogen integrals."""
    prob = _bound_problem(HI)
    S, HPT, HTP = tr.two_centre_blocks(prob, 1e-9, R, 0.0)
    e = math.exp
    assert S[0, 0].real == pytest.approx((1 + R + R * R / 3) * e(-R), abs=2e-8)
    ref_1s2s = (16 * math.sqrt(2) / (27 * R)) * (e(-R / 2) * (-3 * R * R + 22 * R - 64) + e(-R) * (10 * R + 64))
    ref_1s2p0 = (16 * math.sqrt(2) / (27 * R * R)) * (e(-R / 2) * (3 * R**3 - 16 * R * R + 32 * R + 64) - e(-R) * (8 * R * R + 64 * R + 64))
    assert S[0, 1].real == pytest.approx(ref_1s2s, abs=2e-8)          # <1s_P | 2s_T>
    assert S[0, 3].real == pytest.approx(ref_1s2p0, abs=2e-8)         # <1s_P | 2p0_T>, z' from T to P
    assert HPT[0, 0].real == pytest.approx(-(1 + R) * e(-R), abs=5e-7)  # <1s_P|-1/r_P|1s_T>
    assert HTP[0, 0].real == pytest.approx(-(1 + R) * e(-R), abs=5e-7)  # <1s_T|-1/r_T|1s_P>
    assert np.abs(S.imag).max() < 1e-15


def _spheroidal_bessel(beta, alpha, b, z, v, sign, NQ=64):
    """Independent evaluation of Int conj psi_beta(r_P) e^{i sign v z_m} psi_alpha(r_T) d^3r in the paper's own
    prolate-spheroidal form, eq. (9): Gauss-Laguerre(eta) x Gauss-Legendre(tau), analytic
    azimuth (Bessel), analytic hydrogen R_nl, rotated to the lab frame by eq. (8)."""
    from scipy.special import jv, lpmv, roots_laguerre, roots_legendre
    from wpccc_inputs import hydrogenic_bound_u
    R = math.hypot(b, z)
    Theta = math.acos(z / R)
    xe, we = roots_laguerre(NQ)
    xt, wt = roots_legendre(NQ)
    s = 0.5 * R
    eta = 1 + xe / s
    weta = we * np.exp(xe) / s
    E, T = np.meshgrid(eta, xt, indexing="ij")
    W = weta[:, None] * wt[None, :] * (R / 2) ** 3 * (E**2 - T**2)
    rT, rP = R * (E + T) / 2, R * (E - T) / 2
    cTb, cPb = (E * T + 1) / (E + T), (E * T - 1) / (E - T)
    x = (v * b / 2) * np.sqrt((E**2 - 1) * (1 - T**2))
    pz = np.exp(1j * sign * (v * z / 2) * E * T)

    def Th(l, q, c):
        aq = abs(q)
        t = math.sqrt((2 * l + 1) / 2 * math.factorial(l - aq) / math.factorial(l + aq)) * lpmv(aq, l, c)
        return t if q >= 0 else (-1) ** aq * t

    (nb, lb, mb), (na, la, ma) = beta, alpha
    fb = hydrogenic_bound_u(nb, lb, 1.0, rP.ravel()).reshape(rP.shape) / rP
    fa = hydrogenic_bound_u(na, la, 1.0, rT.ravel()).reshape(rT.shape) / rT
    tot = 0.0
    for qp in range(-lb, lb + 1):
        for q in range(-la, la + 1):
            d = q - qp
            body = np.sum(W * fb * Th(lb, qp, cPb) * fa * Th(la, q, cTb) * pz * (-1j * sign) ** d * jv(d, x))
            tot += ang.wigner_small_d(lb, mb, qp, Theta) * ang.wigner_small_d(la, ma, q, Theta) * body
    return tot


def test_translation_factor_elements_vs_paper_spheroidal_form():
    """Cylindrical Gauss-Legendre oracle (high resolution, Bessel azimuth) against eq. (9)'s spheroidal rule.
    Also reproduces SURVEY.md App. B.2's printed values for e^{+i v z_m} at b=0.9, z=-1.3, v=1."""
    b, z, v = 0.9, -1.3, 1.0
    prob = _bound_problem(HI)
    S, _, _ = tr.two_centre_blocks(prob, b, z, v)                 # e^{-i v z_m}
    stT = prob.centres[0].states(); stP = prob.centres[1].states()
    nl = {(n, l): i for i, (n, l) in enumerate(RAD)}
    for beta, alpha in [((1, 0, 0), (1, 0, 0)), ((1, 0, 0), (2, 1, 0)), ((2, 1, 1), (1, 0, 0)), ((2, 1, -1), (2, 1, 1))]:
        i = stP.index((nl[beta[:2]], beta[1], beta[2])); j = stT.index((nl[alpha[:2]], alpha[1], alpha[2]))
        ref = _spheroidal_bessel(beta, alpha, b, z, v, -1)
        assert abs(S[i, j] - ref) < 5e-9, (beta, alpha, S[i, j], ref)
    printed = {((1, 0, 0), (1, 0, 0)): 0.403240479255, ((1, 0, 0), (2, 1, 0)): -0.082163614445 + 0.243694370036j,
               ((2, 1, 1), (1, 0, 0)): 0.062932251848 + 0.022323617770j}
    for (beta, alpha), val in printed.items():
        assert abs(_spheroidal_bessel(beta, alpha, b, z, v, +1) - val) < 1e-10


def test_L0_lab_frame_definition_equals_L1_factorised():
    prob = tiny_problem(True, seed=5)
    b, z, v = 0.7, -0.4, 1.2
    S, HPT, HTP = tr.two_centre_blocks(prob, b, z, v)
    Ts = prob.centres[0].states(); Ps = prob.centres[1].states()
    for i, j in [(0, 0), (3, 1), (5, 7), (len(Ps) - 1, len(Ts) - 2)]:
        assert abs(tr.lab_frame_element(prob, Ps[i], Ts[j], b, z, v, "S") - S[i, j]) < 2e-15
        assert abs(tr.lab_frame_element(prob, Ps[i], Ts[j], b, z, v, "HPT") - HPT[i, j]) < 2e-15
        assert abs(tr.lab_frame_element(prob, Ps[i], Ts[j], b, z, v, "HTP") - HTP[j, i]) < 2e-15


def test_matmul_form_equals_loops():
    prob = tiny_problem(True, seed=7, Z_P=2.0)
    a = tr.body_frame_blocks(prob, 1.1, 0.3, 0.8)
    b = tr.body_frame_blocks_loops(prob, 1.1, 0.3, 0.8)
    for x, y in zip(a, b):
        np.testing.assert_allclose(x, y, rtol=0, atol=3e-15)


def test_galerkin_identity_and_hermiticity():
    """H_PT - H_TP^dagger = -i v dS_PT/dz (follows from i d/dt <chi_P|chi_T>), S Hermitian,
    H not Hermitian (amb. A1).  Bound states, converged quadrature; derivative by central differences."""
    prob = _bound_problem(HI, Nr=4000, h=0.0125)
    b, z, v, dz = 1.0, 0.4, 1.0, 1e-3
    S0, H0 = S_and_H(prob, b, z, v)
    Sp, _ = S_and_H(prob, b, z + dz, v)
    Sm, _ = S_and_H(prob, b, z - dz, v)
    n = prob.centres[0].n_states
    lhs = H0[n:, :n] - H0[:n, n:].conj().T
    rhs = -1j * v * (Sp[n:, :n] - Sm[n:, :n]) / (2 * dz)
    assert np.abs(lhs - rhs).max() < 5e-7
    assert np.abs(S0 - S0.conj().T).max() < 1e-15
    assert np.abs(H0 - H0.conj().T).max() > 1e-3
    assert np.abs(H0[:n, :n] - H0[:n, :n].conj().T).max() < 1e-15     # direct blocks Hermitian
    assert np.linalg.eigvalsh(S0).min() > 0.1                          # S positive definite


def test_survey_B4_elements():
    """SURVEY.md App. B.4 printed elements at z=0.4 (b=1, v=1, with time phases), independent prototype."""
    prob = _bound_problem(HI)
    S, H = S_and_H(prob, 1.0, 0.4, 1.0)
    assert abs(S[5, 0] - 0.5182285778229) < 1e-9
    assert abs(S[5, 3] - (-2.921033024100e-03 - 0.2347018820158j)) < 1e-9
    assert abs(S[9, 4] - 0.1131813722346) < 1e-9
    assert abs(H[9, 4] - (-0.05371803399139 + 3.157631557054e-03j)) < 1e-9
    assert abs(H[8, 0] - (9.043423394091e-03 + 0.1192085142157j)) < 1e-9
    assert abs(H[5, 0] - (-0.5380476899624 + 0.03993524629055j)) < 5e-7     # cusp-limited (1/r_P on the axis)
