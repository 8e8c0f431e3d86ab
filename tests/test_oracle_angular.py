"""Pins for oracle/angular.py against library routines (sympy, scipy) and closed forms."""
import math

import numpy as np
import pytest
from scipy.special import lpmv, sph_harm_y

from oracle import angular as ang


def test_clebsch_gordan_vs_sympy():
    from sympy.physics.wigner import clebsch_gordan as cg_sym
    for j1 in range(0, 4):
        for j2 in range(0, 4):
            for j in range(abs(j1 - j2), j1 + j2 + 1):
                for m1 in range(-j1, j1 + 1):
                    for m2 in range(-j2, j2 + 1):
                        m = m1 + m2
                        if abs(m) > j:
                            continue
                        ref = float(cg_sym(j1, j2, j, m1, m2, m))
                        assert ang.clebsch_gordan(j1, m1, j2, m2, j, m) == pytest.approx(ref, abs=1e-14)


def test_clebsch_gordan_selection_rules():
    assert ang.clebsch_gordan(1, 0, 1, 0, 1, 0) == 0.0          # <10;10|10> vanishes
    assert ang.clebsch_gordan(2, 1, 1, 1, 2, 1) == 0.0          # m1 + m2 != m
    assert ang.clebsch_gordan(1, 1, 1, -1, 0, 0) == pytest.approx(1 / math.sqrt(3), abs=1e-15)


def test_assoc_legendre_vs_scipy():
    x = np.linspace(-0.999, 0.999, 41)
    for l in range(0, 9):
        for m in range(-l, l + 1):
            ref = lpmv(m, l, x)
            got = ang.assoc_legendre(l, m, x)
            np.testing.assert_allclose(got, ref, rtol=1e-12, atol=1e-13 * max(1.0, np.abs(ref).max()))


def test_sph_harm_vs_scipy_and_theta_tilde_norm():
    th = np.linspace(0.1, 3.0, 7)
    ph = np.linspace(0.0, 6.0, 7)
    for l in range(0, 5):
        for m in range(-l, l + 1):
            ref = sph_harm_y(l, m, th, ph)
            got = ang.sph_harm(l, m, np.cos(th), ph)
            np.testing.assert_allclose(got, ref, rtol=0, atol=1e-13)
    # Theta~ normalised: Int_{-1}^{1} Theta~_lq^2 dc = 1
    c, w = np.polynomial.legendre.leggauss(40)
    for l in range(0, 5):
        for q in range(-l, l + 1):
            assert np.sum(w * ang.theta_tilde(l, q, c) ** 2) == pytest.approx(1.0, abs=1e-13)


def test_wigner_small_d_closed_forms_and_group_law():
    for beta in (0.0, 0.3, 1.1, 2.9, math.pi):
        c, s = math.cos(beta), math.sin(beta)
        # textbook d^1 (Varshalovich / Sakurai), rows/cols m = 1, 0, -1
        d1 = {(1, 1): (1 + c) / 2, (1, 0): -s / math.sqrt(2), (1, -1): (1 - c) / 2,
              (0, 1): s / math.sqrt(2), (0, 0): c, (0, -1): -s / math.sqrt(2),
              (-1, 1): (1 - c) / 2, (-1, 0): s / math.sqrt(2), (-1, -1): (1 + c) / 2}
        for (mp, m), ref in d1.items():
            assert ang.wigner_small_d(1, mp, m, beta) == pytest.approx(ref, abs=1e-15)
        assert ang.wigner_small_d(2, 0, 0, beta) == pytest.approx((3 * c * c - 1) / 2, abs=1e-15)
    for j in (1, 2, 3):
        a, b = 0.4, 0.9
        da = np.array([[ang.wigner_small_d(j, mp, m, a) for m in range(-j, j + 1)] for mp in range(-j, j + 1)])
        db = np.array([[ang.wigner_small_d(j, mp, m, b) for m in range(-j, j + 1)] for mp in range(-j, j + 1)])
        dab = np.array([[ang.wigner_small_d(j, mp, m, a + b) for m in range(-j, j + 1)] for mp in range(-j, j + 1)])
        np.testing.assert_allclose(da @ db, dab, atol=1e-14)            # rotations about y compose
        np.testing.assert_allclose(da @ da.T, np.eye(2 * j + 1), atol=1e-14)  # orthogonal


def test_wigner_d_rotates_spherical_harmonics():
    """Y_lm(lab direction) = sum_q d^l_{m q}(Theta) Y_lq(body direction) for the frame of SURVEY App. A.1:
    body z' = (sin Th, 0, cos Th), x' = (cos Th, 0, -sin Th).  Pins the rotation convention of eq. (8)."""
    Th = 0.77
    rng = np.random.default_rng(1)
    for _ in range(4):
        vb = rng.normal(size=3); vb /= np.linalg.norm(vb)             # direction in body coordinates
        zp = np.array([math.sin(Th), 0, math.cos(Th)]); xp = np.array([math.cos(Th), 0, -math.sin(Th)])
        yp = np.array([0.0, 1.0, 0.0])
        vl = vb[0] * xp + vb[1] * yp + vb[2] * zp                      # same direction in lab coordinates
        for l in (1, 2, 3):
            for m in range(-l, l + 1):
                lab = ang.sph_harm(l, m, vl[2], math.atan2(vl[1], vl[0]))
                body = sum(ang.wigner_small_d(l, m, q, Th) * ang.sph_harm(l, q, vb[2], math.atan2(vb[1], vb[0]))
                           for q in range(-l, l + 1))
                assert abs(lab - body) < 1e-14


def test_direct_angular_coefficient_is_gaunt():
    """G^lam P_lam^mu(cos Th) (with phi_R = 0) must equal the multipole angular integral
       4 pi/(2 lam+1) conj(Y_{lam mu}(R^)) <l'm'|Y_{lam mu}|l m>  (Laplace expansion of 1/|r - R|)."""
    from sympy.physics.wigner import gaunt
    cT = 0.37
    for lp in range(0, 3):
        for l in range(0, 3):
            for lam in range(0, 5):
                for mp in range(-lp, lp + 1):
                    for m in range(-l, l + 1):
                        mu = mp - m
                        G = ang.direct_angular_coefficient(lp, mp, l, m, lam)
                        if abs(mu) > lam:
                            assert G == 0.0
                            continue
                        # <l'm'|Y_{lam mu}|lm> = (-1)^{m'} gaunt(l', lam, l, -m', mu, m)
                        integral = (-1) ** mp * float(gaunt(lp, lam, l, -mp, mu, m))
                        ref = 4 * math.pi / (2 * lam + 1) * np.conj(ang.sph_harm(lam, mu, cT, 0.0)) * integral
                        got = G * float(ang.assoc_legendre(lam, mu, cT))
                        assert abs(got - ref) < 1e-13, (lp, mp, l, m, lam)
