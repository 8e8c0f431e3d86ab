"""Pins for oracle/propagate.py, assemble.py, observables.py: library solve, RK4 order on a solvable ODE,
unitarity, the one-centre end-to-end values of SURVEY.md App. B.3, conservation of c^H S c (two centres)."""
import math

import numpy as np
import pytest

from oracle.assemble import S_and_H
from oracle.observables import cross_sections, probabilities
from oracle.propagate import gauss_solve, propagate
from wpccc_inputs import make_problem, tiny_problem
from wpccc_inputs.configs import bound_only_centre


def test_gauss_solve_vs_lapack():
    rng = np.random.default_rng(3)
    for n in (1, 2, 7, 40):
        A = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
        y = rng.normal(size=n) + 1j * rng.normal(size=n)
        np.testing.assert_allclose(gauss_solve(A, y), np.linalg.solve(A, y), rtol=1e-10, atol=1e-12)
    A = np.array([[0, 1], [1, 0]], complex)                      # needs the row exchange
    np.testing.assert_allclose(gauss_solve(A, np.array([2, 3], complex)), [3, 2])
    with pytest.raises(ZeroDivisionError):
        gauss_solve(np.zeros((2, 2)), np.ones(2))


class _Dummy:
    def __init__(self, n, two):
        self.centres = [None, None] if two else [None]
        self.n_tot = n


def test_rk4_constant_generator_matches_matrix_exponential_and_order():
    """dc/dz = -(i/v) S^-1 H c with constant S, H: exact solution by eigen-decomposition; RK4 global error ~ h^4."""
    rng = np.random.default_rng(0)
    n, v = 5, 1.3
    K = 0.2 * (rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n)))
    S = np.eye(n) + 0.5 * (K + K.conj().T)
    H = 0.5 * (rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n)))
    M = (-1j / v) * np.linalg.solve(S, H)
    w, V = np.linalg.eig(M)
    c0 = np.zeros(n, complex); c0[0] = 1
    exact = V @ (np.exp(w * 2.0) * np.linalg.solve(V, c0))
    errs = []
    for ns in (20, 40, 80):
        c = propagate(_Dummy(n, True), 0.0, v, 0.0, 2.0, ns, matrices=lambda i: (S, H))
        errs.append(np.abs(c - exact).max())
    assert errs[2] < 1e-5 * np.abs(exact).max()
    assert 12 < errs[0] / errs[1] < 20 and 12 < errs[1] / errs[2] < 20
    # one-centre path ignores S (eq. (5))
    c1 = propagate(_Dummy(n, False), 0.0, v, 0.0, 2.0, 80, matrices=lambda i: (None, H))
    w1, V1 = np.linalg.eig((-1j / v) * H)
    assert np.abs(c1 - V1 @ (np.exp(w1 * 2.0) * np.linalg.solve(V1, c0))).max() < 1e-5


def test_evaluation_count_is_2n_plus_1():
    """4 n_z + 1 evaluations per path = 2 n_steps + 1: M_new is reused as the next M_z."""
    calls = []
    H = np.eye(2, dtype=complex)
    propagate(_Dummy(2, False), 0.0, 1.0, 0.0, 1.0, 7, matrices=lambda i: (calls.append(i), (None, H))[1])
    assert calls == list(range(15))


RAD14 = [(1, 0), (2, 0), (3, 0), (2, 1), (3, 1), (3, 2)]


def _b3_problem():
    C = bound_only_centre(1.0, RAD14, 2000, 0.05)
    return make_problem([C], 1.0, 2000, 0.05, 4)


def test_one_centre_end_to_end_survey_B3():
    """hydrogen n<=3 (14 states), b=1, v=2, z in [-50,50], 1000 RK4 steps.
    Grid sums, elements at z=0.3 and final probabilities printed there (independent prototype)."""
    from oracle.direct import direct_block, radial_F
    prob = _b3_problem()
    C = prob.centres[0]
    r = prob.h * np.arange(prob.Nr + 1)
    assert radial_F(C.u[0], C.u[0], prob.w, r, 1.5, 0) == pytest.approx(5.837294241354868e-01, rel=1e-13)
    assert radial_F(C.u[0], C.u[3], prob.w, r, 0.07, 1) == pytest.approx(1.265297973743750e-02, rel=1e-12)
    assert radial_F(C.u[3], C.u[3], prob.w, r, 7.3, 2) == pytest.approx(5.825665312897638e-02, rel=1e-12)
    D = direct_block(C, prob.w, r, 4, 1.0, 0.3, 2.0, 1.0, False)
    assert abs(D[3, 0] - (-4.974809418271389e-02 - 2.801285401873574e-03j)) < 1e-15
    assert abs(D[4, 0] - (-2.110632884862242e-02 - 1.188484742222212e-03j)) < 1e-15
    assert abs(D[5, 0] + D[3, 0]) < 1e-16
    assert abs(D[13, 2] - 1.612059467213394e-04) < 1e-16
    c = propagate(prob, 1.0, 2.0, -50.0, 50.0, 1000)
    _, P_nl, P_class = probabilities(prob, c)
    ref = [8.992143926451e-01, 3.908868632836e-02, 1.076501700116e-02, 3.856576451394e-02, 1.064398208030e-02,
           1.722156081428e-03]
    np.testing.assert_allclose(P_nl[0], ref, rtol=0, atol=2e-12)
    P = np.abs(c) ** 2
    assert P[3] == pytest.approx(6.535283109244e-03, abs=1e-13) and P[4] == pytest.approx(2.549519829545e-02, abs=1e-13)
    assert abs(P[3] - P[5]) < 1e-15                                  # m-symmetry (reflection in the collision plane)
    assert P.sum() - 1 == pytest.approx(-1.35e-09, abs=2e-11)
    assert P_class[0, 0] == pytest.approx(ref[0], abs=1e-12) and P_class[0, 1] == pytest.approx(sum(ref[1:]), abs=1e-11)


def test_unitarity_one_centre_norm_drift_fifth_order():
    """H Hermitian (one centre) => norm conserved up to RK4 truncation: drift falls ~32x on halving the step."""
    C = bound_only_centre(1.0, [(1, 0), (2, 0), (2, 1)], 600, 0.1)
    prob = make_problem([C], 1.0, 600, 0.1, 2)
    d = []
    for ns in (200, 400):
        c = propagate(prob, 1.0, 1.0, -10.0, 10.0, ns)
        d.append(abs(np.sum(np.abs(c) ** 2) - 1))
    print(d)
    assert d[1] < 1e-8 and 20 < d[0] / d[1] < 45


def test_two_centre_conserves_cSc_and_matches_survey_B4_trend():
    """Galerkin H (amb. A1): c^H S c is conserved up to RK4 truncation and quadrature error; sum |c|^2 is not."""
    rad = [(1, 0), (2, 0), (2, 1)]
    T = bound_only_centre(1.0, rad, 1000, 0.05); P = bound_only_centre(1.0, rad, 1000, 0.05)
    quad = dict(n_rho=64, n_phi=16, n_z=128, rho_max=40.0, z_pad=40.0, phi_rule=1)
    prob = make_problem([T, P], 1.0, 1000, 0.05, 2, quad=quad)
    c, drift = propagate(prob, 1.0, 1.0, -6.0, 6.0, 60, track_norm=True)
    assert drift < 2e-4
    # start is not asymptotic at z=-6, so only structure is checked: capture happened, m-symmetry holds
    P_ = np.abs(c) ** 2
    assert 0.2 < P_[5] < 0.9 and abs(P_[2] - P_[4]) < 1e-12 and abs(P_[7] - P_[9]) < 1e-12
    # the literal Hermitian reading H_PT := H_TP^dagger (eq. (1) as printed) does NOT conserve c^H S c (amb. A1)
    cache = {}
    def herm(i):
        if i not in cache:
            S, H = S_and_H(prob, 1.0, -6.0 + 0.1 * i, 1.0)
            H = H.copy(); H[5:, :5] = H[:5, 5:].conj().T
            cache[i] = (S, H)
        return cache[i]
    _, drift_h = propagate(prob, 1.0, 1.0, -6.0, 6.0, 60, matrices=herm, track_norm=True)
    assert drift_h > 50 * drift


def test_probabilities_and_cross_sections():
    prob = tiny_problem(True, seed=1)
    n = prob.n_tot
    rng = np.random.default_rng(5)
    C = rng.normal(size=(3, n)) + 1j * rng.normal(size=(3, n))
    Ps, Pnl, Pc = probabilities(prob, C, init_state=0)
    np.testing.assert_allclose(Ps, np.abs(C) ** 2, rtol=1e-15)
    np.testing.assert_allclose(Pnl.sum(1), Ps.sum(1), rtol=1e-14)
    np.testing.assert_allclose(Pc.sum(1), Ps.sum(1), rtol=1e-14)
    assert Pc[0, 0] == pytest.approx(Ps[0, 0])
    # sigma = 2 pi Int b P db with P = 1/b^2 on [b0,b1] -> 2 pi ln(b1/b0), exact for the ln-b trapezoid rule
    b = np.array([0.1, 0.3, 1.0, 4.0]); vg = np.zeros(4, int)
    sig = cross_sections(b, vg, (1 / b**2)[:, None], 1)
    assert sig[0, 0] == pytest.approx(2 * math.pi * math.log(40.0), rel=1e-14)
    # P = const: trapezoid in ln b of b^2 -> converges to pi (b1^2 - b0^2) under refinement
    bb = np.exp(np.linspace(math.log(0.1), math.log(4.0), 400))
    sig = cross_sections(bb, np.zeros(400, int), np.ones((400, 1)), 1)
    assert sig[0, 0] == pytest.approx(math.pi * (16 - 0.01), rel=1e-4)
