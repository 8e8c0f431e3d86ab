"""Pins for oracle/nonuniform.py (radial grid "denser around the origin")."""
import math

import numpy as np
import pytest

from oracle import direct
from oracle import nonuniform as nu
from oracle import transfer as tr
from wpccc_inputs import hydrogenic_bound_u, make_problem
from wpccc_inputs.configs import bound_only_centre
from wpccc_inputs.paper_shape import exponential_grid, resample_problem, trapezoid_weights


def test_interp5_grid_exact_for_quartics_and_equals_the_uniform_rule():
    g = exponential_grid(60, 5.0, 3.0)
    poly = lambda x: 0.3 * x**4 - 1.1 * x**3 + 0.2 * x**2 + 2 * x
    r = np.array([0.001, 0.02, 0.149, 1.7, 2.5, 4.87, 4.999, 5.0])
    np.testing.assert_allclose(nu.interp5_grid(poly(g), g, r), poly(r), rtol=2e-12)
    assert nu.interp5_grid(poly(g), g, np.array([5.0001, 77.0])).tolist() == [0.0, 0.0]
    np.testing.assert_allclose(nu.interp5_grid(np.sin(g), g, g[3:10]), np.sin(g[3:10]), rtol=0, atol=1e-15)   # table values on grid points
    h, Nr = 0.1, 50
    gu = h * np.arange(Nr + 1)
    rr = np.array([0.003, 0.149, 0.151, 0.25, 2.5, 4.87, 4.999])           # 0.25: a tie, the uniform rule rounds up, this one down:
    a, b_ = tr.interp5(np.cos(gu), h, rr), nu.interp5_grid(np.cos(gu), gu, rr)   # both stencils interpolate the same smooth function
    np.testing.assert_allclose(np.delete(a, 3), np.delete(b_, 3), rtol=0, atol=1e-15)
    assert abs(a[3] - b_[3]) < 1e-7


def test_radial_integral_on_the_exponential_grid_converges_to_the_closed_form():
    """F[1s,1s,0](R) = (e^{2R} - R - 1) e^{-2R} / R by the trapezoid sum of eq. (7) on the non-uniform grid."""
    R = 1.5
    exact = (math.exp(2 * R) - R - 1) * math.exp(-2 * R) / R
    errs = []
    for Nr in (400, 800, 1600):
        g = exponential_grid(Nr, 60.0, 4.0)
        u = hydrogenic_bound_u(1, 0, 1.0, g)
        errs.append(abs(direct.radial_F(u, u, trapezoid_weights(g), g, R, 0) - exact))
    assert errs[0] < 5e-4 and errs[2] < errs[1] < errs[0] and 2.5 < errs[0] / errs[1] < 6.0    # second order (kink at r = R)


def test_static_overlap_closed_forms_on_the_exponential_grid():
    rad = [(1, 0), (2, 0), (2, 1)]
    fine = make_problem([bound_only_centre(1.0, rad, 4000, 0.0125), bound_only_centre(1.0, rad, 4000, 0.0125)], 1.0, 4000, 0.0125, 2,
                        quad=dict(n_rho=160, n_phi=16, n_z=320, rho_max=40.0, z_pad=40.0, phi_rule=1))
    g = exponential_grid(1500, 50.0, 4.0)
    prob = resample_problem(fine, g)
    for R in (0.8, 2.0):
        S, HPT, HTP = nu.two_centre_blocks_grid(prob, g, 1e-9, R, 0.0)
        e = math.exp
        nrm = 1.0                                                   # resampled functions are grid-normalised: 1s norm = 1 to 1e-6
        assert S[0, 0].real == pytest.approx((1 + R + R * R / 3) * e(-R) * nrm, abs=2e-6)
        assert HPT[0, 0].real == pytest.approx(-(1 + R) * e(-R), abs=3e-6)
        assert HTP[0, 0].real == pytest.approx(-(1 + R) * e(-R), abs=3e-6)
