"""Pins the judge's round-1 review found printed in SURVEY.md but not asserted: App. B.2b (same-node values of the
configured cylindrical 64 x 16 x 128 rule: pins the node layout of reading A10), App. B.4 (two-centre end-to-end: final
probabilities and the conserved c^H S c with converged integrals), and BASELINE.json north_star's "total probability = 1
to 1e-8" for TWO centres (converged quadrature + one step refinement, as DESIGN.md A24 says)."""
import numpy as np
import pytest

from oracle import propagate as oprop
from oracle import spheroidal as sph
from oracle import transfer as tr
from wpccc_inputs import make_problem
from wpccc_inputs.configs import bound_only_centre


def _problem(rad, quad, Nr=8000, h=0.0125):
    T = bound_only_centre(1.0, rad, Nr, h)
    P = bound_only_centre(1.0, rad, Nr, h)
    return make_problem([T, P], 1.0, Nr, h, 4, quad=quad)


def test_survey_B2b_same_node_values_of_the_configured_rule():
    """b = 1.3, z = -0.8, v = 1; value = sum_nodes W conj psi_beta(r_P) e^{-i v z_m} (-1/r_P) psi_alpha(r_T) on the rule
    64 x 16 x 128, rho_max = z_pad = 40, z' panels 32/64/32, one 16-node GL panel in phi'.  The rule itself is only good
    to 1e-3 here, so agreement to 2e-8 (the five-point interpolation error of the tabulated u on h = 0.0125) pins the
    node layout and the discrete azimuthal sum; H_PT = that value for bound states (g = 0, Z_P = 1)."""
    rad = [(1, 0), (2, 0), (3, 0), (2, 1), (3, 1), (3, 2)]
    prob = _problem(rad, dict(n_rho=64, n_phi=16, n_z=128, rho_max=40.0, z_pad=40.0, phi_rule=0))
    _, HPT, _ = tr.two_centre_blocks(prob, 1.3, -0.8, 1.0)
    st = prob.centres[0].states()
    nl = {x: i for i, x in enumerate(rad)}
    idx = lambda n, l, m: st.index((nl[(n, l)], l, m))
    printed = {((1, 0, 0), (1, 0, 0)): -3.970663999321e-01 - 6.020530287319e-02j,
               ((2, 1, 1), (1, 0, 0)): -5.050123515143e-02 + 4.737430524087e-03j,
               ((3, 2, -1), (2, 1, 1)): -5.391294729332e-04 + 1.061757370399e-03j,
               ((3, 2, 2), (3, 2, -2)): -8.537510036841e-04 + 3.388638153907e-03j,
               ((2, 1, 0), (3, 2, 1)): -7.846324472049e-03 + 9.938998795516e-04j}
    for (beta, alpha), val in printed.items():
        got = HPT[idx(*beta), idx(*alpha)]
        assert abs(got - val) < 2e-8, (beta, alpha, got, val)


@pytest.fixture(scope="module")
def b4_runs():
    """p + H, hydrogen n <= 2 on both centres (order 1s, 2s, 2p-1, 2p0, 2p+1), b = 1, v = 1, z in [-30, 30]; converged
    integrals from the spheroidal rule of eq. (9) (64 x 64 nodes: identical at 90 x 90)."""
    rad = [(1, 0), (2, 0), (2, 1)]
    prob = _problem(rad, dict(kind=1, n_rho=64, n_phi=1, n_z=64, rho_max=40.0, z_pad=40.0, phi_rule=1, eta_scale=1.0), Nr=4000)
    out = {}
    for n in (600, 1200):
        h = 60.0 / n
        out[n] = oprop.propagate(prob, 1.0, 1.0, -30.0, 30.0, n, track_norm=True,
                                 matrices=lambda i, h=h: sph.S_and_H_spheroidal(prob, 1.0, -30.0 + 0.5 * i * h, 1.0))
    return out


def test_survey_B4_final_probabilities(b4_runs):
    c, drift = b4_runs[600]
    P = np.abs(c) ** 2
    printed_T = [3.2297305261e-01, 1.6983055194e-02, 7.8503987429e-04, 2.6337859681e-03, 7.8503987429e-04]
    printed_P = [6.1559344058e-01, 3.9152390893e-02, 5.0451179332e-04, 8.6529452801e-05, 5.0451179332e-04]
    np.testing.assert_allclose(P, printed_T + printed_P, rtol=0, atol=1e-6)
    assert abs(P.sum() - 1.00000136) < 2e-7                       # S != I at z_max = 30 (A17): sum |c|^2 is not 1
    assert abs(drift - 1.07e-7) < 2e-8                            # max |c^H S c - 1|: RK4 truncation at 600 steps
    assert abs(P[2] - P[4]) < 1e-12 and abs(P[7] - P[9]) < 1e-12  # reflection symmetry m <-> -m


def test_two_centre_total_probability_to_1e8_after_step_refinement(b4_runs):
    """north_star: 'unitarity, i.e. total probability = 1 to 1e-8'.  The conserved quantity is c^H S c (A17); with converged
    integrals its drift is pure RK4 truncation (global error, fourth order): 1.07e-7 at the 600 steps above, 7.7e-9 < 1e-8 after one
    refinement (ratio ~14-16)."""
    d600, d1200 = b4_runs[600][1], b4_runs[1200][1]
    assert d1200 < 1e-8
    assert 10.0 < d600 / d1200 < 20.0
