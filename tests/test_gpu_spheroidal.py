"""-m gpu: SURVEY.md 8(f) NEXT-2, the paper's own quadrature of eq. (9) (prolate spheroidal Gauss-Laguerre x Gauss-Legendre,
analytic Bessel azimuth; wpccc_quad.kind = 1) through the C ABI against oracle/spheroidal.py, element by element
(1e-11 relative, 1e-13 floor), and a propagation through it (1e-9)."""
import numpy as np
import pytest

from oracle import propagate as oprop
from oracle import spheroidal as sph
from wpccc_inputs import build_config, tiny_problem
from wpccc_inputs.basis import make_problem

pytestmark = pytest.mark.gpu
REL, FLOOR, PTOL = 1e-11, 1e-13, 1e-9


def assert_elements(got, ref, what):
    err = np.abs(np.asarray(got) - np.asarray(ref))
    bad = err > REL * np.abs(ref) + FLOOR
    assert not bad.any(), "%s: %d of %d elements out of tolerance; worst |err| %.3e" % (what, bad.sum(), bad.size, err[bad].max())


def test_spheroidal_elements_and_propagation_tiny(lib):
    q = dict(kind=1, n_rho=20, n_phi=1, n_z=32, rho_max=30.0, z_pad=30.0, phi_rule=1, eta_scale=1.2)
    prob = tiny_problem(True, l_max=2, n_max=3, bins=2, k_max=2.0, Nr=400, h=0.1, Z_T=1.0, Z_P=2.0, quad=q, seed=11)
    basis = lib.setup_basis(prob)
    pos = [(1.3, -0.8, 1.0), (0.4, 2.2, 1.5), (2.5, 0.0, 0.8), (0.2, -6.0, 1.0), (0.05, 0.02, 2.0)]
    b, z, v = map(np.array, zip(*pos))
    S, H = lib.matrix_elements(basis, b, z, v, phases=True)
    S, H = S.cpu().numpy(), H.cpu().numpy()
    for p in range(len(b)):
        So, Ho = sph.S_and_H_spheroidal(prob, b[p], z[p], v[p])
        assert_elements(S[p], So, "S (spheroidal) at position %d" % p)
        assert_elements(H[p], Ho, "H (spheroidal) at position %d" % p)
    bt, vt, n_steps = np.array([1.6, 0.9]), np.array([1.0, 1.3]), 30
    basis.set_option("solve_route", 1)                    # no definiteness requirement on the coarse rule
    Cg = lib.propagate(basis, bt, vt, -6.0, 6.0, n_steps).cpu().numpy()
    h = 12.0 / n_steps
    for t in range(2):
        co = oprop.propagate(prob, bt[t], vt[t], -6.0, 6.0, n_steps,
                             matrices=lambda i, t=t: sph.S_and_H_spheroidal(prob, bt[t], -6.0 + 0.5 * i * h, vt[t]))
        assert np.abs(Cg[t] - co).max() < PTOL, (t, np.abs(Cg[t] - co).max())
    basis.close()


def test_spheroidal_elements_at_config1_size(lib):
    """The configs[1] basis (172 states, l <= 2) with a 48 x 64 spheroidal rule; a batch that spans a whole launch chunk,
    sampled positions against the oracle."""
    prob, run = build_config(1)
    q = dict(kind=1, n_rho=48, n_phi=1, n_z=64, rho_max=40.0, z_pad=40.0, phi_rule=1, eta_scale=1.0)
    prob = make_problem(prob.centres, prob.Z_proj, prob.Nr, prob.h, prob.lambda_max, quad=q, meta=dict(config="1-spheroidal"))
    basis = lib.setup_basis(prob)
    rng = np.random.default_rng(21)
    n = 150
    b, z, v = rng.choice(run["b"], n), rng.uniform(-20.0, 20.0, n), np.ones(n)
    b[:3] = [run["b"][0], run["b"][8], run["b"][15]]; z[:3] = [-0.37, 5.3, -0.37]
    S, H = lib.matrix_elements(basis, b, z, v, phases=True)
    for p in (0, 1, 2, 149):
        So, Ho = sph.S_and_H_spheroidal(prob, b[p], z[p], v[p])
        assert_elements(S[p].cpu().numpy(), So, "configs[1] basis, spheroidal S at %d" % p)
        assert_elements(H[p].cpu().numpy(), Ho, "configs[1] basis, spheroidal H at %d" % p)
    basis.close()
