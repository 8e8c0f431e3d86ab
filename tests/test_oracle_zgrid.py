"""Pins for oracle/zgrid.py: the z-grid of PAPER.md L67 and Algorithm 1 on a non-uniform grid."""
import numpy as np
import scipy.linalg

from oracle import propagate as oprop
from oracle import zgrid
from wpccc_inputs import tiny_problem


def test_paper_zgrid_layout():
    g = zgrid.paper_zgrid(1e-3, 100.0, 500)                      # the paper's typical values (L67)
    assert len(g) == 1001 and g[500] == 0.0 and np.all(np.diff(g) > 0)
    assert g[-1] == 100.0 and g[0] == -100.0 and np.array_equal(g, -g[::-1])
    assert abs(g[501] - 1e-3 * (1e5) ** (1 / 500)) < 1e-18        # zgrid[1] = z_min (z_max/z_min)^(1/n_z)
    ratio = g[502:] / g[501:-1]
    assert np.allclose(ratio, (100.0 / 1e-3) ** (1 / 500), rtol=1e-13)   # geometric: denser near closest approach
    assert np.diff(g)[500] < 1.1e-3 and np.diff(g)[-1] > 2.0


def test_grid_propagation_reduces_to_the_uniform_algorithm_and_counts_evaluations():
    prob = tiny_problem(False, l_max=1, n_max=2, bins=2, k_max=2.0, Nr=300, h=0.1)
    n = 24
    zg = -6.0 + 0.5 * np.arange(n + 1)
    calls = []
    from oracle.assemble import S_and_H

    def mats(z):
        calls.append(z)
        return S_and_H(prob, 0.8, float(z), 1.2)
    c_grid = zgrid.propagate_grid(prob, 0.8, 1.2, zg, matrices=mats)
    assert len(calls) == 2 * n + 1                                # 4 n_z + 1 evaluations for 2 n_z steps
    c_uni = oprop.propagate(prob, 0.8, 1.2, -6.0, 6.0, n)
    assert np.abs(c_grid - c_uni).max() < 1e-14


def test_nonuniform_grid_against_the_matrix_exponential():
    """Constant M: the exact solution is exp(M (z_end - z_0)) c_0 whatever the grid; RK4 local error h^5."""
    rng = np.random.default_rng(3)
    A = rng.normal(size=(5, 5)); Hc = 0.25 * (A + A.T).astype(np.complex128)
    prob = tiny_problem(False, l_max=0, n_max=5, bins=0, Nr=300, h=0.1)
    assert prob.n_tot == 5
    v = 1.3
    errs = []
    for nz in (20, 40):
        g = zgrid.paper_zgrid(0.05, 2.0, nz)
        c = zgrid.propagate_grid(prob, 1.0, v, g, matrices=lambda z: (np.eye(5), Hc))
        exact = scipy.linalg.expm((-1j / v) * Hc * (g[-1] - g[0]))[:, 0]
        errs.append(np.abs(c - exact).max())
    assert errs[0] < 1e-3 and 8.0 < errs[0] / errs[1] < 40.0       # fourth order on the refined geometric grid
