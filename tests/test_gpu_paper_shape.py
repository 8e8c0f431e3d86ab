"""-m gpu: SURVEY.md 8(f) NEXT-3, the paper's own workload shape at its large end: the two-centre basis of
l_max = 5 (N = 1910, the largest two-centre size the paper reports) and a one-centre basis of l_max = 5 (N = 1387,
multipoles up to lambda = 10), one position each against the oracle, element by element.  These sizes take the paths the
five BASELINE.json configs do not: l > 4 (generic direct assembly), rotation in passes over blocks of target states,
18 column tiles per side in the contraction.  (The oracle needs a minute or two per position at these sizes.)"""
import numpy as np
import pytest

from oracle import assemble
from wpccc_inputs.paper_shape import SIZES_1C, SIZES_2C, paper_problem

pytestmark = pytest.mark.gpu
REL, FLOOR = 1e-11, 1e-13


def assert_elements(got, ref, what):
    err = np.abs(np.asarray(got) - np.asarray(ref))
    bad = err > REL * np.abs(ref) + FLOOR
    assert not bad.any(), "%s: %d of %d elements out of tolerance; worst |err| %.3e" % (what, bad.sum(), bad.size, err[bad].max())


@pytest.mark.parametrize("two,l_max", [(True, 5), (False, 5)])
def test_paper_shaped_basis_elements(lib, two, l_max):
    prob, run = paper_problem(two, l_max)
    assert prob.n_tot == (SIZES_2C if two else SIZES_1C)[l_max]
    basis = lib.setup_basis(prob)
    b, z, v = 1.3, -0.8, 2.0
    S, H = lib.matrix_elements(basis, [b, 0.7, 4.0], [z, 3.1, -9.0], [v, v, v], phases=True)      # three positions, the first one compared
    So, Ho = assemble.S_and_H(prob, b, z, v)
    assert_elements(H[0].cpu().numpy(), Ho, "paper-shaped %s l_max = %d: H" % ("2C" if two else "1C", l_max))
    assert_elements(S[0].cpu().numpy(), So, "paper-shaped %s l_max = %d: S" % ("2C" if two else "1C", l_max))
    if not two:                                              # a few RK4 steps on the central part of the paper's z-grid run through
        g = run["zgrid"]
        mid = len(g) // 2
        C = lib.propagate_grid(basis, run["b"][:2], run["v"][:2], g[mid - 4: mid + 5])
        assert bool(C.isfinite().all()) and abs(float((C.abs() ** 2).sum(1)[0]) - 1.0) < 1e-6
    basis.close()
    lib.release_workspace()
