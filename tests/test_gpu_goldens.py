"""-m gpu: full-trajectory parity (SURVEY.md 8(d) "T2 propagation"; X(z_max) is what yields the
observables).  The expected final amplitudes and the drift max |c^H S c - 1| come from tests/golden/traj_cfg*_pick*.npz,
written by tests/golden/make_trajectory_goldens.py, which runs the CPU oracle only (hours of CPU time, run once).
The CUDA path propagates the same trajectories through the C ABI, in the launch configuration of the timed runs
(windows of 64 RK4 steps, mirror pairs on the symmetric z-grids), and must agree to 1e-9 on every amplitude and
probability.  The CPU-side test checks that the stored files were computed with the oracle sources as they stand.
"""
import glob
import hashlib
import os

import numpy as np
import pytest

from wpccc_inputs import build_config

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
GOLD = sorted(glob.glob(os.path.join(HERE, "golden", "traj_cfg*_pick*.npz")))
PTOL = 1e-9
EXPECTED = {0: 4, 1: 3, 2: 3, 3: 2, 4: 3}         # picks per config (make_trajectory_goldens.PICKS)
# the sources a trajectory golden depends on (oracle.propagate -> assemble -> direct / transfer / angular; the input generators
# behind build_config); modules added later (oracle/spheroidal.py, oracle/zgrid.py, wpccc_inputs/paper_shape.py) are not among them
DEPENDS = {"oracle/__init__.py", "oracle/angular.py", "oracle/assemble.py", "oracle/direct.py", "oracle/propagate.py", "oracle/transfer.py",
           "wpccc_inputs/__init__.py", "wpccc_inputs/basis.py", "wpccc_inputs/configs.py"}


def test_goldens_present_and_written_by_the_current_oracle():
    per_cfg = {}
    for f in GOLD:
        g = np.load(f)
        per_cfg[int(g["config"])] = per_cfg.get(int(g["config"]), 0) + 1
        assert DEPENDS <= {str(n) for n, _ in g["sources"]}
        for name, digest in g["sources"]:
            if str(name) not in DEPENDS:
                continue
            cur = hashlib.sha256(open(os.path.join(ROOT, str(name)), "rb").read()).hexdigest()
            assert cur == str(digest), "%s was computed with another version of %s: regenerate it (tests/golden/make_trajectory_goldens.py)" % (os.path.basename(f), name)
        C = g["C"]
        assert np.isfinite(C).all() and abs((np.abs(C) ** 2).sum() - 1.0) < 0.05
    assert per_cfg == EXPECTED, per_cfg


_basis = {}


def basis_of(lib, cfg):
    key = 2 if cfg == 4 else cfg
    if key not in _basis:
        _basis.clear()                             # one staged basis at a time (configs[2]: 0.5 GB of pair products, 40 GB windows)
        prob, _ = build_config(key)
        _basis[key] = (prob, lib.setup_basis(prob))
    return _basis[key]


@pytest.mark.gpu
@pytest.mark.parametrize("cfg", sorted(EXPECTED))
def test_full_trajectories_match_the_oracle_goldens(lib, cfg):
    files = [f for f in GOLD if int(np.load(f)["config"]) == cfg]
    assert len(files) == EXPECTED[cfg], "goldens of configs[%d] missing" % cfg
    gs = [np.load(f) for f in files]
    prob, basis = basis_of(lib, cfg)
    z0, z1, n = float(gs[0]["z_min"]), float(gs[0]["z_max"]), int(gs[0]["n_steps"])
    b = np.array([float(g["b"]) for g in gs]); v = np.array([float(g["v"]) for g in gs])
    Cg, drift = lib.propagate(basis, b, v, z0, z1, n, track_norm=True)
    Cg, drift = Cg.cpu().numpy(), drift.cpu().numpy()
    worst = 0.0
    for t, g in enumerate(gs):
        co, do = g["C"], float(g["drift"])
        err = np.abs(Cg[t] - co).max()
        worst = max(worst, err)
        assert err < PTOL, "configs[%d] b=%.4g v=%.4g: amplitudes differ by %.3e after %d steps" % (cfg, b[t], v[t], err, n)
        assert np.abs(np.abs(Cg[t]) ** 2 - np.abs(co) ** 2).max() < PTOL
        assert abs(drift[t] - do) < 1e-9 + 1e-3 * do, (cfg, t, drift[t], do)
    print("configs[%d]: %d full trajectories x %d RK4 steps, max |c_gpu - c_oracle| = %.3e" % (cfg, len(gs), n, worst))
    if len(prob.centres) == 2:
        # the explicit-inverse route of the overlap solve (wpccc_set_option "solve_route" 1) on the same trajectories
        basis.set_option("solve_route", 1)
        try:
            Ci = lib.propagate(basis, b, v, z0, z1, n).cpu().numpy()
        finally:
            basis.set_option("solve_route", 0)
        worst_i = max(np.abs(Ci[t] - g["C"]).max() for t, g in enumerate(gs))
        assert worst_i < PTOL
        print("configs[%d]: explicit Gauss-Jordan inverse route: max |c_gpu - c_oracle| = %.3e (Cholesky + triangular solves: %.3e)" % (cfg, worst_i, worst))
