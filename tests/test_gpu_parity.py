"""-m gpu: parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances (BASELINE.json north_star): matrix elements 1e-11 relative with a 1e-13 absolute floor;
transition probabilities 1e-9 absolute."""
import numpy as np
import pytest

from oracle import assemble, direct, observables
from oracle import propagate as oprop
from oracle import transfer as otr
from wpccc_inputs import tiny_problem

pytestmark = pytest.mark.gpu

REL, FLOOR, PTOL = 1e-11, 1e-13, 1e-9


def assert_elements(got, ref, what, scale=None):
    got, ref = np.asarray(got), np.asarray(ref)
    assert got.shape == ref.shape, (what, got.shape, ref.shape)
    err = np.abs(got - ref)
    tol = REL * np.abs(ref) + FLOOR
    bad = err > tol
    assert not bad.any(), "%s: %d of %d elements out of tolerance; worst |err| %.3e at |ref| %.3e" % (
        what, bad.sum(), bad.size, err[bad].max(), np.abs(ref[bad][np.argmax(err[bad])]))


POS1 = [(0.5, -0.37, 2.0), (0.5, 5.3, 2.0), (1.7, 0.0, 1.0), (4.0, -12.25, 0.7), (0.05, 0.02, 3.0), (3.0, 90.0, 1.0)]


@pytest.fixture(scope="module")
def one_centre(lib):
    prob = tiny_problem(False, l_max=2, n_max=3, bins=3, k_max=2.5, Nr=437, h=0.1, lambda_max=4)   # ragged Nr (not a multiple of 32)
    return prob, lib.setup_basis(prob)


def test_fp64_peaks_report(lib):
    dfma, dmma = lib.fp64_peak(0), lib.fp64_peak(1)
    print("FP64 peak: DFMA %.2f TFLOP/s, DMMA %.2f TFLOP/s" % (dfma, dmma))
    assert dfma > 5 and dmma > 5


def test_direct_radial_entries_and_elements(lib, one_centre):
    prob, basis = one_centre
    b, z, v = map(np.array, zip(*POS1))
    S, H, F = lib.matrix_elements(basis, b, z, v, phases=True, want_F=True)
    S, H, F = S.cpu().numpy(), H.cpu().numpy(), F.cpu().numpy()
    ent = basis.radial_entries(0)
    r = prob.h * np.arange(prob.Nr + 1)
    for p in range(len(b)):
        R = float(np.hypot(b[p], z[p]))
        Fo = direct.radial_F_all(prob.centres[0], prob.w, r, R, prob.lambda_max)
        ref = np.array([Fo[lam, a1, a] for (a1, a, lam) in ent])
        assert_elements(F[p], ref, "F at position %d" % p)
        So, Ho = assemble.S_and_H(prob, b[p], z[p], v[p])
        assert_elements(H[p], Ho, "D^T at position %d" % p)
        assert_elements(S[p], So, "S (identity) at position %d" % p)
    # element-by-element definition (loops) at one position
    Dl = direct.direct_block_loops(prob.centres[0], prob.w, r, prob.lambda_max, b[0], z[0], v[0], prob.Z_proj, False)
    assert_elements(H[0], Dl, "D^T vs loop definition")


def test_direct_many_positions_span_tiles(lib, one_centre):
    """300 positions (3 M-tiles with a ragged tail); sampled rows against the oracle, all rows for symmetry."""
    prob, basis = one_centre
    rng = np.random.default_rng(7)
    n = 300
    b, z, v = rng.uniform(0.05, 6.0, n), rng.uniform(-30.0, 30.0, n), np.full(n, 1.3)
    _, H, F = lib.matrix_elements(basis, b, z, v, phases=False, want_S=False, want_F=True)
    H, F = H.cpu().numpy(), F.cpu().numpy()
    assert np.abs(H.imag).max() == 0.0 and np.abs(H - H.transpose(0, 2, 1)).max() < 1e-15
    ent = basis.radial_entries(0)
    r = prob.h * np.arange(prob.Nr + 1)
    for p in (0, 127, 128, 255, 256, 299):
        Fo = direct.radial_F_all(prob.centres[0], prob.w, r, float(np.hypot(b[p], z[p])), prob.lambda_max)
        assert_elements(F[p], np.array([Fo[lam, a1, a] for (a1, a, lam) in ent]), "F at position %d" % p)


def test_direct_tables_route(lib, one_centre):
    """prefix/suffix tables instead of the GEMM, ragged Nr, all positions against the oracle."""
    prob, basis = one_centre
    b, z, v = map(np.array, zip(*POS1))
    basis.enable_direct_tables(True)
    try:
        S, H, F = lib.matrix_elements(basis, b, z, v, phases=True, want_F=True)
        H, F = H.cpu().numpy(), F.cpu().numpy()
        ent = basis.radial_entries(0)
        r = prob.h * np.arange(prob.Nr + 1)
        for p in range(len(b)):
            Fo = direct.radial_F_all(prob.centres[0], prob.w, r, float(np.hypot(b[p], z[p])), prob.lambda_max)
            assert_elements(F[p], np.array([Fo[lam, a1, a] for (a1, a, lam) in ent]), "table F at position %d" % p)
            So, Ho = assemble.S_and_H(prob, b[p], z[p], v[p])
            assert_elements(H[p], Ho, "D^T (tables) at position %d" % p)
    finally:
        basis.enable_direct_tables(False)


def test_one_centre_propagation_and_probabilities(lib, one_centre):
    prob, basis = one_centre
    b = np.array([0.6, 0.6, 2.0, 0.6, 1.1])          # repeated b: trajectories share matrices
    v = np.array([1.0, 2.0, 2.0, 0.7, 1.5])
    n_steps = 90
    Cg, drift = lib.propagate(basis, b, v, -15.0, 15.0, n_steps, track_norm=True)
    Cg, drift = Cg.cpu().numpy(), drift.cpu().numpy()
    for t in range(len(b)):
        co, do = oprop.propagate(prob, b[t], v[t], -15.0, 15.0, n_steps, track_norm=True)
        assert np.abs(np.abs(Cg[t]) ** 2 - np.abs(co) ** 2).max() < PTOL
        assert np.abs(Cg[t] - co).max() < PTOL
        assert abs(drift[t] - do) < 1e-12 + 1e-6 * do
    out = lib.probabilities(basis, lib._torch().as_tensor(Cg, device="cuda"), b=b, vgroup=np.array([0, 1, 1, 2, 3]), n_vgroups=4)
    Ps, Pnl, Pc = observables.probabilities(prob, Cg)
    assert np.abs(out["P_state"].cpu().numpy() - Ps).max() < 1e-15
    assert np.abs(out["P_nl"].cpu().numpy() - Pnl).max() < 1e-15
    assert np.abs(out["P_class"].cpu().numpy() - Pc).max() < 1e-14
    sig = observables.cross_sections(b, np.array([0, 1, 1, 2, 3]), Pnl, 4)
    assert np.abs(out["sigma_nl"].cpu().numpy() - sig).max() < 1e-13


def test_one_centre_windows_do_not_change_the_result(lib, one_centre):
    """A workspace that forces short windows gives the same amplitudes (window boundaries are exact restarts)."""
    prob, basis = one_centre
    b, v = np.array([0.9, 2.5]), np.array([1.0, 1.0])
    big = lib.propagate(basis, b, v, -10.0, 10.0, 70).cpu().numpy()
    small_ws = lib._lib.wpccc_workspace_bytes(basis._h, 2, 70, 2) + (1 << 20)
    small = lib.propagate(basis, b, v, -10.0, 10.0, 70, ws_bytes=small_ws).cpu().numpy()
    assert np.abs(big - small).max() < 1e-14


def test_one_centre_mirror_of_the_radial_entries(lib, one_centre):
    """On a z-grid symmetric about 0 the direct radial entries F(R) of eq. (7) are contracted for z <= 0 only and reused at
    +z (same R; wpccc.h, wpccc_last_units): several windows (150 steps > 64), repeated b, GEMM and table routes, against the
    run with the mirror switched off and against the oracle; an asymmetric grid switches it off by itself."""
    prob, basis = one_centre
    b, v = np.array([0.6, 2.0, 0.6]), np.array([1.0, 1.3, 0.8])          # two distinct b
    n_steps = 150
    n_pos = 2 * (2 * n_steps + 3)          # windows of 64, 64, 22 steps; consecutive windows share their boundary position
    Cm = lib.propagate(basis, b, v, -12.0, 12.0, n_steps).cpu().numpy()
    assert lib.last_units(basis)["direct_gemm"] == 2 * (n_steps + 2), lib.last_units(basis)
    small_ws = lib._lib.wpccc_workspace_bytes(basis._h, 3, n_steps, 2) + (1 << 20)                 # short windows
    Cs = lib.propagate(basis, b, v, -12.0, 12.0, n_steps, ws_bytes=small_ws).cpu().numpy()
    assert lib.last_units(basis)["direct_gemm"] >= 2 * (n_steps + 2)                               # short windows, with or without the table
    basis.set_option("mirror_pairs", 0)
    try:
        C0 = lib.propagate(basis, b, v, -12.0, 12.0, n_steps).cpu().numpy()
        assert lib.last_units(basis)["direct_gemm"] == n_pos
    finally:
        basis.set_option("mirror_pairs", 1)
    assert np.abs(Cm - C0).max() < 1e-13 and np.abs(Cs - C0).max() < 1e-13, (np.abs(Cm - C0).max(), np.abs(Cs - C0).max())
    for t in (0, 1):
        co = oprop.propagate(prob, b[t], v[t], -12.0, 12.0, n_steps)
        assert np.abs(Cm[t] - co).max() < PTOL
    basis.enable_direct_tables(True)
    try:
        Ct = lib.propagate(basis, b, v, -12.0, 12.0, n_steps).cpu().numpy()
        assert lib.last_units(basis)["direct_gemm"] == 2 * (n_steps + 2)
    finally:
        basis.enable_direct_tables(False)
    assert np.abs(Ct - C0).max() < 1e-11
    Ca = lib.propagate(basis, b[:1], v[:1], -6.0, 4.0, 25).cpu().numpy()
    assert lib.last_units(basis)["direct_gemm"] == 51
    assert np.abs(Ca[0] - oprop.propagate(prob, b[0], v[0], -6.0, 4.0, 25)).max() < PTOL


# ------------------------------------------------------------------------------------------------ two centres
QUAD = dict(n_rho=24, n_phi=8, n_z=48, rho_max=30.0, z_pad=30.0, phi_rule=0)
POS2 = [(1.3, -0.8, 1.0), (0.4, 2.2, 1.5), (2.5, 0.0, 0.8), (0.2, -6.0, 1.0)]


@pytest.fixture(scope="module")
def two_centre(lib):
    prob = tiny_problem(True, l_max=2, n_max=3, bins=2, k_max=2.0, Nr=400, h=0.1, Z_T=1.0, Z_P=2.0, quad=dict(QUAD), seed=11)
    return prob, lib.setup_basis(prob)


def test_two_centre_elements(lib, two_centre):
    prob, basis = two_centre
    b, z, v = map(np.array, zip(*POS2))
    S, H = lib.matrix_elements(basis, b, z, v, phases=True)
    S, H = S.cpu().numpy(), H.cpu().numpy()
    NT = prob.centres[0].n_states
    for p in range(len(b)):
        So, Ho = assemble.S_and_H(prob, b[p], z[p], v[p])
        assert_elements(S[p], So, "S at position %d" % p)
        assert_elements(H[p][:NT, :NT], Ho[:NT, :NT], "D^T at position %d" % p)
        assert_elements(H[p][NT:, NT:], Ho[NT:, NT:], "D^P at position %d" % p)
        assert_elements(H[p][NT:, :NT], Ho[NT:, :NT], "H_PT at position %d" % p)
        assert_elements(H[p][:NT, NT:], Ho[:NT, NT:], "H_TP at position %d" % p)
    # lab-frame definition (L0) on a few seeded pairs, no time phases
    S0, H0 = lib.matrix_elements(basis, b[:1], z[:1], v[:1], phases=False)
    S0, H0 = S0.cpu().numpy()[0], H0.cpu().numpy()[0]
    T, P = prob.centres
    rng = np.random.default_rng(3)
    stT, stP = T.states(), P.states()
    for _ in range(6):
        ia, ib = int(rng.integers(len(stT))), int(rng.integers(len(stP)))
        for kind, got in (("S", S0[NT + ib, ia]), ("HPT", H0[NT + ib, ia]), ("HTP", H0[ia, NT + ib])):
            ref = otr.lab_frame_element(prob, stP[ib], stT[ia], b[0], z[0], v[0], kind)
            assert abs(got - ref) <= REL * abs(ref) + FLOOR, (kind, ia, ib, got, ref)


def test_two_centre_bessel_rule(lib):
    q = dict(QUAD); q["phi_rule"] = 1
    prob = tiny_problem(True, l_max=1, n_max=2, bins=1, k_max=1.5, Nr=300, h=0.1, quad=q)
    basis = lib.setup_basis(prob)
    S, H = lib.matrix_elements(basis, [0.9], [-1.3], [1.0])
    So, Ho = assemble.S_and_H(prob, 0.9, -1.3, 1.0)
    assert_elements(S.cpu().numpy()[0], So, "S (Bessel azimuth)")
    assert_elements(H.cpu().numpy()[0], Ho, "H (Bessel azimuth)")


def test_two_centre_propagation(lib, two_centre):
    prob, basis = two_centre
    b, v = np.array([0.7, 1.9, 0.7]), np.array([1.0, 1.0, 1.6])
    n_steps = 40
    Cg, drift = lib.propagate(basis, b, v, -8.0, 8.0, n_steps, track_norm=True)
    Cg, drift = Cg.cpu().numpy(), drift.cpu().numpy()
    for t in range(len(b)):
        co, do = oprop.propagate(prob, b[t], v[t], -8.0, 8.0, n_steps, track_norm=True)
        assert np.abs(np.abs(Cg[t]) ** 2 - np.abs(co) ** 2).max() < PTOL, t
        assert np.abs(Cg[t] - co).max() < PTOL, t
        assert abs(drift[t] - do) < 1e-10 + 1e-4 * do
    small_ws = lib._lib.wpccc_workspace_bytes(basis._h, 3, n_steps, 2) + (4 << 20)
    Cs = lib.propagate(basis, b, v, -8.0, 8.0, n_steps, ws_bytes=small_ws).cpu().numpy()
    assert np.abs(Cs - Cg).max() < 1e-13


def test_two_centre_mirror_pairs(lib, two_centre):
    """On a z-grid symmetric about 0 the body-frame integrals of (b, -z) and (b, +z) are evaluated together (wpccc.h,
    wpccc_last_units).  Several windows (150 steps > 64), full and partial stash, against the run with the pairing
    switched off; and an asymmetric grid, where pairing must switch itself off, against the oracle."""
    prob, basis = two_centre
    b, v = np.array([0.7, 1.9, 0.4]), np.array([1.0, 1.3, 1.6])
    n_steps = 150
    n_pos = 3 * (2 * n_steps + 3)          # windows of 64, 64, 22 steps; consecutive windows share their boundary position
    Cm = lib.propagate(basis, b, v, -9.0, 9.0, n_steps).cpu().numpy()
    um = lib.last_units(basis)
    assert um["transfer_contraction"] == 3 * (n_steps + 2) and um["rotation"] == n_pos, um       # z <= 0 evaluated, z > 0 fetched
    assert um["direct_gemm"] == 3 * (n_steps + 2), um                                            # F(R) of eq. (7): the same at -z and +z
    base = lib._lib.wpccc_workspace_bytes(basis._h, 3, n_steps, 1)
    part = lib._lib.wpccc_workspace_bytes(basis._h, 3, 64, 1)                                   # room for 64 of the 150 mirror indices
    Cp = lib.propagate(basis, b, v, -9.0, 9.0, n_steps, ws_bytes=part).cpu().numpy()
    up = lib.last_units(basis)
    assert 3 * (n_steps + 2) < up["transfer_contraction"] < n_pos and part < base, (up, part, base)
    basis.set_option("mirror_pairs", 0)
    try:
        C0 = lib.propagate(basis, b, v, -9.0, 9.0, n_steps).cpu().numpy()
        assert lib.last_units(basis)["transfer_contraction"] == n_pos and lib.last_units(basis)["direct_gemm"] == n_pos
    finally:
        basis.set_option("mirror_pairs", 1)
    assert np.abs(Cm - C0).max() < 1e-12 and np.abs(Cp - C0).max() < 1e-12, (np.abs(Cm - C0).max(), np.abs(Cp - C0).max())
    Ca = lib.propagate(basis, b[:1], v[:1], -6.0, 4.0, 25).cpu().numpy()
    assert lib.last_units(basis)["transfer_contraction"] == 51
    co = oprop.propagate(prob, b[0], v[0], -6.0, 4.0, 25)
    assert np.abs(Ca[0] - co).max() < PTOL


def test_sweep_cluster_sizes_agree(lib, two_centre):
    """wpccc_set_option "sweep_cluster": the two-centre RK4 sweep on one CTA per trajectory and on thread-block clusters of two
    and four CTAs (products split by rows, partial sums exchanged through distributed shared memory) -- the same amplitudes
    to rounding, on both solve routes, with the norm tracked, over several windows; and against the oracle."""
    prob, basis = two_centre
    b, v = np.array([0.7, 1.9, 1.2]), np.array([1.0, 1.3, 0.8])
    n_steps = 70
    ref = {}
    try:
        for route in (0, 1):
            basis.set_option("solve_route", route)
            for nc in (1, 2, 4):
                basis.set_option("sweep_cluster", nc)
                C, drift = lib.propagate(basis, b, v, -7.0, 7.0, n_steps, track_norm=True)
                C, drift = C.cpu().numpy(), drift.cpu().numpy()
                assert np.isfinite(C).all()
                if nc == 1:
                    ref[route] = (C, drift)
                else:
                    assert np.abs(C - ref[route][0]).max() < 1e-13, (route, nc, np.abs(C - ref[route][0]).max())
                    assert np.abs(drift - ref[route][1]).max() < 1e-12
    finally:
        basis.set_option("solve_route", 0)
        basis.set_option("sweep_cluster", 0)
    co = oprop.propagate(prob, b[0], v[0], -7.0, 7.0, n_steps)
    assert np.abs(ref[0][0][0] - co).max() < PTOL
    with pytest.raises(lib.WpcccError):
        basis.set_option("sweep_cluster", 3)


ROUTES = (("cholesky + triangular solves", {"solve_route": 0}),
          ("inverse, registers", {"solve_route": 1}),
          ("inverse, registers, K staged in chunks of 5 columns", {"solve_route": 1, "inverse_chunk_cols": 5}),
          ("inverse, shared memory", {"solve_route": 1, "inverse_kernel": 1}),
          ("inverse, global-memory blocked", {"solve_route": 1, "inverse_kernel": 2}))
ROUTE_DEFAULTS = {"solve_route": 0, "inverse_kernel": 0, "inverse_chunk_cols": 0}


def with_route(basis, opts, fn):
    for k, val in {**ROUTE_DEFAULTS, **opts}.items():
        basis.set_option(k, val)
    try:
        return fn()
    finally:
        for k, val in ROUTE_DEFAULTS.items():
            basis.set_option(k, val)


def test_two_centre_factor_routes(lib, two_centre):
    """The routes of the a7 overlap solve (wpccc_set_option "solve_route": blocked Cholesky factor + triangular solves per
    stage; explicit Gauss-Jordan inverse with the matrix in registers for N_P <= 90, in shared memory, blocked in global
    memory) solve the same systems and differ by rounding only; each against the oracle's plain partial-pivoting solve
    on the full S.  N_P = 32 (whole panels) and N_P = 9 (one lane group, ragged last panel / block)."""
    small = tiny_problem(True, l_max=1, n_max=2, bins=1, k_max=1.5, Nr=300, h=0.1, quad=dict(QUAD), seed=5)
    for prob, basis, b, v, zr, n_steps in ((two_centre[0], two_centre[1], np.array([1.6, 1.1]), np.array([0.9, 1.4]), 7.0, 30),
                                           (small, lib.setup_basis(small), np.array([0.5]), np.array([1.2]), 6.0, 24)):
        out = {name: with_route(basis, opts, lambda: lib.propagate(basis, b, v, -zr, zr, n_steps).cpu().numpy()) for name, opts in ROUTES}
        for t in range(len(b)):
            co = oprop.propagate(prob, b[t], v[t], -zr, zr, n_steps)
            for route, C in out.items():
                assert np.abs(C[t] - co).max() < PTOL, (route, t, np.abs(C[t] - co).max())
        for route, C in out.items():
            assert np.abs(C - out["inverse, shared memory"]).max() < 1e-11, route


def test_overlap_not_positive_definite_is_reported(lib, two_centre):
    """With the coarse 24 x 8 x 48 rule the discretised overlap matrix of this basis is indefinite at small R: the default
    route (Cholesky) reports the first such position of the trajectory (WPCCC_ESINGULAR, wpccc_last_status) and returns
    NaN for it, the other trajectory is complete; the oracle confirms the sign change of the smallest eigenvalue of
    I - K K^H exactly there; the explicit-inverse route propagates straight through (S is indefinite, not singular)."""
    prob, basis = two_centre
    b, v, zr, n_steps = np.array([0.3, 1.1]), np.array([0.9, 1.4]), 7.0, 30
    with pytest.raises(lib.WpcccError) as ei:
        lib.propagate(basis, b, v, -zr, zr, n_steps)
    assert ei.value.code == -4 and "not positive definite" in str(ei.value)
    C = lib.propagate(basis, b, v, -zr, zr, n_steps, allow_singular=True).cpu().numpy()
    st = lib.last_status(basis, 2)
    assert st[1] is None and st[0] is not None and st[0][0] == 3
    assert np.isnan(C[0]).all() and np.isfinite(C[1]).all()
    assert np.abs(C[1] - oprop.propagate(prob, b[1], v[1], -zr, zr, n_steps)).max() < PTOL
    i_bad = st[0][1]
    h = 2 * zr / n_steps
    NT = prob.centres[0].n_states

    def min_eig(i):
        S, _ = assemble.S_and_H(prob, b[0], -zr + 0.5 * i * h, v[0], time_phase=False)
        K = S[NT:, :NT]
        return np.linalg.eigvalsh(np.eye(K.shape[0]) - K @ K.conj().T).min()

    assert min_eig(i_bad) < 0.0 < min(min_eig(i) for i in range(max(0, i_bad - 3), i_bad))
    Ci = with_route(basis, {"solve_route": 1}, lambda: lib.propagate(basis, b, v, -zr, zr, n_steps).cpu().numpy())
    assert np.abs(Ci[0] - oprop.propagate(prob, b[0], v[0], -zr, zr, n_steps)).max() < PTOL


def test_argument_errors(lib, one_centre):
    prob, basis = one_centre
    with pytest.raises(lib.WpcccError):
        lib.propagate(basis, [1.0], [0.0], -1.0, 1.0, 10)             # v = 0
    with pytest.raises(lib.WpcccError):
        lib.propagate(basis, [1.0], [1.0], -1.0, 1.0, 10, ws_bytes=1024)   # workspace too small
    assert lib.propagate(basis, np.zeros(0), np.zeros(0), -1.0, 1.0, 10).shape == (0, basis.n_tot)   # empty batch


def test_workspace_query_is_sufficient_for_a_first_call(lib):
    """wpccc_workspace_bytes(what = 0) must cover wpccc_matrix_elements on a fresh basis (no larger workspace cached by
    an earlier call): one centre and two centres, with and without the H output."""
    for two in (False, True):
        prob = tiny_problem(two, l_max=1, n_max=2, bins=2, k_max=2.0, Nr=300, h=0.1, quad=dict(QUAD) if two else None, seed=5 if two else None)
        for kw in ({}, {"want_H": False}, {"want_S": False}):
            basis = lib.setup_basis(prob)
            out = lib.matrix_elements(basis, [0.8, 1.1, 0.3], [-0.6, 0.2, 1.4], [1.2, 1.2, 0.9], **kw)
            assert all(t is None or bool(t.isfinite().all()) for t in out)
            basis.close()


def test_paper_zgrid_propagation(lib, one_centre, two_centre):
    """wpccc_propagate_grid on the z-grid of PAPER.md L67 (geometric, symmetric about 0, step sizes
    from 1e-3 to ~1) against Algorithm 1 on the same grid (oracle/zgrid.py), one and two centres; windows of 64 steps,
    mirror pairs on the symmetric grid."""
    from oracle import zgrid
    g = zgrid.paper_zgrid(1e-3, 9.0, 70)                                   # 141 points, 140 steps: three windows
    for (prob, basis), b, v in ((one_centre, np.array([0.6, 2.0, 0.6]), np.array([1.0, 2.0, 0.7])),
                                (two_centre, np.array([1.6, 1.1]), np.array([0.9, 1.4]))):
        Cg, drift = lib.propagate_grid(basis, b, v, g, track_norm=True)
        Cg, drift = Cg.cpu().numpy(), drift.cpu().numpy()
        for t in range(len(b)):
            co, do = zgrid.propagate_grid(prob, b[t], v[t], g, track_norm=True)
            assert np.abs(Cg[t] - co).max() < PTOL, (t, np.abs(Cg[t] - co).max())
            assert abs(drift[t] - do) < 1e-10 + 1e-4 * do
    if True:                                                               # continuation: two calls = one call
        prob, basis = two_centre
        b, v = np.array([1.6, 1.1]), np.array([0.9, 1.4])
        C1 = lib.propagate(basis, b, v, -8.0, 8.0, 40).cpu().numpy()
        Ca = lib.propagate(basis, b, v, -8.0, -1.6, 16)
        Cb = lib.propagate(basis, b, v, -1.6, 8.0, 24, C0=Ca).cpu().numpy()
        assert np.abs(Cb - C1).max() < 1e-12


def test_explicit_coupling_matrix(lib, one_centre, two_centre):
    """M = -(i/v) S^{-1} H of eq. (4) with N_tot right-hand sides (the paper's ZGESV usage)
    against the oracle's S and H and a library solve; one centre: M = -(i/v) D^T (eq. (5))."""
    for (prob, basis), pos in ((two_centre, POS2), (one_centre, POS1[:3])):
        b, z, v = map(np.array, zip(*pos))
        M = lib.coupling_matrix(basis, b, z, v).cpu().numpy()
        for p in range(len(b)):
            So, Ho = assemble.S_and_H(prob, b[p], z[p], v[p])
            Mo = (-1j / v[p]) * np.linalg.solve(So, Ho)
            assert np.abs(M[p] - Mo).max() < 1e-12 + 1e-13 * np.abs(Mo).max() * np.linalg.cond(So), (p, np.abs(M[p] - Mo).max())


def test_nonuniform_radial_grid(lib):
    """wpccc_setup_basis_grid (radial grid denser around the origin): eq. (7) sums over the given
    points, the node tables interpolate on the actual abscissae; elements (GEMM and table routes) and a propagation against
    oracle/nonuniform.py, one and two centres."""
    from oracle import nonuniform as nu
    from wpccc_inputs.paper_shape import exponential_grid, resample_problem
    g = exponential_grid(437, 40.0, 4.0)                                        # ragged Nr
    for two in (False, True):
        fine = tiny_problem(two, l_max=2, n_max=3, bins=2, k_max=2.0, Nr=2000, h=0.02, Z_P=2.0 if two else 1.0, quad=dict(QUAD) if two else None, seed=11 if two else None)
        prob = resample_problem(fine, g)
        basis = lib.setup_basis(prob)
        pos = POS2 + [(0.03, 0.01, 1.0), (3.0, 38.5, 1.0)] if two else POS1      # incl. R below r_1-ish and nodes beyond r_max
        b, z, v = map(np.array, zip(*pos))
        S, H = lib.matrix_elements(basis, b, z, v, phases=True)
        S, H = S.cpu().numpy(), H.cpu().numpy()
        for p in range(len(b)):
            So, Ho = nu.S_and_H_grid(prob, g, b[p], z[p], v[p])
            assert_elements(S[p], So, "S on the non-uniform grid, position %d" % p)
            assert_elements(H[p], Ho, "H on the non-uniform grid, position %d" % p)
        if not two:
            basis.enable_direct_tables(True)
            _, Ht = lib.matrix_elements(basis, b, z, v, phases=True)
            basis.enable_direct_tables(False)
            for p in range(len(b)):
                assert_elements(Ht[p].cpu().numpy(), nu.S_and_H_grid(prob, g, b[p], z[p], v[p])[1], "D^T (tables) on the non-uniform grid, position %d" % p)
        bt, vt, n_steps = np.array([1.6, 0.9]), np.array([1.0, 1.3]), 30
        basis.set_option("solve_route", 1)
        Cg = lib.propagate(basis, bt, vt, -6.0, 6.0, n_steps).cpu().numpy()
        h = 12.0 / n_steps
        for t in range(2):
            co = oprop.propagate(prob, bt[t], vt[t], -6.0, 6.0, n_steps, matrices=lambda i, t=t: nu.S_and_H_grid(prob, g, bt[t], -6.0 + 0.5 * i * h, vt[t]))
            assert np.abs(Cg[t] - co).max() < PTOL, (two, t, np.abs(Cg[t] - co).max())
        basis.close()
