"""-m gpu, collected last: wpccc_cross_sections_static (include/wpccc.h) -- the cross-section integral of P:L106 with its
index scratch in the library's file-scope static device array, for callers that may not allocate device memory --
against the existing path (sigma_nl / sigma_class of wpccc_probabilities, whose scratch is the basis arena).
Two calls in a row on different sizes (the second smaller than the first, so stale contents of the shared array would
show), the limits, and that the call leaves the device allocator untouched.  Passes alone in a fresh process and after
the rest of the suite (it stages its own small basis and releases the shared workspace first)."""
import numpy as np
import pytest

from wpccc_inputs import tiny_problem

RTOL, ATOL = 1e-11, 1e-13          # the element tolerance of the parity tests; the arithmetic is the same, so ~0 is expected


def _case(lib, basis, n_traj, n_vgroups, seed):
    import torch
    rng = np.random.default_rng(seed)
    N = basis.n_tot
    Cc = rng.normal(size=(n_traj, N)) + 1j * rng.normal(size=(n_traj, N))
    Cc /= np.linalg.norm(Cc, axis=1)[:, None]
    b = np.exp(rng.uniform(np.log(0.05), np.log(30.0), n_traj))          # unsorted on purpose
    vg = rng.integers(0, n_vgroups, n_traj).astype(np.int32)
    dC = torch.from_numpy(Cc).cuda()
    ref = lib.probabilities(basis, dC, b=b, vgroup=vg, n_vgroups=n_vgroups, init_state=0)
    return b, vg, ref


@pytest.mark.gpu
def test_static_scratch_cross_sections_match_the_arena_path_twice(lib):
    import torch
    lib.release_workspace()
    prob = tiny_problem(True, l_max=2, n_max=3, bins=2, k_max=1.5, Nr=400, h=0.1, Z_P=2.0, seed=11)
    basis = lib.setup_basis(prob)
    worst = 0.0
    # untimed first touch: with lazy module loading the first launch loads the kernel's module (and with it the static array)
    lib.cross_sections_static(torch.ones((2, 1), dtype=torch.float64, device="cuda"), np.array([1.0, 2.0]), np.zeros(2, np.int32), 1)
    # first call large, second small: the array still holds the first call's b / order / offsets beyond the second's ranges
    for n_traj, n_vg, seed in ((1500, 7, 1), (37, 3, 2)):
        b, vg, ref = _case(lib, basis, n_traj, n_vg, seed)
        out_nl = torch.empty_like(ref["sigma_nl"]); out_cl = torch.empty_like(ref["sigma_class"])
        torch.cuda.synchronize()
        before = (torch.cuda.memory_allocated(), torch.cuda.memory_reserved(), torch.cuda.mem_get_info()[0])
        lib.cross_sections_static_into(ref["P_nl"], b, vg, n_vg, out_nl)
        lib.cross_sections_static_into(ref["P_class"], b, vg, n_vg, out_cl)
        torch.cuda.synchronize()
        after = (torch.cuda.memory_allocated(), torch.cuda.memory_reserved(), torch.cuda.mem_get_info()[0])
        assert after[:2] == before[:2] and after[2] >= before[2], "device memory moved during the call: %r -> %r" % (before, after)
        for got, want in ((out_nl, ref["sigma_nl"]), (out_cl, ref["sigma_class"])):
            g, w = got.cpu().numpy(), want.cpu().numpy()
            assert np.isfinite(g).all() and np.abs(w).max() > 0
            err = np.abs(g - w)
            worst = max(worst, float(err.max()))
            assert (err <= ATOL + RTOL * np.abs(w)).all(), (n_traj, float(err.max()))
        # a closed form through the new entry point alone: P = 1 for one velocity group gives pi (b_max^2 - b_min^2) up to the
        # trapezoid error of b^2 in ln b; with P = 1 / b^2 the rule is exact: 2 pi ln(b_max / b_min)
        one = np.zeros(n_traj, np.int32)
        Pinv = torch.from_numpy((1.0 / b**2)[:, None].copy()).cuda()
        s = lib.cross_sections_static(Pinv, b, one, 1).cpu().numpy()
        assert s.shape == (1, 1) and abs(s[0, 0] - 2 * np.pi * np.log(b.max() / b.min())) < 1e-12 * abs(s[0, 0]) + 1e-12
    print("static-scratch cross sections: max |sigma_static - sigma_arena| = %.3e over two calls in a row" % worst)
    del basis
    lib.release_workspace()


@pytest.mark.gpu
def test_static_scratch_limits_are_reported(lib):
    import torch
    n = lib.STATIC_MAX_TRAJ
    b = np.linspace(0.1, 20.0, n + 1)
    P = torch.ones((n + 1, 3), dtype=torch.float64, device="cuda")
    with pytest.raises(lib.WpcccError) as e:
        lib.cross_sections_static(P, b, np.zeros(n + 1, np.int32), 1)
    assert "%d" % n in str(e.value) and "static scratch" in str(e.value)
    with pytest.raises(lib.WpcccError) as e:
        lib.cross_sections_static(P[:8], b[:8], np.zeros(8, np.int32), lib.STATIC_MAX_VGROUPS + 1)
    assert "velocity groups" in str(e.value)
    with pytest.raises(lib.WpcccError):
        lib.cross_sections_static(P[:8], np.r_[0.0, b[:7]], np.zeros(8, np.int32), 1)          # b = 0 has no place on a ln b grid
    # the largest size the array holds, all groups in use
    vg = (np.arange(n) % lib.STATIC_MAX_VGROUPS).astype(np.int32)
    s = lib.cross_sections_static(P[:n], b[:n], vg, lib.STATIC_MAX_VGROUPS).cpu().numpy()
    ref = np.zeros(lib.STATIC_MAX_VGROUPS)
    for g in range(lib.STATIC_MAX_VGROUPS):
        bg = b[:n][vg == g]
        ref[g] = np.sum(np.pi * np.diff(np.log(bg)) * (bg[:-1] ** 2 + bg[1:] ** 2))
    assert np.abs(s[:, 0] - ref).max() < 1e-10 * np.abs(ref).max()
    assert np.array_equal(s[:, 0], s[:, 2])
