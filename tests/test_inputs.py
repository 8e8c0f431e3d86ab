"""Pins for the seeded input generators (wpccc_inputs): counts fixed by the paper, closed forms, residual tables."""
import math

import numpy as np
import pytest

from wpccc_inputs import (CONFIGS, build_config, coulomb_wave_table, hydrogenic_bound_u, make_centre, radial_grid,
                          splitmix64_uniform, log_spaced)


def test_state_count_rule_reproduces_paper_sizes():
    """1C N = 42 (l_max=0) .. 4257 (l_max=10); 2C N = 60 .. 1910 (l_max=5), all m kept."""
    count = lambda N0, lmax: sum((2 * l + 1) * (N0 - l) for l in range(lmax + 1))
    assert count(42, 0) == 42 and count(42, 10) == 4257
    assert 2 * count(30, 0) == 60 and 2 * count(30, 5) == 1910


def test_config_sizes_rule_literal():
    """per-centre N_rad / N = 30/86 (cfg 0,1), 120/580 (cfg 2,4), 74/286 (cfg 3)."""
    def sizes(c):
        nl = [(c["n_max"] - l) + c["bins"] for l in range(c["l_max"] + 1)]
        return sum(nl), sum((2 * l + 1) * n for l, n in enumerate(nl))
    assert sizes(CONFIGS[0]) == (30, 86) and sizes(CONFIGS[1]) == (30, 86)
    assert sizes(CONFIGS[2]) == (120, 580) and sizes(CONFIGS[4]) == (120, 580)
    assert sizes(CONFIGS[3]) == (74, 286)
    assert len(CONFIGS[4]["v"]) * len(CONFIGS[4]["b"]) == 1152


def test_splitmix64_reference_values():
    """SplitMix64 with seed 0: first outputs 0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4 (published test vector)."""
    u = splitmix64_uniform(0, 2)
    assert u[0] == (0xE220A8397B1DCDAF >> 11) / 2.0**53
    assert u[1] == (0x6E789E6AA1B965F4 >> 11) / 2.0**53


def test_hydrogenic_bound_states_orthonormal_and_eigen():
    r, w = radial_grid(4000, 0.025)
    for Z in (1.0, 2.0):
        U = {(n, l): hydrogenic_bound_u(n, l, Z, r) for l in range(3) for n in range(l + 1, 5)}
        for (n, l), u in U.items():
            assert np.sum(w * u * u) == pytest.approx(1.0, abs=2e-6)
            for (n2, l2), u2 in U.items():
                if l2 == l and n2 != n:
                    assert abs(np.sum(w * u * u2)) < 2e-6
            # (H - eps) u = 0 by second differences
            h = r[1]
            k = slice(40, 1500)
            d2 = (u[41:1501] - 2 * u[40:1500] + u[39:1499]) / h**2
            res = -0.5 * d2 + (l * (l + 1) / (2 * r[k] ** 2) - Z / r[k] + Z * Z / (2 * n * n)) * u[k]
            assert np.abs(res).max() < 2e-3 * np.abs(u).max()


def test_coulomb_wave_Z0_l0_is_sine_and_packet_closed_form():
    """Z=0, l=0: phi_k = sqrt(2/pi) sin(kr); wave packet u = sqrt(2/(pi dk)) (cos k0 r - cos k1 r)/r."""
    Nr, h = 600, 0.05
    r, _ = radial_grid(Nr, h)
    ks = np.array([0.4, 1.3])
    tab = coulomb_wave_table(0, ks, 1e-300, Nr, h, sub=8)           # Numerov path with Z -> 0
    np.testing.assert_allclose(tab, math.sqrt(2 / math.pi) * np.sin(np.outer(ks, r)), atol=3e-5)
    C = make_centre(0.0, 0, 0, 2, 1.0, Nr, h, renormalise=False)
    for i, (k0, k1) in enumerate(((0.0, 0.5), (0.5, 1.0))):
        ref = math.sqrt(2 / (math.pi * (k1 - k0))) * (np.cos(k0 * r[1:]) - np.cos(k1 * r[1:])) / r[1:]
        np.testing.assert_allclose(C.u[i][1:], ref, atol=1e-12)
        assert C.eps[i] == pytest.approx((k0 * k0 + k0 * k1 + k1 * k1) / 6)


def test_coulomb_wave_vs_mpmath():
    import mpmath
    Nr, h, Z = 2000, 0.05, 1.0
    r, _ = radial_grid(Nr, h)
    for l, k in ((0, 0.7), (1, 1.9), (2, 3.1)):
        tab = coulomb_wave_table(l, np.array([k]), Z, Nr, h, sub=10)[0]
        for j in (20, 133, 400, 1999):
            ref = float(mpmath.coulombf(l, -Z / k, k * r[j])) * math.sqrt(2 / math.pi)
            assert tab[j] == pytest.approx(ref, abs=5e-5)


def test_wave_packet_residual_table():
    """g = (H_c - eps) u for a wave packet (amb. A5): finite-difference check; g = 0 for bound states; <u|g> ~ 0."""
    Nr, h = 1600, 0.025
    r, w = radial_grid(Nr, h)
    C = make_centre(1.0, 1, 2, 3, 2.0, Nr, h, nk=16, sub=8)
    for i in range(C.n_rad):
        u, g, l = C.u[i], C.g[i], int(C.l[i])
        if C.kind[i] == 0:
            assert np.abs(g).max() == 0.0
            continue
        k = slice(40, 1200)
        d2 = (u[41:1201] - 2 * u[40:1200] + u[39:1199]) / h**2
        res = -0.5 * d2 + (l * (l + 1) / (2 * r[k] ** 2) - 1.0 / r[k] - C.eps[i]) * u[k]
        assert np.abs(res - g[k]).max() < 3e-4
        assert abs(np.sum(w * u * g)) < 2e-2                       # small box (r_max=40): truncation of the packet
        assert np.sum(w * u * u) == pytest.approx(1.0, abs=1e-13)           # grid-renormalised (amb. A6)


def test_config1_edge_perturbation_is_seeded_and_small():
    from wpccc_inputs.configs import SEED
    d = (2 * splitmix64_uniform(SEED, 2 * 3 * 7) - 1) * 1e-3
    assert np.abs(d).max() <= 1e-3 and np.abs(d).max() > 5e-4
    np.testing.assert_allclose(log_spaced(0.1, 10.0, 16)[[0, 15]], [0.1, 10.0])
    assert log_spaced(0.1, 10, 16)[5] == pytest.approx(0.1 * 100 ** (5 / 15))


@pytest.mark.timeout(300)
def test_build_config0_shapes():
    prob, run = build_config(0)
    C = prob.centres[0]
    assert C.n_rad == 30 and C.n_states == 86 and C.u.shape == (30, 2001) and prob.n_tot == 86
    assert list(C.l[:11]) == [0] * 11 and C.kind[:3].tolist() == [0, 0, 0] and C.kind[3] == 1
    assert len(run["b"]) == 4 and run["n_steps"] == 1000 and np.all(run["v"] == 2.0)
    r, w = radial_grid(prob.Nr, prob.h)
    G = (C.u * w) @ C.u.T
    np.testing.assert_allclose(np.diag(G), 1.0, atol=1e-13)
    same_l = C.l[:, None] == C.l[None, :]
    assert np.abs((G - np.eye(30))[same_l]).max() < 2e-2                      # <= 7.6e-3
