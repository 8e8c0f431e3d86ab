"""The five BASELINE.json workloads (rule-literal sizes) and tiny test problems.

Nothing here is read from a dataset: the paper's own workload is p + H generated from first
principles, so these *are* the workload shapes.  SEED = 240304252.
"""
from __future__ import annotations

import numpy as np

from .basis import make_centre, make_problem, splitmix64_uniform, hydrogenic_bound_u, radial_grid, Centre

SEED = 240304252


def log_spaced(b_min: float, b_max: float, n: int) -> np.ndarray:
    """b_i = b_min (b_max/b_min)^(i/(n-1))."""
    if n == 1:
        return np.array([b_min])
    return b_min * (b_max / b_min) ** (np.arange(n) / (n - 1.0))


# name -> recipe.  Keys mirror BASELINE.json configs[i]; unstated values follow SURVEY.md amb. A7, A19.
CONFIGS = {
    0: dict(two_centre=False, Z_T=1.0, Z_P=1.0, l_max=2, n_max=3, bins=8, k_max=4.0, Nr=2000, h=0.05,
            lambda_max=4, v=[2.0], b=[0.5, 1.0, 2.0, 4.0], z_min=-50.0, z_max=50.0, n_steps=1000, perturb=False),
    1: dict(two_centre=True, Z_T=1.0, Z_P=1.0, l_max=2, n_max=3, bins=8, k_max=4.0, Nr=2000, h=0.05,
            lambda_max=4, v=[1.0], b=log_spaced(0.1, 10.0, 16), z_min=-40.0, z_max=40.0, n_steps=1600,
            perturb=True, quad=dict(n_rho=64, n_phi=16, n_z=128, rho_max=40.0, z_pad=40.0, phi_rule=0)),
    2: dict(two_centre=False, Z_T=1.0, Z_P=1.0, l_max=4, n_max=6, bins=20, k_max=6.0, Nr=8000, h=0.0125,
            lambda_max=8, v=[1.0, 2.0, 4.0], b=log_spaced(0.05, 15.0, 64), z_min=-100.0, z_max=100.0,
            n_steps=4000, perturb=False),
    3: dict(two_centre=True, Z_T=1.0, Z_P=2.0, l_max=3, n_max=4, bins=16, k_max=4.0, Nr=2000, h=0.05,
            lambda_max=6, v=[1.5], b=log_spaced(0.05, 12.0, 128), z_min=-60.0, z_max=60.0, n_steps=3000,
            perturb=False, quad=dict(n_rho=96, n_phi=24, n_z=192, rho_max=40.0, z_pad=40.0, phi_rule=0)),
    4: dict(two_centre=False, Z_T=1.0, Z_P=1.0, l_max=4, n_max=6, bins=20, k_max=6.0, Nr=8000, h=0.0125,
            lambda_max=8, v=log_spaced(0.632456, 6.32456, 12), b=log_spaced(0.05, 15.0, 96),
            z_min=-100.0, z_max=100.0, n_steps=4000, perturb=False),
}


def build_config(idx: int, bins: int | None = None, nk: int = 32, sub: int = 10):
    """Return (Problem, run) for BASELINE.json configs[idx].

    run = dict(b=[n_traj], v=[n_traj], vgroup=[n_traj], z_min, z_max, n_steps): trajectories are the
    outer product velocities x impact parameters (velocity-major).
    `bins` overrides the wave packets per l (label-matched secondary sizes, amb. A18).
    """
    c = CONFIGS[idx]
    nb = c["bins"] if bins is None else bins
    n_centres = 2 if c["two_centre"] else 1
    pert = [None] * n_centres
    if c["perturb"]:
        # draws ordered: centre T, P; l ascending; interior edge ascending
        n_edge = nb - 1
        draws = splitmix64_uniform(SEED, n_centres * (c["l_max"] + 1) * n_edge)
        draws = (2.0 * draws - 1.0) * 1e-3
        draws = draws.reshape(n_centres, c["l_max"] + 1, n_edge)
        pert = [draws[i] for i in range(n_centres)]
    Zs = [c["Z_T"], c["Z_P"]][:n_centres]
    centres = [make_centre(Z, c["l_max"], c["n_max"], nb, c["k_max"], c["Nr"], c["h"],
                           edge_perturb=pert[i], nk=nk, sub=sub) for i, Z in enumerate(Zs)]
    prob = make_problem(centres, c["Z_P"], c["Nr"], c["h"], c["lambda_max"], quad=c.get("quad"),
                        meta=dict(config=idx, bins=nb))
    vs = np.asarray(c["v"], float); bs = np.asarray(c["b"], float)
    run = dict(b=np.tile(bs, len(vs)), v=np.repeat(vs, len(bs)),
               vgroup=np.repeat(np.arange(len(vs), dtype=np.int32), len(bs)),
               z_min=c["z_min"], z_max=c["z_max"], n_steps=c["n_steps"])
    return prob, run


def bound_only_centre(Z: float, nl_list, Nr: int, h: float, renormalise: bool = False) -> Centre:
    """Centre made of analytic hydrogenic bound states only, in the given (n,l) order."""
    r, w = radial_grid(Nr, h)
    U = np.array([hydrogenic_bound_u(n, l, Z, r) for n, l in nl_list])
    if renormalise:
        U /= np.sqrt((w * U * U).sum(1))[:, None]
    return Centre(Z=float(Z), l=np.array([l for _, l in nl_list], np.int32),
                  eps=np.array([-Z * Z / (2.0 * n * n) for n, _ in nl_list]),
                  kind=np.zeros(len(nl_list), np.int32), nq=np.array([n for n, _ in nl_list], np.int32),
                  u=np.ascontiguousarray(U), g=np.zeros_like(U))


def tiny_problem(two_centre: bool, l_max: int = 1, n_max: int = 2, bins: int = 2, k_max: float = 2.0,
                 Nr: int = 400, h: float = 0.1, lambda_max: int | None = None, Z_T: float = 1.0,
                 Z_P: float = 1.0, quad: dict | None = None, seed: int | None = None):
    """Small problems for parity tests the oracle finishes in seconds."""
    n_centres = 2 if two_centre else 1
    pert = [None] * n_centres
    if seed is not None and bins > 1:
        d = (2.0 * splitmix64_uniform(seed, n_centres * (l_max + 1) * (bins - 1)) - 1.0) * 1e-3
        d = d.reshape(n_centres, l_max + 1, bins - 1)
        pert = [d[i] for i in range(n_centres)]
    Zs = [Z_T, Z_P][:n_centres]
    centres = [make_centre(Z, l_max, n_max, bins, k_max, Nr, h, edge_perturb=pert[i], nk=16, sub=4)
               for i, Z in enumerate(Zs)]
    if two_centre and quad is None:
        quad = dict(n_rho=24, n_phi=8, n_z=48, rho_max=30.0, z_pad=30.0, phi_rule=0)
    return make_problem(centres, Z_P, Nr, h, 2 * l_max if lambda_max is None else lambda_max, quad=quad,
                        meta=dict(config="tiny"))
