"""Transition probabilities and cross sections from the final amplitudes X(z_max).

TEST INFRASTRUCTURE (see oracle/__init__.py).

    P_j      = |c_j(z_max)|^2
    P_nl     = sum over m of P_j for one radial function
    classes  = [elastic (init radial fn), target excitation (bound), target continuum (wave packets),
                capture bound, capture continuum]
    sigma    = 2 pi Int b P(b) db, trapezoid rule in the variable ln b over the given b-set
               (db = b dln b; no extrapolation to 0 or infinity), units a0^2
"""
import numpy as np


def state_radial_index(prob) -> np.ndarray:
    """Global radial-function index of every state (centre T radial functions first, then P)."""
    out, off = [], 0
    for c in prob.centres:
        out += [off + ir for (ir, _, _) in c.states()]
        off += c.n_rad
    return np.array(out, dtype=np.int64)


def probabilities(prob, C: np.ndarray, init_state: int = 0):
    """C [n_traj, N_tot] complex -> (P_state [n_traj,N_tot], P_nl [n_traj,n_rad_tot], P_class [n_traj,5])."""
    C = np.atleast_2d(C)
    P_state = C.real ** 2 + C.imag ** 2
    ridx = state_radial_index(prob)
    n_rad_tot = sum(c.n_rad for c in prob.centres)
    P_nl = np.zeros((C.shape[0], n_rad_tot))
    for j, r in enumerate(ridx):
        P_nl[:, r] += P_state[:, j]
    kinds = np.concatenate([c.kind for c in prob.centres])
    centre_of = np.concatenate([np.full(c.n_rad, ic) for ic, c in enumerate(prob.centres)])
    r_init = ridx[init_state]
    P_class = np.zeros((C.shape[0], 5))
    for r in range(n_rad_tot):
        if r == r_init:
            k = 0
        elif centre_of[r] == 0:
            k = 1 if kinds[r] == 0 else 2
        else:
            k = 3 if kinds[r] == 0 else 4
        P_class[:, k] += P_nl[:, r]
    return P_state, P_nl, P_class


def cross_sections(b: np.ndarray, vgroup: np.ndarray, P: np.ndarray, n_vgroups: int) -> np.ndarray:
    """sigma[g, :] = 2 pi sum over consecutive b in group g of the trapezoid rule in ln b of b^2 P(b)."""
    b = np.asarray(b, float)
    P = np.atleast_2d(P)
    out = np.zeros((n_vgroups, P.shape[1]))
    for g in range(n_vgroups):
        idx = np.where(np.asarray(vgroup) == g)[0]
        idx = idx[np.argsort(b[idx], kind="stable")]
        for i0, i1 in zip(idx[:-1], idx[1:]):
            dl = np.log(b[i1]) - np.log(b[i0])
            out[g] += 2.0 * np.pi * 0.5 * dl * (b[i0] ** 2 * P[i0] + b[i1] ** 2 * P[i1])
    return out
