"""Assembly of the overlap matrix S and the coupling matrix H at one projectile position
(eq. (1), in the Galerkin reading, amb. A1; interaction picture, amb. A2).

TEST INFRASTRUCTURE (see oracle/__init__.py).

    S = [[I, S_PT^dagger], [S_PT, I]]          (same-centre blocks are I by fiat, amb. A6)
    H = [[D^T, H_TP], [H_PT, D^P]]            (H_TP and H_PT computed independently, amb. A1)
every element multiplied by e^{i (eps_row - eps_col) z / v}.  State order: centre T then P; inside a
centre radial functions in caller order, each expanded to m = -l..l ascending.
One centre (eq. (5)): S = I, H = D^T.
"""
import math

import numpy as np

from .direct import direct_block
from .transfer import two_centre_blocks


def state_energies(prob) -> np.ndarray:
    """eps of every state in the binding order."""
    return np.concatenate([[c.eps[ir] for (ir, _, _) in c.states()] for c in prob.centres])


def time_phase_matrix(prob, z: float, v: float) -> np.ndarray:
    e = state_energies(prob)
    return np.exp(1j * (e[:, None] - e[None, :]) * z / v)


def S_and_H(prob, b: float, z: float, v: float, time_phase: bool = True, residual: bool = True):
    """(S, H) at the position R = (b, 0, z), both [N_tot, N_tot] complex128."""
    T = prob.centres[0]
    NT = T.n_states
    DT = direct_block(T, prob.w, prob.h * np.arange(prob.Nr + 1), prob.lambda_max, b, z, v,
                      charge=prob.Z_proj, projectile_centre=False, time_phase=False)
    if len(prob.centres) == 1:
        S = np.eye(NT, dtype=np.complex128)
        H = DT.astype(np.complex128)
    else:
        P = prob.centres[1]
        NP = P.n_states
        DP = direct_block(P, prob.w, prob.h * np.arange(prob.Nr + 1), prob.lambda_max, b, z, v,
                          charge=T.Z, projectile_centre=True, time_phase=False)
        if residual:
            S_PT, H_PT, H_TP = two_centre_blocks(prob, b, z, v)
        else:
            import copy
            p2 = copy.copy(prob)
            p2.centres = [copy.copy(c) for c in prob.centres]
            for c in p2.centres:
                c.g = np.zeros_like(c.g)
            S_PT, H_PT, H_TP = two_centre_blocks(p2, b, z, v)
        N = NT + NP
        S = np.eye(N, dtype=np.complex128)
        S[NT:, :NT] = S_PT
        S[:NT, NT:] = S_PT.conj().T
        H = np.zeros((N, N), dtype=np.complex128)
        H[:NT, :NT] = DT
        H[NT:, NT:] = DP
        H[NT:, :NT] = H_PT
        H[:NT, NT:] = H_TP
    if time_phase:
        ph = time_phase_matrix(prob, z, v)
        S = S * ph
        H = H * ph
    return S, H
