"""RK4 propagation along one straight-line trajectory: Algorithm 1 of the paper.

TEST INFRASTRUCTURE (see oracle/__init__.py).

    dX/dz = M X,   M = -(i/v) S^{-1} H     (eq. (2)-(4))
M is never formed; each RK4 stage solves S x = H c by Gaussian elimination with partial pivoting
(amb. A14: same result as the paper's ZGESV with N right-hand sides).
Uniform grid z_i = z_min + i (z_max - z_min)/n_steps (amb. A13).  4 n_z + 1 = 2 n_steps + 1 evaluations
of (S, H) per path: the evaluation at z_new is reused as the next step's z.
"""
import numpy as np

from .assemble import S_and_H


def gauss_solve(A: np.ndarray, y: np.ndarray) -> np.ndarray:
    """Solve A x = y by Gaussian elimination with partial pivoting (first maximal |pivot| wins ties),
    then back substitution.  Plain loops over columns; complex128."""
    A = np.array(A, dtype=np.complex128)
    x = np.array(y, dtype=np.complex128)
    n = A.shape[0]
    for j in range(n):
        p = j + int(np.argmax(np.abs(A[j:, j])))
        if A[p, j] == 0:
            raise ZeroDivisionError("singular matrix at column %d" % j)
        if p != j:
            A[[j, p]] = A[[p, j]]
            x[[j, p]] = x[[p, j]]
        for i in range(j + 1, n):
            f = A[i, j] / A[j, j]
            if f != 0:
                A[i, j:] -= f * A[j, j:]
                x[i] -= f * x[j]
    for i in range(n - 1, -1, -1):
        x[i] = (x[i] - np.dot(A[i, i + 1:], x[i + 1:])) / A[i, i]
    return x


def rhs(S: np.ndarray, H: np.ndarray, c: np.ndarray, v: float, one_centre: bool) -> np.ndarray:
    """f = -(i/v) S^{-1} H c  (eq. (4)); eq. (5) when there is no second centre."""
    y = H @ c
    x = y if one_centre else gauss_solve(S, y)
    return (-1j / v) * x


def propagate(prob, b: float, v: float, z_min: float, z_max: float, n_steps: int, init_state: int = 0,
              matrices=None, track_norm: bool = False, residual: bool = True):
    """Algorithm 1.  Returns the amplitudes c(z_max) [N_tot]; with track_norm also max |c^H S c - 1|.

    matrices: optional callable i -> (S, H) at half-step index i (z = z_min + i h/2), used by tests that
    precompute or substitute the matrices; default evaluates S_and_H."""
    one = len(prob.centres) == 1
    h = (z_max - z_min) / n_steps
    if matrices is None:
        def matrices(i):
            return S_and_H(prob, b, z_min + 0.5 * i * h, v, residual=residual)
    c = np.zeros(prob.n_tot, dtype=np.complex128)      # lines 1-2: X[:] = 0, X[1] = 1
    c[init_state] = 1.0
    S_new, H_new = matrices(0)                          # lines 3-4
    drift = 0.0
    for i in range(n_steps):
        S_z, H_z = S_new, H_new                          # line 12
        S_mid, H_mid = matrices(2 * i + 1)               # lines 13-15
        S_new, H_new = matrices(2 * i + 2)
        k1 = rhs(S_z, H_z, c, v, one)                    # line 16
        k2 = rhs(S_mid, H_mid, c + 0.5 * h * k1, v, one)  # line 17
        k3 = rhs(S_mid, H_mid, c + 0.5 * h * k2, v, one)  # line 18
        k4 = rhs(S_new, H_new, c + h * k3, v, one)        # line 19
        c = c + (h / 6.0) * (k1 + 2.0 * k2 + 2.0 * k3 + k4)   # line 20
        if track_norm:
            drift = max(drift, abs(np.vdot(c, S_new @ c).real - 1.0))
    return (c, drift) if track_norm else c
