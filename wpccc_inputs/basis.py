"""Radial basis generator: hydrogenic bound states + Coulomb wave-packet pseudostates.

What the paper fixes ("bound eigenstates and wave-packet pseudostates";
L148, r-grid "from 0 to 100 atomic units", radial functions "precomputed and stored").
BASELINE.json configs fix the recipe: bound n <= n_max, `bins` wave packets per l built
from Coulomb waves binned uniformly in k in [0, k_max].  Everything here is *input
generation*; none of the method's couplings/propagation lives here.

Conventions (amb. A5-A8):
  * reduced radial functions u(r) = r f(r) on the uniform grid r_k = k h, k = 0..Nr, u(0) = 0
  * trapezoid weights w_k = h (k < Nr), w_Nr = h/2, w_0 = 0
  * wave packet  u_i = dk^-1/2 Int_bin phi_kl dk  (32-point Gauss-Legendre in k per bin),
    phi_kl energy-normalised in k: phi -> sqrt(2/pi) sin(kr + ...)
  * residual table g_i = (H_c - eps_i) u_i = dk^-1/2 Int_bin (k^2/2 - eps_i) phi_kl dk,
    eps_i = (k0^2 + k0 k1 + k1^2)/6; g = 0 for bound eigenstates
  * every u (and its g) is divided by its grid norm sqrt(sum w u^2)
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

MASK64 = (1 << 64) - 1


def splitmix64_uniform(seed: int, n: int) -> np.ndarray:
    """n doubles in [0,1) from SplitMix64 (53 high bits), counter-based on `seed`."""
    out = np.empty(n)
    x = seed & MASK64
    for i in range(n):
        x = (x + 0x9E3779B97F4A7C15) & MASK64
        z = x
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK64
        z = z ^ (z >> 31)
        out[i] = (z >> 11) * (1.0 / (1 << 53))
    return out


def radial_grid(Nr: int, h: float):
    """r_k = k h (k = 0..Nr) and trapezoid weights (amb. A7, A8)."""
    r = h * np.arange(Nr + 1, dtype=np.float64)
    w = np.full(Nr + 1, h)
    w[0] = 0.0
    w[Nr] = 0.5 * h
    return r, w


def _genlaguerre(n: int, alpha: int, x: np.ndarray) -> np.ndarray:
    """Generalised Laguerre L_n^alpha(x) by the three-term recurrence."""
    L0 = np.ones_like(x)
    if n == 0:
        return L0
    L1 = 1.0 + alpha - x
    for k in range(1, n):
        L0, L1 = L1, ((2 * k + 1 + alpha - x) * L1 - (k + alpha) * L0) / (k + 1)
    return L1


def hydrogenic_bound_u(n: int, l: int, Z: float, r: np.ndarray) -> np.ndarray:
    """Reduced hydrogen-like radial function u_nl(r) = r R_nl(r), normalised on [0, inf)."""
    rho = 2.0 * Z * r / n
    N = math.sqrt((2.0 * Z / n) ** 3 * math.factorial(n - l - 1) / (2.0 * n * math.factorial(n + l)))
    return r * N * np.exp(-0.5 * rho) * rho ** l * _genlaguerre(n - l - 1, 2 * l + 1, rho)


def coulomb_wave_table(l: int, ks: np.ndarray, Z: float, Nr: int, h: float, sub: int = 10,
                       r_norm_factor: float = 2.0) -> np.ndarray:
    """Regular Coulomb continuum functions phi_kl(r_j) on the coarse grid, shape [len(ks), Nr+1].

    Numerov integration of u'' = [l(l+1)/r^2 - 2Z/r - k^2] u on a grid `sub` times finer
    than h, carried out to r_norm_factor * r_max, where the WKB amplitude
    A^2 = (kappa/k) u^2 + u'^2 / (k kappa) fixes the normalisation phi -> sqrt(2/pi) sin(.).
    Vectorised over k.
    """
    ks = np.asarray(ks, dtype=np.float64)
    hf = h / sub
    Nf = int(round(Nr * sub * r_norm_factor))
    k2 = ks * ks

    def gfun(rr):
        return l * (l + 1) / (rr * rr) - 2.0 * Z / rr - k2

    out = np.zeros((len(ks), Nr + 1))
    r1, r2 = hf, 2 * hf
    # series start u ~ r^(l+1) (1 - Z r/(l+1) + ...)
    def start(rr):
        a1 = -Z / (l + 1.0)
        a2 = (-(k2) / 2.0 - Z * a1) / (2.0 * l + 3.0)  # from the radial equation
        return rr ** (l + 1) * (1.0 + a1 * rr + a2 * rr * rr)
    u_prev = start(r1) * np.ones_like(ks)
    u_cur = start(r2) * np.ones_like(ks)
    f_prev = 1.0 - hf * hf * gfun(r1) / 12.0
    f_cur = 1.0 - hf * hf * gfun(r2) / 12.0
    scale = np.zeros_like(ks)  # log-scale bookkeeping to avoid overflow
    if sub == 1:
        out[:, 1] = u_prev
    if 2 % sub == 0 and 2 // sub <= Nr:
        out[:, 2 // sub] = u_cur
    u_last = u_nm2 = None
    for i in range(3, Nf + 1):
        rr = i * hf
        f_next = 1.0 - hf * hf * gfun(rr) / 12.0
        u_next = ((12.0 - 10.0 * f_cur) * u_cur - f_prev * u_prev) / f_next
        u_prev, u_cur = u_cur, u_next
        f_prev, f_cur = f_cur, f_next
        if i % sub == 0:
            j = i // sub
            if j <= Nr:
                out[:, j] = u_cur
        if i % 4096 == 0:
            big = np.abs(u_cur) > 1e150
            if big.any():
                s = np.where(big, 1e-150, 1.0)
                u_prev = u_prev * s
                u_cur = u_cur * s
                out *= s[:, None]
        if i == Nf - 2:
            u_nm2 = u_cur.copy()
        if i == Nf - 1:
            u_last = u_cur.copy()
    # centred derivative at i = Nf-1
    rN = (Nf - 1) * hf
    up = (u_cur - u_nm2) / (2.0 * hf)
    kap = np.sqrt(k2 + 2.0 * Z / rN - l * (l + 1) / (rN * rN))
    A2 = (kap / ks) * u_last ** 2 + up ** 2 / (ks * kap)
    out *= (math.sqrt(2.0 / math.pi) / np.sqrt(A2))[:, None]
    return out


@dataclass
class Centre:
    """One expansion centre: charge and radial tables (see include/wpccc.h wpccc_centre)."""
    Z: float
    l: np.ndarray       # [n_rad] int32
    eps: np.ndarray     # [n_rad] float64 energies (a.u.)
    kind: np.ndarray    # [n_rad] int32: 0 bound, 1 wave packet
    nq: np.ndarray      # [n_rad] int32: principal q.n. or bin index (labels only)
    u: np.ndarray       # [n_rad][Nr+1]
    g: np.ndarray       # [n_rad][Nr+1]

    @property
    def n_rad(self) -> int:
        return len(self.l)

    @property
    def n_states(self) -> int:
        return int(np.sum(2 * self.l + 1))

    def states(self):
        """[(irad, l, m)] in the binding order: radial functions in order, m = -l..l ascending."""
        return [(ir, int(l), m) for ir, l in enumerate(self.l) for m in range(-int(l), int(l) + 1)]


@dataclass
class Problem:
    """Full static problem description handed to both oracle and CUDA library."""
    centres: list           # [Centre] (T[, P])
    Z_proj: float           # charge seen by target-centred states
    Nr: int
    h: float
    w: np.ndarray           # [Nr+1]
    lambda_max: int
    quad: dict | None = None   # n_rho, n_phi, n_z, rho_max, z_pad, phi_rule
    meta: dict = field(default_factory=dict)

    @property
    def n_tot(self) -> int:
        return sum(c.n_states for c in self.centres)


def gauss_legendre_k(n: int):
    x, w = np.polynomial.legendre.leggauss(n)
    return x, w


def make_centre(Z: float, l_max: int, n_max: int, bins: int, k_max: float, Nr: int, h: float,
                edge_perturb: np.ndarray | None = None, nk: int = 32, sub: int = 10,
                renormalise: bool = True) -> Centre:
    """Bound n<=n_max (n>l) then `bins` wave packets per l, l ascending (binding order).

    edge_perturb: optional [l_max+1][bins-1] additive shifts of the interior bin edges
    (BASELINE.json configs[1]: "seeded random +-1e-3 perturbation of the bin edges").
    """
    r, w = radial_grid(Nr, h)
    xg, wg = gauss_legendre_k(nk)
    ls, eps, kind, nq, us, gs = [], [], [], [], [], []
    for l in range(l_max + 1):
        for n in range(l + 1, n_max + 1):
            ls.append(l); eps.append(-Z * Z / (2.0 * n * n)); kind.append(0); nq.append(n)
            us.append(hydrogenic_bound_u(n, l, Z, r)); gs.append(np.zeros(Nr + 1))
        if bins > 0:
            edges = np.linspace(0.0, k_max, bins + 1)
            if edge_perturb is not None:
                edges[1:-1] += edge_perturb[l]
            kall, wall = [], []
            for i in range(bins):
                a, c = edges[i], edges[i + 1]
                kall.append(0.5 * (c - a) * xg + 0.5 * (c + a)); wall.append(0.5 * (c - a) * wg)
            kall = np.concatenate(kall); wall = np.concatenate(wall)
            if Z == 0.0 and l == 0:
                phi = math.sqrt(2.0 / math.pi) * np.sin(np.outer(kall, r))
            else:
                phi = coulomb_wave_table(l, kall, Z, Nr, h, sub=sub)
            for i in range(bins):
                a, c = edges[i], edges[i + 1]
                sl = slice(i * nk, (i + 1) * nk)
                e_i = (a * a + a * c + c * c) / 6.0
                u = (wall[sl, None] * phi[sl]).sum(0) / math.sqrt(c - a)
                g = (wall[sl, None] * (0.5 * kall[sl, None] ** 2 - e_i) * phi[sl]).sum(0) / math.sqrt(c - a)
                ls.append(l); eps.append(e_i); kind.append(1); nq.append(i)
                us.append(u); gs.append(g)
    U = np.array(us); G = np.array(gs)
    U[:, 0] = 0.0; G[:, 0] = 0.0
    if renormalise:
        nrm = np.sqrt((w[None, :] * U * U).sum(1))
        U /= nrm[:, None]; G /= nrm[:, None]
    return Centre(Z=float(Z), l=np.array(ls, np.int32), eps=np.array(eps), kind=np.array(kind, np.int32),
                  nq=np.array(nq, np.int32), u=np.ascontiguousarray(U), g=np.ascontiguousarray(G))


def make_problem(centres, Z_proj, Nr, h, lambda_max, quad=None, meta=None) -> Problem:
    _, w = radial_grid(Nr, h)
    return Problem(centres=list(centres), Z_proj=float(Z_proj), Nr=Nr, h=h, w=w, lambda_max=lambda_max,
                   quad=quad, meta=meta or {})
