"""Angular-momentum algebra used by eq. (6) and eq. (8)-(9) of the paper.

TEST INFRASTRUCTURE (see oracle/__init__.py).  All functions are the textbook definitions
written out; nothing is tabulated or cached.

Conventions: Condon-Shortley phase everywhere;
  P_l^m(x) = (-1)^m (1-x^2)^{m/2} d^m/dx^m P_l(x),  P_l^{-m} = (-1)^m (l-m)!/(l+m)! P_l^m
  Theta~_{lq}(c) = sqrt[(2l+1)/2 (l-q)!/(l+q)!] P_l^q(c)   (so Y_lq = Theta~_lq e^{iq phi}/sqrt(2 pi))
  d^j_{m'm}(beta) = <j m'| exp(-i beta J_y) |j m>   (Wigner's sum formula)
"""
import math

import numpy as np


def fact(n: int) -> int:
    if n < 0:
        raise ValueError("factorial of negative integer")
    return math.factorial(n)


def clebsch_gordan(j1: int, m1: int, j2: int, m2: int, j: int, m: int) -> float:
    """<j1 m1; j2 m2 | j m> for integer angular momenta, Racah's closed formula.

    The paper writes C^{l' m'}_{lambda mu l m} = <lambda mu; l m | l' m'> (eq. (6)).
    """
    if m1 + m2 != m or j < abs(j1 - j2) or j > j1 + j2:
        return 0.0
    if abs(m1) > j1 or abs(m2) > j2 or abs(m) > j:
        return 0.0
    pref = (2 * j + 1) * fact(j + j1 - j2) * fact(j - j1 + j2) * fact(j1 + j2 - j) / fact(j1 + j2 + j + 1)
    pref *= fact(j + m) * fact(j - m) * fact(j1 - m1) * fact(j1 + m1) * fact(j2 - m2) * fact(j2 + m2)
    s = 0.0
    for k in range(0, j1 + j2 - j + 1):
        d = [k, j1 + j2 - j - k, j1 - m1 - k, j2 + m2 - k, j - j2 + m1 + k, j - j1 - m2 + k]
        if min(d) < 0:
            continue
        den = 1
        for x in d:
            den *= fact(x)
        s += (-1) ** k / den
    return math.sqrt(pref) * s


def assoc_legendre(l: int, m: int, x):
    """Associated Legendre function P_l^m(x), Condon-Shortley phase, any integer |m| <= l.

    "P_lambda^mu are Legendre polynomials" in eq. (6) = these functions (amb. A3).
    Upward recurrence in l from P_m^m = (-1)^m (2m-1)!! (1-x^2)^{m/2}.
    """
    x = np.asarray(x, dtype=np.float64)
    am = abs(m)
    if am > l:
        return np.zeros_like(x)
    s = np.sqrt(np.maximum(0.0, 1.0 - x * x))
    pmm = np.ones_like(x)
    for i in range(1, am + 1):
        pmm = -pmm * (2 * i - 1) * s
    if l == am:
        p = pmm
    else:
        pm1 = x * (2 * am + 1) * pmm
        if l == am + 1:
            p = pm1
        else:
            p0, p1 = pmm, pm1
            for ll in range(am + 2, l + 1):
                p0, p1 = p1, ((2 * ll - 1) * x * p1 - (ll + am - 1) * p0) / (ll - am)
            p = p1
    if m < 0:
        p = (-1) ** am * fact(l - am) / fact(l + am) * p
    return p


def theta_tilde(l: int, q: int, c):
    """Normalised polar function: Y_lq(theta,phi) = Theta~_lq(cos theta) e^{i q phi} / sqrt(2 pi)."""
    aq = abs(q)
    t = math.sqrt((2 * l + 1) / 2.0 * fact(l - aq) / fact(l + aq)) * assoc_legendre(l, aq, c)
    return t if q >= 0 else (-1) ** aq * t


def sph_harm(l: int, m: int, cos_theta, phi):
    """Complex spherical harmonic Y_lm with Condon-Shortley phase."""
    return theta_tilde(l, m, cos_theta) * np.exp(1j * m * np.asarray(phi)) / math.sqrt(2.0 * math.pi)


def wigner_small_d(j: int, mp: int, m: int, beta: float) -> float:
    """d^j_{m'm}(beta) = <j m'|exp(-i beta J_y)|j m>, Wigner's sum formula (eq. (8))."""
    tot = 0.0
    cb, sb = math.cos(beta / 2.0), math.sin(beta / 2.0)
    for k in range(max(0, m - mp), min(j + m, j - mp) + 1):
        num = math.sqrt(fact(j + m) * fact(j - m) * fact(j + mp) * fact(j - mp))
        den = fact(j + m - k) * fact(k) * fact(j - k - mp) * fact(k - m + mp)
        tot += (-1) ** (k - m + mp) * num / den * cb ** (2 * j - 2 * k + m - mp) * sb ** (2 * k - m + mp)
    return tot


def direct_angular_coefficient(lp: int, mp: int, l: int, m: int, lam: int) -> float:
    """G^lambda_{alpha' alpha} of eq. (6) with the factorials restored (amb. A3):

        sqrt[(2l+1)(lambda-mu)! / ((2l'+1)(lambda+mu)!)] <lambda 0; l 0|l' 0> <lambda mu; l m|l' m'>,  mu = m'-m.
    """
    mu = mp - m
    if abs(mu) > lam or lam < abs(lp - l) or lam > lp + l or (lp + l + lam) % 2:
        return 0.0
    return (math.sqrt((2 * l + 1) * fact(lam - mu) / ((2 * lp + 1) * fact(lam + mu)))
            * clebsch_gordan(lam, 0, l, 0, lp, 0) * clebsch_gordan(lam, mu, l, m, lp, mp))
