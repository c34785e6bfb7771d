"""Oracle special functions (TEST INFRASTRUCTURE ONLY - see oracle/__init__.py).

PAPER.md:215-221 (Eq. I3): scalar wavefunctions use the spherical Hankel function of the
first kind h_l^(1), the spherical Bessel function j_l and the "normalized associated
legendre polynomial" P_l^{|m|}.  Reading R2: the normalisation is
    Pbar_l^m(x) = sqrt((2l+1)/2 * (l-m)!/(l+m)!) * (1-x^2)^{m/2} d^m P_l(x)/dx^m ,  m >= 0,
with NO Condon-Shortley phase (Doicu et al., appendix B convention).
Angular functions of PAPER.md:430-432 (Eq. II7):
    pibar_l^m(theta)  = Pbar_l^m(cos theta) / sin theta
    taubar_l^m(theta) = d Pbar_l^m(cos theta) / d theta
Library primitives used as steps: scipy spherical_jn / spherical_yn, numpy Legendre series.
"""
from math import factorial, sqrt

import numpy as np
from numpy.polynomial import legendre as _leg
from scipy.special import spherical_jn, spherical_yn


def sph_jn(l, x):
    """j_l(x)."""
    return spherical_jn(l, x)


def sph_h1(l, x):
    """h_l^(1)(x) = j_l(x) + i y_l(x)."""
    return spherical_jn(l, x) + 1j * spherical_yn(l, x)


def sph_jn_rd(l, x):
    """[x j_l(x)]' / x  (radial factor of the p=1 VSWF, Eq. I6b)."""
    return spherical_jn(l, x) / x + spherical_jn(l, x, derivative=True)


def sph_h1_rd(l, x):
    """[x h_l^(1)(x)]' / x."""
    return sph_h1(l, x) / x + spherical_jn(l, x, derivative=True) + 1j * spherical_yn(l, x, derivative=True)


def sph_jn_d(l, x):
    """d j_l(x) / dx."""
    return spherical_jn(l, x, derivative=True)


def sph_h1_d(l, x):
    """d h_l^(1)(x) / dx."""
    return spherical_jn(l, x, derivative=True) + 1j * spherical_yn(l, x, derivative=True)


def _norm(l, m):
    return sqrt((2 * l + 1) / 2.0 * factorial(l - m) / factorial(l + m))


def _dm_legendre(l, m):
    """Legendre-series coefficients of d^m P_l / dx^m."""
    c = np.zeros(l + 1)
    c[l] = 1.0
    return _leg.legder(c, m) if m > 0 else c


def pbar(l, m, x):
    """Normalised associated Legendre function Pbar_l^m(x), m >= 0 (reading R2)."""
    assert 0 <= m
    x = np.asarray(x, dtype=float)
    if m > l:
        return np.zeros_like(x)
    q = _leg.legval(x, _dm_legendre(l, m))
    return _norm(l, m) * (1.0 - x * x) ** (m / 2.0) * q


def pibar(l, m, theta):
    """pibar_l^m(theta) = Pbar_l^m(cos theta)/sin theta for m >= 1 (regular at the poles);
    returns 0 for m = 0 (it is always multiplied by m, Eq. II7)."""
    theta = np.asarray(theta, dtype=float)
    if m == 0 or m > l:
        return np.zeros_like(theta)
    x, s = np.cos(theta), np.sin(theta)
    q = _leg.legval(x, _dm_legendre(l, m))
    return _norm(l, m) * s ** (m - 1) * q


def taubar(l, m, theta):
    """taubar_l^m(theta) = d/dtheta [ sin^m(theta) Q(cos theta) ] * norm,  Q = d^m P_l/dx^m."""
    theta = np.asarray(theta, dtype=float)
    if m > l:
        return np.zeros_like(theta)
    x, s = np.cos(theta), np.sin(theta)
    q = _leg.legval(x, _dm_legendre(l, m))
    dq = _leg.legval(x, _dm_legendre(l, m + 1)) if m + 1 <= l else np.zeros_like(x)
    first = m * s ** (m - 1) * x * q if m >= 1 else np.zeros_like(x)
    return _norm(l, m) * (first - s ** (m + 1) * dq)
