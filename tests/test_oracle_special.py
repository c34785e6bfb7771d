"""Pins for oracle/special.py and oracle/wigner.py: library routines (mpmath, sympy) at random
arguments, orthogonality relations, and closed forms (SURVEY.md 8(c) "what pins each part")."""
import math

import mpmath as mp
import numpy as np
import pytest

from oracle import special as sp
from oracle.wigner import wigner_3j


def test_spherical_bessel_vs_mpmath():
    rng = np.random.default_rng(0)
    for x in rng.uniform(0.3, 60.0, 12):
        for l in range(0, 13):
            j = mp.sqrt(mp.pi / (2 * x)) * mp.besselj(l + 0.5, x)
            y = mp.sqrt(mp.pi / (2 * x)) * mp.bessely(l + 0.5, x)
            h = sp.sph_h1(l, x)
            assert abs(h.real - float(j)) <= 1e-12 * max(1.0, abs(float(y)))
            assert abs(h.imag - float(y)) <= 1e-12 * abs(float(y))
            assert abs(sp.sph_jn(l, x) - float(j)) <= 1e-13 * max(abs(float(j)), 1e-3)


def test_radial_derivative_combination():
    # [x z_l(x)]'/x by central differences of x z_l(x)
    for l in (1, 2, 3, 5):
        for x in (0.7, 3.1, 11.0):
            h = 1e-5
            fd = ((x + h) * sp.sph_h1(l, x + h) - (x - h) * sp.sph_h1(l, x - h)) / (2 * h) / x
            assert abs(sp.sph_h1_rd(l, x) - fd) < 1e-8 * abs(fd)
            fdj = ((x + h) * sp.sph_jn(l, x + h) - (x - h) * sp.sph_jn(l, x - h)) / (2 * h) / x
            assert abs(sp.sph_jn_rd(l, x) - fdj) < 1e-8 * max(abs(fdj), 1e-3)


def test_pbar_vs_mpmath_no_condon_shortley():
    rng = np.random.default_rng(1)
    for x in rng.uniform(-0.99, 0.99, 8):
        for l in range(0, 8):
            for m in range(0, l + 1):
                # mpmath legenp(type=2) carries the Condon-Shortley factor (-1)^m: remove it (reading R2)
                ref = (-1) ** m * float(mp.legenp(l, m, x)) * math.sqrt(
                    (2 * l + 1) / 2.0 * math.factorial(l - m) / math.factorial(l + m))
                assert abs(float(sp.pbar(l, m, x)) - ref) < 1e-12 * max(1.0, abs(ref))


def test_pbar_orthonormal_and_positive_leading_sign():
    xg, wg = np.polynomial.legendre.leggauss(40)
    for m in range(0, 4):
        for l in range(m, 7):
            for l2 in range(m, 7):
                v = np.sum(wg * sp.pbar(l, m, xg) * sp.pbar(l2, m, xg))
                assert abs(v - (1.0 if l == l2 else 0.0)) < 1e-12
    # no CS phase: Pbar_m^m > 0 on (-1, 1)
    for m in range(0, 7):
        assert float(sp.pbar(m, m, 0.3)) > 0


def test_pi_tau_definitions():
    th = np.array([0.2, 0.9, 1.7, 2.8])
    h = 1e-6
    for l in range(1, 6):
        for m in range(0, l + 1):
            fd = (sp.pbar(l, m, np.cos(th + h)) - sp.pbar(l, m, np.cos(th - h))) / (2 * h)
            assert np.allclose(sp.taubar(l, m, th), fd, rtol=1e-7, atol=1e-8)
            if m >= 1:
                assert np.allclose(sp.pibar(l, m, th), sp.pbar(l, m, np.cos(th)) / np.sin(th), rtol=1e-12)
    # normal-incidence limit quoted in SURVEY.md 8(c) O6: pibar_l^1(0) = taubar_l^1(0) = 1/2 sqrt(l(l+1)(2l+1)/2)
    for l in range(1, 7):
        v = 0.5 * math.sqrt(l * (l + 1) * (2 * l + 1) / 2.0)
        assert abs(float(sp.pibar(l, 1, 0.0)) - v) < 1e-13
        assert abs(float(sp.taubar(l, 1, 0.0)) - v) < 1e-13


def test_wigner3j_vs_sympy_and_orthogonality():
    from sympy.physics.wigner import wigner_3j as w3
    rng = np.random.default_rng(2)
    n = 0
    for j1 in range(0, 7):
        for j2 in range(0, 7):
            for j3 in range(abs(j1 - j2), min(j1 + j2, 12) + 1):
                for _ in range(3):
                    m1 = int(rng.integers(-j1, j1 + 1))
                    m2 = int(rng.integers(-j2, j2 + 1))
                    m3 = -m1 - m2
                    ref = float(w3(j1, j2, j3, m1, m2, m3)) if abs(m3) <= j3 else 0.0
                    assert abs(wigner_3j(j1, j2, j3, m1, m2, m3) - ref) < 1e-14
                    n += 1
    assert n > 500
    # orthogonality: sum_{m1 m2} (2 j3 + 1) (j1 j2 j3; m1 m2 m3)(j1 j2 j3'; m1 m2 m3') = delta delta
    j1, j2 = 3, 2
    for j3 in range(1, 6):
        for j3p in range(1, 6):
            for m3 in range(-min(j3, j3p), min(j3, j3p) + 1):
                s = sum(wigner_3j(j1, j2, j3, a, b, m3) * wigner_3j(j1, j2, j3p, a, b, m3)
                        for a in range(-j1, j1 + 1) for b in range(-j2, j2 + 1) if a + b + m3 == 0)
                assert abs((2 * j3 + 1) * s - (1.0 if j3 == j3p else 0.0)) < 1e-13


def test_wigner3j_zero_m_closed_form():
    # (j1 j2 j3; 0 0 0) = (-1)^g sqrt((2g-2j1)!(2g-2j2)!(2g-2j3)!/(2g+1)!) g!/((g-j1)!(g-j2)!(g-j3)!), 2g = j1+j2+j3 even
    f = math.factorial
    for j1 in range(0, 7):
        for j2 in range(0, 7):
            for j3 in range(abs(j1 - j2), j1 + j2 + 1):
                J = j1 + j2 + j3
                if J % 2:
                    assert wigner_3j(j1, j2, j3, 0, 0, 0) == 0.0
                    continue
                g = J // 2
                ref = ((-1) ** g * math.sqrt(f(2 * g - 2 * j1) * f(2 * g - 2 * j2) * f(2 * g - 2 * j3) / f(2 * g + 1))
                       * f(g) / (f(g - j1) * f(g - j2) * f(g - j3)))
                assert abs(wigner_3j(j1, j2, j3, 0, 0, 0) - ref) < 1e-14
