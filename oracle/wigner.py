"""Wigner 3j symbols (TEST INFRASTRUCTURE ONLY - see oracle/__init__.py).

PAPER.md:327 (Eq. I19).  The oracle uses the Racah single-sum formula with exact integer
factorials (python ints / Fractions) and takes one square root at the end.  (The paper
cites a recursion, which neither side uses: the CUDA path's build-time generator
csrc/gen_tables.py has its own, separately typed Racah sum in binomial form with mpmath square
roots; nothing is shared or imported between the two.)
"""
from fractions import Fraction
from functools import lru_cache
from math import factorial as f
from math import sqrt


@lru_cache(maxsize=None)
def wigner_3j(j1, j2, j3, m1, m2, m3):
    if m1 + m2 + m3 != 0:
        return 0.0
    if j3 < abs(j1 - j2) or j3 > j1 + j2:
        return 0.0
    if abs(m1) > j1 or abs(m2) > j2 or abs(m3) > j3:
        return 0.0
    tri = Fraction(f(j1 + j2 - j3) * f(j1 - j2 + j3) * f(-j1 + j2 + j3), f(j1 + j2 + j3 + 1))
    pre = tri * f(j1 + m1) * f(j1 - m1) * f(j2 + m2) * f(j2 - m2) * f(j3 + m3) * f(j3 - m3)
    tmin = max(0, j2 - j3 - m1, j1 - j3 + m2)
    tmax = min(j1 + j2 - j3, j1 - m1, j2 + m2)
    s = Fraction(0)
    for t in range(tmin, tmax + 1):
        den = (f(t) * f(j3 - j2 + t + m1) * f(j3 - j1 + t - m2)
               * f(j1 + j2 - j3 - t) * f(j1 - t - m1) * f(j2 - t + m2))
        s += Fraction((-1) ** t, den)
    sign = (-1) ** (j1 - j2 - m3)
    # s * sqrt(pre): keep the sign of s, exact magnitude under one sqrt
    val = s * s * pre
    mag = sqrt(val.numerator) / sqrt(val.denominator) if val.denominator < 10 ** 300 else sqrt(float(val))
    return sign * (1 if s >= 0 else -1) * mag
