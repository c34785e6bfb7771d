"""T-matrix look-up table: interpolation in a geometry parameter (TEST INFRASTRUCTURE ONLY - see oracle/__init__.py).

PAPER.md:560: "in our implementation, we are setting up a lookup table for the transition matrices and interpolating between
them, this derivative [dGamma_k^{-1}/dp_i] can be numerically approximated using the same lookup table"; PAPER.md:59 (Fig. 2c,
"computing the Look-Up Tables").  The paper states neither the order of the interpolation nor the node set.
Reading R20: entry by entry, the CUBIC LAGRANGE polynomial through the four table nodes nearest to the interval that
holds p,
        T(p) = sum_{a=0..3} w_a(p) T_tab[i0 + a],      w_a(p) = prod_{b != a} (p - x_b) / (x_a - x_b),     x_a = p_tab[i0 + a],
with  i0 = clamp(i - 1, 0, n_tab - 4)  for  p_tab[i] <= p < p_tab[i+1]  (the last interval is closed on the right), nodes
strictly increasing and not necessarily equidistant; the derivative is the exact derivative of that piece,
        dT/dp = sum_a w'_a(p) T_tab[i0 + a],   w'_a(p) = sum_{c != a} 1/(x_a - x_c) prod_{b != a, c} (p - x_b) / (x_a - x_b);
p outside [p_tab[0], p_tab[-1]] is an error (no extrapolation).  Plain loops, no vectorised shortcuts.

Pins (tests/test_oracle_ttable.py): exactness on cubics incl. the derivative and the end intervals; the remainder of x^4 equals
prod_b (p - x_b) over the stencil (fixes WHICH four nodes are used); a library polynomial fit through the same four nodes; fourth /
third order convergence to the Lorenz-Mie T(R) and its radius derivative.
"""
import numpy as np


def stencil_start(p_tab, p):
    """i0 of reading R20.  Raises ValueError outside the table."""
    n = len(p_tab)
    if n < 4:
        raise ValueError("the table needs at least four nodes")
    if not (p_tab[0] <= p <= p_tab[n - 1]):
        raise ValueError("parameter outside the table: no extrapolation")
    i = 0
    while i < n - 2 and p >= p_tab[i + 1]:
        i += 1
    return min(max(i - 1, 0), n - 4)


def lagrange_weights(x, p):
    """(w[4], dw[4]) of the cubic through the nodes x[0..3] at p: the formulas of the module docstring, written out."""
    w = np.zeros(4)
    dw = np.zeros(4)
    for a in range(4):
        prod = 1.0
        for b in range(4):
            if b != a:
                prod *= (p - x[b]) / (x[a] - x[b])
        w[a] = prod
        acc = 0.0
        for c in range(4):
            if c == a:
                continue
            term = 1.0 / (x[a] - x[c])
            for b in range(4):
                if b != a and b != c:
                    term *= (p - x[b]) / (x[a] - x[b])
            acc += term
        dw[a] = acc
    return w, dw


def interp_table(p_tab, T_tab, p):
    """p_tab (n_tab,), T_tab (n_tab, ...) complex, p (n_out,)  ->  (T (n_out, ...), dT/dp (n_out, ...))."""
    p_tab = np.asarray(p_tab, dtype=float)
    T_tab = np.asarray(T_tab, dtype=complex)
    p = np.atleast_1d(np.asarray(p, dtype=float))
    if np.any(np.diff(p_tab) <= 0):
        raise ValueError("table nodes must be strictly increasing")
    T = np.zeros((len(p),) + T_tab.shape[1:], dtype=complex)
    dT = np.zeros_like(T)
    for j, pj in enumerate(p):
        i0 = stencil_start(p_tab, pj)
        w, dw = lagrange_weights(p_tab[i0:i0 + 4], pj)
        for a in range(4):
            T[j] += w[a] * T_tab[i0 + a]
            dT[j] += dw[a] * T_tab[i0 + a]
    return T, dT
