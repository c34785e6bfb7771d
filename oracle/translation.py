"""Translation (addition-theorem) coefficients (TEST INFRASTRUCTURE ONLY - see oracle/__init__.py).

PAPER.md:292-336, Eqs. I15-I21, with the repairs listed in DESIGN.md "Readings":
  R3  argument of xi is d = x_dest - x_source (Eq. I21 is right, the text of Eq. I15 is not);
  R4  the right-hand side of Eq. I15 is the REGULAR wavefunction about the destination;
  R5  normalisation sqrt((2l+1)(2l'+1) / (2 l(l+1) l'(l'+1)))  (an l' is missing in print);
  R6  b5's second 3j symbol is (l l' q-1; 0 0 0)  (the printed one vanishes identically);
  R8  h_q is evaluated at k|d|.

    Phi_{l,m,p}(k(x - x_src)) = sum_{l'm'p'} xi_{lmp;l'm'p'}(k d) RPhi_{l'm'p'}(k(x - x_dst)),  |x - x_dst| < |d|
    xi = delta_{pp'} alpha + (1 - delta_{pp'}) beta                                           (I16)
    alpha = e^{i(m-m')phi_d} sum_{q=|l-l'|}^{l+l'}   a5(l,m|l',m'|q) h_q(k|d|) Pbar_q^{|m-m'|}(cos theta_d)   (I17a)
    beta  = e^{i(m-m')phi_d} sum_{q=|l-l'|+1}^{l+l'} b5(l,m|l',m'|q) h_q(k|d|) Pbar_q^{|m-m'|}(cos theta_d)   (I17b)
The first index triple is the SOURCE mode, the second the DESTINATION mode.
"""
from functools import lru_cache
from math import sqrt

import numpy as np

from . import special as sp
from .modes import mode_list, n_modes
from .vswf import cart_to_sph
from .wigner import wigner_3j


def _phase(l, m, lp, mp, q):
    """i^{|m-m'|-|m|-|m'|+l'-l+q} (-1)^{m-m'}  (Eq. I18)."""
    e = abs(m - mp) - abs(m) - abs(mp) + lp - l + q
    return (1j) ** (e % 4) * (-1) ** ((m - mp) % 2)


def _norm(l, lp):
    return sqrt((2 * l + 1) * (2 * lp + 1) / (2.0 * l * (l + 1) * lp * (lp + 1)))


@lru_cache(maxsize=None)
def a5(l, m, lp, mp, q):
    """Eq. I18a (repair R5)."""
    return (_phase(l, m, lp, mp, q) * (l * (l + 1) + lp * (lp + 1) - q * (q + 1)) * sqrt(2 * q + 1)
            * _norm(l, lp) * wigner_3j(l, lp, q, m, -mp, mp - m) * wigner_3j(l, lp, q, 0, 0, 0))


@lru_cache(maxsize=None)
def b5(l, m, lp, mp, q):
    """Eq. I18b (repairs R5, R6)."""
    rad = (l + lp + 1 + q) * (l + lp + 1 - q) * (q + l - lp) * (q - l + lp) * (2 * q + 1)
    if rad <= 0:
        return 0.0
    return (_phase(l, m, lp, mp, q) * sqrt(rad) * _norm(l, lp)
            * wigner_3j(l, lp, q, m, -mp, mp - m) * wigner_3j(l, lp, q - 1, 0, 0, 0))


def xi_matrix(lmax, k, d, regular=False):
    """xi[(l m p), (l' m' p')](k d): rows = source mode, columns = destination mode (Eq. I16-I17).
    regular=True replaces h_q by j_q (regular translation RgA, used only for cross-sections)."""
    r, theta, phi = cart_to_sph(np.asarray(d, dtype=float))
    kr = k * float(r)
    ct = float(np.cos(theta))
    modes = mode_list(lmax)
    L = n_modes(lmax)
    zq = [(sp.sph_jn(q, kr) + 0j) if regular else sp.sph_h1(q, kr) for q in range(2 * lmax + 1)]
    pq = {(q, mu): float(sp.pbar(q, mu, ct)) for q in range(2 * lmax + 1) for mu in range(q + 1)}
    xi = np.zeros((L, L), dtype=complex)
    for a, (l, m, p) in enumerate(modes):
        for b, (lp, mp, pp) in enumerate(modes):
            mu = abs(m - mp)
            s = 0.0
            if p == pp:
                for q in range(abs(l - lp), l + lp + 1):
                    if q >= mu:
                        s += a5(l, m, lp, mp, q) * zq[q] * pq[(q, mu)]
            else:
                for q in range(abs(l - lp) + 1, l + lp + 1):
                    if q >= mu:
                        s += b5(l, m, lp, mp, q) * zq[q] * pq[(q, mu)]
            xi[a, b] = np.exp(1j * (m - mp) * float(phi)) * s
    return xi


def d_xi_matrix(lmax, k, d, regular=False):
    """Gradient of xi_matrix with respect to the displacement d, analytically: (3, L, L), [alpha, source mode, destination mode].

    PAPER.md:517-546 (App. IV, Eqs. IV2-IV6) needs dOmega/dq_i for a scatterer position q_i, and PAPER.md:560 (observation b)
    notes that it "can be computed analytically": Omega depends on the positions only through xi(k(x_j - x_i)) (Eq. I23).
    Chain rule on Eq. I17 in the spherical coordinates (r, theta, phi) of d,
        d/d d_alpha = r_hat_alpha d/dr + (theta_hat_alpha / r) d/dtheta + (phi_hat_alpha / (r sin theta)) d/dphi ,
    applied term by term to  e^{i mu phi} h_q(k r) Pbar_q^{|mu|}(cos theta),  mu = m - m':
        d/dr     -> k h_q'(k r)
        d/dtheta -> taubar_q^{|mu|}(theta)                       (= d Pbar_q^{|mu|}(cos theta) / d theta, Eq. II7 notation)
        d/dphi   -> i mu ;  Pbar_q^{|mu|} / sin theta = pibar_q^{|mu|}(theta)   (regular at the poles; absent for mu = 0)."""
    from .vswf import sph_unit_vectors
    r, theta, phi = cart_to_sph(np.asarray(d, dtype=float))
    r, theta, phi = float(r), float(theta), float(phi)
    kr = k * r
    ct = float(np.cos(theta))
    rh, th, ph = sph_unit_vectors(theta, phi)
    modes = mode_list(lmax)
    L = n_modes(lmax)
    nq = 2 * lmax + 1
    zq = [(sp.sph_jn(q, kr) + 0j) if regular else sp.sph_h1(q, kr) for q in range(nq)]
    dzq = [(sp.sph_jn_d(q, kr) + 0j) if regular else sp.sph_h1_d(q, kr) for q in range(nq)]
    pq = {(q, mu): float(sp.pbar(q, mu, ct)) for q in range(nq) for mu in range(q + 1)}
    tq = {(q, mu): float(sp.taubar(q, mu, theta)) for q in range(nq) for mu in range(q + 1)}
    piq = {(q, mu): float(sp.pibar(q, mu, theta)) for q in range(nq) for mu in range(q + 1)}
    out = np.zeros((3, L, L), dtype=complex)
    for a, (l, m, p) in enumerate(modes):
        for b, (lp, mp, pp) in enumerate(modes):
            mu = m - mp
            am = abs(mu)
            s_r = s_t = s_p = 0.0
            q0 = abs(l - lp) + (0 if p == pp else 1)
            for q in range(q0, l + lp + 1):
                if q < am:
                    continue
                c = a5(l, m, lp, mp, q) if p == pp else b5(l, m, lp, mp, q)
                s_r += c * k * dzq[q] * pq[(q, am)]
                s_t += c * zq[q] * tq[(q, am)] / r
                s_p += c * zq[q] * (1j * mu) * piq[(q, am)] / r
            out[:, a, b] = np.exp(1j * mu * phi) * (rh * s_r + th * s_t + ph * s_p)
    return out


def d_block(lmax, k, x_dst, x_src, regular=False):
    """d A_ji / d x_j (= - d A_ji / d x_i): (3, L, L) with destination rows, source columns (see block())."""
    d = np.asarray(x_dst, dtype=float) - np.asarray(x_src, dtype=float)
    return np.transpose(d_xi_matrix(lmax, k, d, regular), (0, 2, 1))


def block(lmax, k, x_dst, x_src, regular=False):
    """A_{ji} = xi^T(x_j, x_i): [A_ji]_{(lmp),(l'm'p')} = xi_{l'm'p';lmp}(k(x_j - x_i))  (Eq. I21).
    Destination modes index rows, source modes index columns."""
    d = np.asarray(x_dst, dtype=float) - np.asarray(x_src, dtype=float)
    return xi_matrix(lmax, k, d, regular).T


@lru_cache(maxsize=None)
def coupling_tables(lmax):
    """Constant part of Eq. I17 arranged for many displacements at once.
    Returns (coef, mu) with coef[q, b, a] = a5 or b5 (l,m,p = source mode a; l',m',p' = destination
    mode b; zero where q is outside the sum range or q < |m-m'|) and mu[b, a] = m - m'.
    Same numbers as xi_matrix uses, only tabulated."""
    modes = mode_list(lmax)
    L = n_modes(lmax)
    nq = 2 * lmax + 1
    coef = np.zeros((nq, L, L), dtype=complex)
    mu = np.zeros((L, L), dtype=int)
    for a, (l, m, p) in enumerate(modes):
        for b, (lp, mp, pp) in enumerate(modes):
            mu[b, a] = m - mp
            for q in range(abs(l - lp) + (0 if p == pp else 1), l + lp + 1):
                if q >= abs(m - mp):
                    coef[q, b, a] = a5(l, m, lp, mp, q) if p == pp else b5(l, m, lp, mp, q)
    return coef, mu


def blocks_many(lmax, k, D, regular=False):
    """A-blocks (destination rows, source columns) for displacements D[(P),3] = x_dst - x_src.
    Returns (P, L, L).  Identical arithmetic to block(), vectorised over P."""
    D = np.atleast_2d(np.asarray(D, dtype=float))
    r, theta, phi = cart_to_sph(D)
    kr = k * r
    ct = np.cos(theta)
    coef, mu = coupling_tables(lmax)
    nq = 2 * lmax + 1
    P = D.shape[0]
    L = n_modes(lmax)
    out = np.zeros((P, L, L), dtype=complex)
    amu = np.abs(mu)
    for q in range(nq):
        zq = (sp.sph_jn(q, kr) + 0j) if regular else sp.sph_h1(q, kr)
        # W[P, mu_abs] = z_q(kr) Pbar_q^{mu_abs}(cos theta)
        W = np.zeros((P, nq), dtype=complex)
        for ma in range(q + 1):
            W[:, ma] = zq * sp.pbar(q, ma, ct)
        out += coef[q][None, :, :] * W[:, amu]
    out *= np.exp(1j * mu[None, :, :] * phi[:, None, None])
    return out
