"""Per-scatterer transition matrices (TEST INFRASTRUCTURE ONLY - see oracle/__init__.py).

PAPER.md:254 (Eq. I9): s = T a.  The paper computes T by the null-field method for cylinders
(oracle/nullfield.py); BASELINE.json's configs use homogeneous spheres, whose T is the
closed-form Lorenz-Mie result (reading R11): diagonal, independent of m,
    T_{l,p=0} = -b_l ,   T_{l,p=1} = -a_l ,
with the Bohren-Huffman coefficients (size parameter x = k_b R, relative index m_r = sqrt(eps_r)):
    a_l = [m_r psi_l(m_r x) psi_l'(x) - psi_l(x) psi_l'(m_r x)] / [m_r psi_l(m_r x) xi_l'(x) - xi_l(x) psi_l'(m_r x)]
    b_l = [psi_l(m_r x) psi_l'(x) - m_r psi_l(x) psi_l'(m_r x)] / [psi_l(m_r x) xi_l'(x) - m_r xi_l(x) psi_l'(m_r x)]
    psi_l(z) = z j_l(z),  xi_l(z) = z h_l^(1)(z).
p = 1 is the type with a radial E component (Eq. I6b) = electric multipoles = a_l.
"""
import numpy as np
from scipy.special import spherical_jn, spherical_yn

from .modes import mode_list, n_modes


def _psi(l, z):
    return z * spherical_jn(l, z), spherical_jn(l, z) + z * spherical_jn(l, z, derivative=True)


def _xi(l, z):
    h = spherical_jn(l, z) + 1j * spherical_yn(l, z)
    hd = spherical_jn(l, z, derivative=True) + 1j * spherical_yn(l, z, derivative=True)
    return z * h, h + z * hd


def mie_ab(l, x, m_r):
    psx, dpsx = _psi(l, x)
    psm, dpsm = _psi(l, m_r * x)
    xix, dxix = _xi(l, x)
    a = (m_r * psm * dpsx - psx * dpsm) / (m_r * psm * dxix - xix * dpsm)
    b = (psm * dpsx - m_r * psx * dpsm) / (psm * dxix - m_r * xix * dpsm)
    return a, b


def mie_tmatrix_diag(lmax, k_b, radius, eps_r):
    """Diagonal of the Mie T-matrix in flat mode order (reading R1), shape (L,) complex."""
    m_r = np.sqrt(eps_r + 0j)
    if abs(m_r.imag) == 0:
        m_r = m_r.real
    x = k_b * radius
    t = np.zeros(n_modes(lmax), dtype=complex)
    for idx, (l, m, p) in enumerate(mode_list(lmax)):
        a, b = mie_ab(l, x, m_r)
        t[idx] = -b if p == 0 else -a
    return t
