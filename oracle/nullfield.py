"""Transition matrix of one homogeneous scatterer by the null-field method (TEST INFRASTRUCTURE ONLY - see
oracle/__init__.py).

PAPER.md:258-267, Eqs. I10-I11: T follows from two matrices of surface integrals over the scatterer surface dS, with the
internal field expanded in regular wavefunctions of the scatterer medium (wavenumber k_s) and the incident / scattered
field in regular / outgoing wavefunctions of the background (k_b).  The integrals are evaluated here LITERALLY: a
two-dimensional quadrature over the surface (the caller's generatrix nodes in theta, trapezoid rule in phi), the
integrand built from the Cartesian wavefunctions of oracle/vswf.py, cross products and the area-weighted normal.  No
use is made of the axial symmetry (the CUDA path integrates phi analytically, m = m').

Readings (R18, R19; both pinned by the Lorenz-Mie limit and by the displaced sphere, tests/test_oracle_nullfield.py):
  R18  the two terms of the integrand ADD.  With curl Phi_p = k Phi_{1-p} (Eq. I6b, pinned in tests/test_oracle_vswf_translation.py)
       the surface form  {E, W} = int [ E x curl W - W x curl E ] . n dS  of a field E = RPhi_{mu}(k_s x) and a test function
       W = Psi_{l,-m,p}(k_b x) is
           k_b int [ RPhi_{l'm'p'}(k_s x) x Psi_{l,-m,1-p}(k_b x) + (k_s/k_b) RPhi_{l'm'1-p'}(k_s x) x Psi_{l,-m,p}(k_b x) ] . n dS ;
       Eq. I10 prints a minus between the terms (printed=True reproduces it; the Mie pin fails for it).
  R19  the matrix to invert is the one with the OUTGOING background function (Eq. I10a, "P"): testing with the outgoing
       function extracts the incident coefficients ( {RPhi_nu, Phi_nubar} = +i pi / k_b ), testing with the regular one the
       scattered coefficients ( {Phi_nu, RPhi_nubar} = -i pi / k_b ), so
           a = (k_b / i pi) B_out c ,  s = -(k_b / i pi) B_rg c   =>   T = - B_rg B_out^{-1} ,
       i.e. Eq. I11 with the printed names P and Q interchanged.
"""
import numpy as np

from .modes import mode_index, mode_list, n_modes
from .vswf import sph_unit_vectors, vswf_all


def surface_quadrature(gen, n_phi):
    """Points x (P,3) and area-weighted outward normals n dS (P,3) of the surface of revolution r = r(theta):
    n dS = r^2 sin(theta) ( r_hat - (r'/r) theta_hat ) dtheta dphi."""
    theta, r, dr, w = (np.asarray(a, dtype=float) for a in gen)
    phi = 2.0 * np.pi * np.arange(n_phi) / n_phi
    T, F = np.meshgrid(theta, phi, indexing="ij")
    R, DR, Wt = (np.repeat(a[:, None], n_phi, axis=1) for a in (r, dr, w))
    rh, th, _ = sph_unit_vectors(T.ravel(), F.ravel())
    R, DR, Wt, T = R.ravel(), DR.ravel(), Wt.ravel(), T.ravel()
    x = R[:, None] * rh
    nds = (R * R * np.sin(T) * Wt * (2.0 * np.pi / n_phi))[:, None] * (rh - (DR / R)[:, None] * th)
    return x, nds


def surface_matrices(lmax, k_b, k_s, gen, n_phi=None, printed=False):
    """B_rg, B_out (L, L): rows nu = (l, m, p) of the background test function, columns mu = (l', m', p') of the
    internal expansion function (the index pairs of Eq. I10), divided by k_b."""
    n_phi = n_phi or 4 * lmax + 4
    modes = mode_list(lmax)
    L = n_modes(lmax)
    bar = np.array([mode_index(l, -m, p, lmax) for (l, m, p) in modes])           # (l, -m, p)
    swap = np.array([mode_index(l, m, 1 - p, lmax) for (l, m, p) in modes])       # (l, m, 1-p)
    x, nds = surface_quadrature(gen, n_phi)
    fs = vswf_all(lmax, k_s, x, regular=True)                                      # (L, P, 3)
    sign = -1.0 if printed else 1.0
    out = []
    for regular in (True, False):
        fb = vswf_all(lmax, k_b, x, regular=regular)
        w1 = np.cross(fb[bar][swap], nds[None])                                    # Psi_{l,-m,1-p} x n dS
        w2 = np.cross(fb[bar], nds[None])                                          # Psi_{l,-m,p}   x n dS
        # (a x b) . n = a . (b x n)
        b = np.einsum("mqc,nqc->nm", fs, w1) + sign * (k_s / k_b) * np.einsum("mqc,nqc->nm", fs[swap], w2)
        out.append(b)
    return out[0], out[1]


def nullfield_tmatrix(lmax, k_b, eps_r, gen, n_phi=None, printed=False, lmax_internal=None):
    """T (L, L) of a homogeneous non-magnetic scatterer of relative permittivity eps_r (vs. the background) bounded by
    the surface of revolution `gen`; s = T a in flat mode order (reading R1).  lmax_internal > lmax: the method is run
    with all expansions truncated at lmax_internal and the block of the modes l <= lmax is returned (the paper uses
    lmax_internal = lmax = 6)."""
    k_s = k_b * np.sqrt(eps_r + 0j)
    if abs(k_s.imag) == 0.0:
        k_s = k_s.real
    li = lmax_internal or lmax
    b_rg, b_out = surface_matrices(li, k_b, k_s, gen, n_phi, printed)
    t = -np.linalg.solve(b_out.T, b_rg.T).T
    return t if li == lmax else sub_block(t, li, lmax)


def sub_block(t, lmax_from, lmax_to):
    """Rows / columns of the modes with l <= lmax_to out of a matrix in the flat order of lmax_from."""
    idx = [mode_index(l, m, p, lmax_from) for (l, m, p) in mode_list(lmax_to)]
    return t[np.ix_(idx, idx)]
