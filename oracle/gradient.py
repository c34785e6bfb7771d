"""Adjoint sensitivities (TEST INFRASTRUCTURE ONLY - see oracle/__init__.py).

PAPER.md:496-560, Appendix IV.  For a figure of merit built on the bilinear functional J = v^T s (Eq. IV3/IV4; v = overlap of
the desired field with the outgoing waves) the paper's Eqs. IV6/IV8 give
        dJ/dq = -v^T Omega^{-1} (dOmega/dq) s ,      Omega^T a = v   (adjoint simulation, Eq. IV9).
With Omega = T^{-1} M, M = I - T A (Eq. I25), a = T^T lambda, M^T lambda = v, and for a GEOMETRY parameter p of scatterer j
(only the diagonal block T_j^{-1} depends on it):
        dJ/dp = lambda_j^T (dT_j/dp) T_j^{-1} s_j = lambda_j^T (dT_j/dp) (a^(0)_j + (A s)_j).
The plain definition of the same number is the derivative of J(p) = v^T s(p) itself: `fd_radius` differentiates the dense-LU
solve numerically (central differences), which is what pins the adjoint formula.
"""
import numpy as np

from . import incident, system, tmatrix
from .modes import n_modes


def _solve_J(lmax, k, pos, radii, eps_r, p_inc, v):
    t = np.stack([tmatrix.mie_tmatrix_diag(lmax, k, r, eps_r) for r in radii])
    type_of = np.arange(len(radii))
    M = system.assemble_M(lmax, k, pos, t, type_of, True)
    s = system.solve_forward(M, t, type_of, True, p_inc)
    return np.sum(v * s), s, M, t


def fd_radius(lmax, k, pos, radii, eps_r, p_inc, v, j, h=1e-6):
    """dJ/dR_j by central differences of the full dense solve (the plain definition)."""
    rp, rm = np.array(radii, dtype=float), np.array(radii, dtype=float)
    rp[j] += h
    rm[j] -= h
    return (_solve_J(lmax, k, pos, rp, eps_r, p_inc, v)[0] - _solve_J(lmax, k, pos, rm, eps_r, p_inc, v)[0]) / (2 * h)


def mie_dT_dR(lmax, k, radius, eps_r, h=1e-4):
    """d(diag T)/dR by Richardson-extrapolated central differences of the closed-form Mie coefficients."""
    d = lambda hh: (tmatrix.mie_tmatrix_diag(lmax, k, radius + hh, eps_r) - tmatrix.mie_tmatrix_diag(lmax, k, radius - hh, eps_r)) / (2 * hh)
    return (4.0 * d(h / 2) - d(h)) / 3.0


def adjoint_radius_gradient(lmax, k, pos, radii, eps_r, p_inc, v):
    """All dJ/dR_j through ONE adjoint solve (Eqs. IV8-IV9): returns (grad (N,), s, lambda)."""
    J, s, M, t = _solve_J(lmax, k, pos, radii, eps_r, p_inc, v)
    lam = system.solve_adjoint(M, v)
    N, L = s.shape
    A = system.assemble_A(lmax, k, pos)
    q = p_inc + (A @ s.reshape(-1)).reshape(N, L)                 # a^(0) + A s  (= T^{-1} s)
    dT = np.stack([mie_dT_dR(lmax, k, r, eps_r) for r in radii])
    return np.sum(lam * dT * q, axis=1), s, lam
