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


# ------------------------------------------------------------------------------------------------ positions (Eqs. IV3-IV6)
def fd_position(lmax, k, pos, radii, eps_r, inc_fn, v, j, alpha, h=1e-5):
    """dJ/dx_{j,alpha} at fixed v by central differences of the full dense solve; inc_fn(pos) -> a^(0) (N, L)."""
    pp, pm = np.array(pos, dtype=float), np.array(pos, dtype=float)
    pp[j, alpha] += h
    pm[j, alpha] -= h
    return (_solve_J(lmax, k, pp, radii, eps_r, inc_fn(pp), v)[0] - _solve_J(lmax, k, pm, radii, eps_r, inc_fn(pm), v)[0]) / (2 * h)


def dA_dposition(lmax, k, pos, j):
    """d A / d x_{j,alpha}, alpha = x, y, z, assembled densely: (3, N L, N L).  Only the block row j (A_ji depends on
    x_j - x_i) and the block column j (A_ij depends on x_i - x_j, hence the minus sign) are non-zero; the blocks are the
    ANALYTIC derivative of the translation coefficients (translation.d_block)."""
    from . import translation as tr
    N, L = len(pos), n_modes(lmax)
    out = np.zeros((3, N * L, N * L), dtype=complex)
    for i in range(N):
        if i == j:
            continue
        out[:, j * L:(j + 1) * L, i * L:(i + 1) * L] = tr.d_block(lmax, k, pos[j], pos[i])
        out[:, i * L:(i + 1) * L, j * L:(j + 1) * L] = -tr.d_block(lmax, k, pos[i], pos[j])
    return out


def adjoint_position_gradient(lmax, k, pos, radii, eps_r, inc_fn, v, h=1e-5, dinc_fn=None):
    """All dJ/dx_{j,alpha} through ONE adjoint solve: lambda^T T (dA/dx_{j,alpha}) s + lambda^T T da^(0)/dx_{j,alpha}
    (Eq. IV6 with Omega = T^{-1} M; dOmega/dq = -dA/dq).  dA/dq is the analytic derivative of Eq. I23's off-diagonal blocks
    (dA_dposition; "can be computed analytically"); da^(0)/dq, which is not part of Omega, by central
    differences of inc_fn, or exactly from dinc_fn(pos) -> (N, 3, L) = d a^(0)_j / d x_{j,alpha} when given (plane wave:
    i k_alpha a^(0)_j, Eq. II6).  Returns (N, 3).  Pinned by fd_position (central differences of the whole dense solve)."""
    p_inc = inc_fn(pos)
    J, s, M, t = _solve_J(lmax, k, pos, radii, eps_r, p_inc, v)
    lam = system.solve_adjoint(M, v)
    N, L = s.shape
    mu = (t * lam).reshape(-1)                                     # T^T lambda (T diagonal)
    out = np.zeros((N, 3), dtype=complex)
    dinc = dinc_fn(pos) if dinc_fn is not None else None
    for j in range(N):
        dA = dA_dposition(lmax, k, pos, j)
        for alpha in range(3):
            if dinc is not None:
                dp = np.zeros((N, L), dtype=complex)
                dp[j] = dinc[j, alpha]
            else:
                pp, pm = np.array(pos, dtype=float), np.array(pos, dtype=float)
                pp[j, alpha] += h
                pm[j, alpha] -= h
                dp = (inc_fn(pp) - inc_fn(pm)) / (2 * h)
            out[j, alpha] = mu @ (dA[alpha] @ s.reshape(-1)) + mu @ dp.reshape(-1)
    return out, s, lam


# ------------------------------------------------------------------------------ shape parameters of null-field T-matrices
def _solve_J_shapes(lmax, k, pos, gen_fn, params, type_of, eps_r, p_inc, v):
    from . import nullfield
    t = np.stack([nullfield.nullfield_tmatrix(lmax, k, eps_r, gen_fn(p)) for p in params])
    M = system.assemble_M(lmax, k, pos, t, type_of, False)
    return np.sum(v * system.solve_forward(M, t, type_of, False, p_inc))


def fd_shape_parameter(lmax, k, pos, gen_fn, params, type_of, eps_r, p_inc, v, which, h=1e-5):
    """dJ/dp_which, J = v^T s, for a library of bodies of revolution gen_fn(p) (a geometry parameter enters only
    through T): central difference of the full dense solve with the null-field T-matrices rebuilt at p +- h - the plain
    definition of the derivative, no adjoint formula."""
    pp, pm = np.array(params, dtype=float), np.array(params, dtype=float)
    pp[which] += h
    pm[which] -= h
    return (_solve_J_shapes(lmax, k, pos, gen_fn, pp, type_of, eps_r, p_inc, v)
            - _solve_J_shapes(lmax, k, pos, gen_fn, pm, type_of, eps_r, p_inc, v)) / (2 * h)
