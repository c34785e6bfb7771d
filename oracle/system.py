"""Dense coupled system and direct solve (TEST INFRASTRUCTURE ONLY - see oracle/__init__.py).

PAPER.md:336-369.  Eq. I21/I22:  T_j^{-1} s_j - sum_{i != j} xi^T(x_j, x_i) s_i = a^(0)_j  (minus sign: reading R7),
left-multiplied by the block-diagonal preconditioner M = diag(T_j) of Eq. I25:
        (I - T A) s = T a^(0) ,     A_jj = 0,  A_ji = xi^T(x_j, x_i)  (translation.block).
The method reaches the exact solution of this fixed linear system iteratively, so the oracle is
the definition: assemble the matrix densely and solve by LU (LAPACK zgesv via numpy; a hand-rolled
LU cross-checks it in the tests).  Adjoint (Eq. IV9): plain transpose, no conjugation.
Windows (reading R16): scatterers interact only inside their own window [win_ptr[w], win_ptr[w+1]).
T is given per type: t_diag (n_types, L) or t_full (n_types, L, L), type_of (N,).
"""
import numpy as np

from .modes import n_modes
from .translation import blocks_many


def assemble_A(lmax, k, pos, win_ptr=None, regular=False, chunk=4096):
    """Dense A (n, n), n = N L; zero diagonal blocks and zero between windows."""
    pos = np.asarray(pos, dtype=float)
    N = pos.shape[0]
    L = n_modes(lmax)
    if win_ptr is None:
        win_ptr = [0, N]
    A = np.zeros((N * L, N * L), dtype=complex)
    A4 = A.reshape(N, L, N, L)
    for w in range(len(win_ptr) - 1):
        lo, hi = win_ptr[w], win_ptr[w + 1]
        jj, ii = np.meshgrid(np.arange(lo, hi), np.arange(lo, hi), indexing="ij")
        mask = jj != ii
        jj, ii = jj[mask], ii[mask]
        for s in range(0, jj.size, chunk):
            j, i = jj[s:s + chunk], ii[s:s + chunk]
            B = blocks_many(lmax, k, pos[j] - pos[i], regular)   # (P, L_dst, L_src)
            A4[j, :, i, :] = B
    return A


def apply_T(t, type_of, x, diag, transpose=False):
    """y_j = T_{type(j)} x_j for x (N, L)."""
    if diag:
        return t[type_of] * x
    Tm = t[type_of]
    if transpose:
        Tm = np.swapaxes(Tm, 1, 2)
    return np.einsum("nab,nb->na", Tm, x)


def assemble_M(lmax, k, pos, t, type_of, diag, win_ptr=None):
    """M = I - diag(T_j) A  (Eqs. I22, I25)."""
    N = len(pos)
    L = n_modes(lmax)
    A = assemble_A(lmax, k, pos, win_ptr)
    A3 = A.reshape(N, L, N * L)
    if diag:
        TA = t[type_of][:, :, None] * A3
    else:
        TA = np.einsum("nab,nbc->nac", t[type_of], A3)
    return np.eye(N * L, dtype=complex) - TA.reshape(N * L, N * L)


def solve_forward(M, t, type_of, diag, p_inc):
    """s = M^{-1} (T a^(0)) by LU."""
    b = apply_T(t, type_of, p_inc, diag).reshape(-1)
    return np.linalg.solve(M, b).reshape(p_inc.shape)


def solve_adjoint(M, w):
    """lambda = M^{-T} w by LU (Eq. IV9 with Omega = T^{-1} M: a = T^T lambda)."""
    return np.linalg.solve(M.T, w.reshape(-1)).reshape(w.shape)


def lu_solve_plain(M, b):
    """Hand-rolled LU with partial pivoting (cross-check of the LAPACK call; small n only)."""
    A = np.array(M, dtype=complex)
    x = np.array(b, dtype=complex).reshape(-1)
    n = A.shape[0]
    for c in range(n):
        piv = c + int(np.argmax(np.abs(A[c:, c])))
        if piv != c:
            A[[c, piv]] = A[[piv, c]]
            x[[c, piv]] = x[[piv, c]]
        f = A[c + 1:, c] / A[c, c]
        A[c + 1:, c:] -= f[:, None] * A[c, c:][None, :]
        x[c + 1:] -= f * x[c]
    for c in range(n - 1, -1, -1):
        x[c] = (x[c] - A[c, c + 1:] @ x[c + 1:]) / A[c, c]
    return x
