"""Scattered fields and cross-sections (TEST INFRASTRUCTURE ONLY - see oracle/__init__.py).

PAPER.md:284, 359 (Eqs. I13, I24):  E_sca(x) = sum_i sum_{lmp} s_{lmp;i} Phi_{lmp}(k_b (x - x_i)).
H (reading R10; the paper gives no formula): curl Phi_p = k Phi_{1-p} and curl E = i omega mu H give
    Z_b H_sca(x) = -i sum_i sum_{lmp} s_{lmp;i} Phi_{l,m,1-p}(k_b (x - x_i)).
Cross-sections (textbook consequence of the normalisation, used as energy pins, not printed in the paper),
for a unit-amplitude plane wave and RgA = translation with j_q in place of h_q:
    C_ext = -(pi/k^2) Re sum_j p_j^H s_j ,   C_sca = (pi/k^2) Re sum_j s_j^H ( s_j + sum_{i != j} RgA_ji s_i ).
"""
import numpy as np

from .modes import mode_list, n_modes
from .system import assemble_A
from .vswf import vswf_all


def e_sca(lmax, k, pos, s, pts):
    pts = np.atleast_2d(np.asarray(pts, dtype=float))
    out = np.zeros((pts.shape[0], 3), dtype=complex)
    for i in range(len(pos)):
        F = vswf_all(lmax, k, pts - pos[i])           # (L, M, 3)
        out += np.einsum("a,amc->mc", s[i], F)
    return out


def zh_sca(lmax, k, pos, s, pts):
    """Z_b * H_sca."""
    L = n_modes(lmax)
    half = L // 2
    swap = np.concatenate([np.arange(half, L), np.arange(0, half)])   # (l,m,p) -> (l,m,1-p)
    pts = np.atleast_2d(np.asarray(pts, dtype=float))
    out = np.zeros((pts.shape[0], 3), dtype=complex)
    for i in range(len(pos)):
        F = vswf_all(lmax, k, pts - pos[i])[swap]
        out += np.einsum("a,amc->mc", s[i], F)
    return -1j * out


def cross_sections(lmax, k, pos, s, p_inc, win_ptr=None):
    """(C_ext, C_sca) for the whole ensemble (one window)."""
    N, L = s.shape
    RgA = assemble_A(lmax, k, pos, win_ptr, regular=True)
    sv = s.reshape(-1)
    c_ext = -(np.pi / k ** 2) * np.real(np.vdot(p_inc.reshape(-1), sv))
    c_sca = (np.pi / k ** 2) * np.real(np.vdot(sv, sv + RgA @ sv))
    return c_ext, c_sca
