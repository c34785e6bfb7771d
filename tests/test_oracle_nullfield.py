"""Pins of the oracle's null-field T-matrix (oracle/nullfield.py, Eqs. I10-I11; readings R18, R19).
None of them restates the oracle's formula: the sphere has the closed-form Lorenz-Mie answer, the displaced sphere follows
from it through the (separately pinned) regular translation operator, and losslessness / reciprocity / mirror symmetry
are properties of the exact T-matrix."""
import numpy as np

from oracle import nullfield as nf, tmatrix, translation
from oracle.modes import mode_index, mode_list
from paper_2107_09879_b200 import workloads as W

K = W.K_B


def perm_neg_m(lmax):
    n = len(mode_list(lmax))
    P = np.zeros((n, n))
    for i, (l, m, p) in enumerate(mode_list(lmax)):
        P[i, mode_index(l, -m, p, lmax)] = 1.0
    return P


def test_sphere_reproduces_lorenz_mie():
    for lmax, radius, eps in ((3, 0.2, 4.0), (6, 0.24, 4.0), (2, 0.1, 2.25)):
        T = nf.nullfield_tmatrix(lmax, K, eps, W.generatrix_sphere(radius, 48))
        d = tmatrix.mie_tmatrix_diag(lmax, K, radius, eps)
        assert np.abs(T - np.diag(d)).max() <= 1e-12 * np.abs(d).max()


def test_lossy_sphere_reproduces_lorenz_mie_and_absorbs():
    eps = 12.0 + 0.8j
    T = nf.nullfield_tmatrix(3, K, eps, W.generatrix_sphere(0.15, 48))
    d = tmatrix.mie_tmatrix_diag(3, K, 0.15, eps)
    assert np.abs(T - np.diag(d)).max() <= 1e-12 * np.abs(d).max()
    Tc = nf.nullfield_tmatrix(6, K, eps, W.generatrix_spheroid(0.12, 0.18, 64))
    S = np.eye(len(Tc)) + 2.0 * Tc
    ev = np.linalg.eigvalsh(np.eye(len(Tc)) - S.conj().T @ S)        # absorbed power is non-negative for every incident field
    assert ev.min() >= -1e-6 and ev.max() > 1e-3


def test_printed_forms_fail_the_mie_limit():
    """Reading R18: the printed minus sign; reading R19: T = -P Q^{-1} with P the OUTGOING matrix as printed."""
    gen = W.generatrix_sphere(0.2, 48)
    d = np.diag(tmatrix.mie_tmatrix_diag(3, K, 0.2, 4.0))
    assert np.abs(nf.nullfield_tmatrix(3, K, 4.0, gen, printed=True) - d).max() > 0.1
    b_rg, b_out = nf.surface_matrices(3, K, K * 2.0, gen)
    assert np.abs(-b_out @ np.linalg.inv(b_rg) - d).max() > 0.1


def test_displaced_sphere_equals_translated_mie():
    """A sphere whose centre sits at c = (0, 0, 0.05) is not a sphere about the origin: its T-matrix is full in (l, p).
    Exact relation: T_0 = RgA(0 <- c) T_Mie RgA(c <- 0) (incident field re-expanded about c, scattered field re-expanded
    about the origin; both with the REGULAR translation operator).  Pins index order, m signs and the p <-> 1-p pairing."""
    lh, off, radius = 6, 0.05, 0.2
    Tn = nf.nullfield_tmatrix(lh, K, 4.0, W.generatrix_sphere(radius, 64, offset=off))
    c, o = np.array([0.0, 0.0, off]), np.zeros(3)
    to_c = translation.block(lh, K, c, o, regular=True)
    to_o = translation.block(lh, K, o, c, regular=True)
    Tt = to_o @ np.diag(tmatrix.mie_tmatrix_diag(lh, K, radius, 4.0)) @ to_c
    a, b = nf.sub_block(Tn, lh, 2), nf.sub_block(Tt, lh, 2)
    assert np.abs(b - np.diag(np.diag(b))).max() > 0.05          # the case is not diagonal
    assert np.abs(a - b).max() <= 1e-9


def test_internal_truncation_converges_to_the_translated_mie_block():
    """lmax_internal: the l <= 2 block of the displaced sphere computed with expansions up to 2 is off by the coupling to
    higher orders; with the expansions carried to 6 it reproduces the exact (translated Lorenz-Mie) block."""
    off, radius = 0.08, 0.2
    gen = W.generatrix_sphere(radius, 64, offset=off)
    c, o = np.array([0.0, 0.0, off]), np.zeros(3)
    exact = nf.sub_block(translation.block(6, K, o, c, regular=True) @ np.diag(tmatrix.mie_tmatrix_diag(6, K, radius, 4.0))
                         @ translation.block(6, K, c, o, regular=True), 6, 2)
    coarse = np.abs(nf.nullfield_tmatrix(2, K, 4.0, gen) - exact).max()
    fine = np.abs(nf.nullfield_tmatrix(2, K, 4.0, gen, lmax_internal=6) - exact).max()
    assert coarse > 1e-4 and fine <= 1e-7 and fine < 1e-3 * coarse


def test_spheroid_is_lossless_reciprocal_and_mirror_symmetric():
    lmax = 6
    T = nf.nullfield_tmatrix(lmax, K, 4.0, W.generatrix_spheroid(0.15, 0.22, 64))
    n = len(T)
    S = np.eye(n) + 2.0 * T
    assert np.abs(S @ S.conj().T - np.eye(n)).max() <= 1e-5      # truncation error of the method at lmax 6
    P = perm_neg_m(lmax)
    assert np.abs(T.T - P @ T @ P).max() <= 1e-5                 # reciprocity in the complex-m basis
    modes = mode_list(lmax)
    for i, (l, m, p) in enumerate(modes):
        for j, (l2, m2, p2) in enumerate(modes):
            if m != m2 or (l + p) % 2 != (l2 + p2) % 2:            # axial symmetry; mirror z -> -z
                assert abs(T[i, j]) <= 1e-13
    assert np.abs(T - np.diag(np.diag(T))).max() > 1e-3


def test_cylinder_converges_with_the_quadrature_and_is_nearly_lossless():
    a = nf.nullfield_tmatrix(4, K, 4.0, W.generatrix_cylinder(0.15, 0.3, 32))
    b = nf.nullfield_tmatrix(4, K, 4.0, W.generatrix_cylinder(0.15, 0.3, 64))
    assert np.abs(a - b).max() <= 1e-12
    T = nf.nullfield_tmatrix(6, K, 4.0, W.generatrix_cylinder(0.15, 0.3, 48))
    S = np.eye(len(T)) + 2.0 * T
    assert np.abs(S @ S.conj().T - np.eye(len(T))).max() <= 2e-3  # sharp edges: slow convergence in lmax (0.4e-3 measured)
