"""Pins for oracle/vswf.py and oracle/translation.py.

VSWFs (Eq. I6): numerical curl identities.  Translation block
(Eqs. I15-I18 with repairs R3-R6, R8): pointwise addition theorem against
direct VSWF evaluation; wrong-direction / printed-normalisation variants must FAIL it;
structural identities S1-S4 of SURVEY.md 8(c)."""
import numpy as np
import pytest

from oracle import translation as tr
from oracle import vswf
from oracle.modes import mode_index, mode_list, n_modes

K = 2 * np.pi


def _curl(f, x, h=1e-4):
    """curl of a vector field f: R^3 -> C^3 by central differences."""
    J = np.zeros((3, 3), dtype=complex)          # J[a, b] = d f_a / d x_b
    for b in range(3):
        e = np.zeros(3)
        e[b] = h
        J[:, b] = (f(x + e) - f(x - e)) / (2 * h)
    return np.array([J[2, 1] - J[1, 2], J[0, 2] - J[2, 0], J[1, 0] - J[0, 1]]), np.trace(J)


@pytest.mark.parametrize("regular", [False, True])
def test_vswf_curl_identities(regular):
    rng = np.random.default_rng(3)
    for _ in range(3):
        x = rng.uniform(-0.6, 0.6, 3) + np.array([0.2, 0.1, 0.3])
        for (l, m, p) in mode_list(3):
            f0 = lambda y: vswf.vswf(l, m, p, K, y, regular)
            c, div = _curl(f0, x)
            other = vswf.vswf(l, m, 1 - p, K, x, regular)
            scale = np.abs(other).max()
            assert np.abs(c / K - other).max() < 2e-6 * scale      # curl Phi_p = k Phi_{1-p}
            assert abs(div) < 2e-6 * K * scale                      # transversality


def test_vswf_p0_is_grad_phi_cross_x():
    # Eq. I6a literally: Phi_{l m 0} = [2l(l+1)]^{-1/2} grad(phi_lm) x x
    from oracle import special as sp
    rng = np.random.default_rng(4)
    h = 1e-5
    for (l, m) in [(1, 0), (1, -1), (2, 1), (3, -2), (3, 3)]:
        def phi(y):
            r, th, ph = vswf.cart_to_sph(y)
            return sp.sph_h1(l, K * r) * sp.pbar(l, abs(m), np.cos(th)) * np.exp(1j * m * ph)
        x = rng.uniform(0.2, 0.7, 3)
        g = np.array([(phi(x + h * e) - phi(x - h * e)) / (2 * h) for e in np.eye(3)])
        ref = np.cross(g, x) / np.sqrt(2 * l * (l + 1))
        got = vswf.vswf(l, m, 0, K, x)
        assert np.abs(got - ref).max() < 1e-7 * np.abs(ref).max()


def _addition_error(xi, lmax, lbig, xs, xd, pt, regular_lhs=False):
    R = vswf.vswf_all(lbig, K, pt - xd, regular=True)
    big = mode_list(lbig)
    err = 0.0
    for (l, m, p) in mode_list(lmax):
        a = big.index((l, m, p))
        lhs = vswf.vswf(l, m, p, K, pt - xs, regular=regular_lhs)
        err = max(err, np.abs(lhs - xi[a, :] @ R).max() / np.abs(lhs).max())
    return err


def test_addition_theorem_pointwise():
    rng = np.random.default_rng(5)
    for trial in range(2):
        xs = rng.uniform(-1, 1, 3)
        xd = xs + rng.uniform(0.8, 1.5) * _unit(rng)
        pt = xd + 0.08 * _unit(rng)
        xi = tr.xi_matrix(12, K, xd - xs)                  # d = x_dest - x_source (R3)
        assert _addition_error(xi, 3, 12, xs, xd, pt) < 1e-10
        # regular -> regular translation (j_q), valid everywhere
        xr = tr.xi_matrix(12, K, xd - xs, regular=True)
        assert _addition_error(xr, 3, 12, xs, xd, pt, regular_lhs=True) < 1e-10
        # the other direction (text of Eq. I15) must fail
        xw = tr.xi_matrix(12, K, xs - xd)
        assert _addition_error(xw, 3, 12, xs, xd, pt) > 1e-2


def test_addition_theorem_pointwise_source_rows_to_lmax6():
    """Entries with BOTH l >= 4 and l' >= 4 (Eqs. I16-I18; the paper's truncation is lmax = 6,
    PAPER.md:271): every source row l <= 6 of the translation matrix, expanded over destination columns l' <= 14,
    must reproduce the outgoing wavefunction pointwise.  The entries (l, l') in [4, 6]^2 carry 1.5e-2 of a row's
    value at this distance (asserted below), so a slip in a5 / b5 / the 3j symbols at high order fails the 1e-11 bound."""
    rng = np.random.default_rng(55)
    xs = rng.uniform(-1, 1, 3)
    xd = xs + 0.9 * _unit(rng)
    pt = xd + 0.05 * _unit(rng)
    xi = tr.xi_matrix(14, K, xd - xs)
    assert _addition_error(xi, 6, 14, xs, xd, pt) < 1e-11
    # the high-order entries matter: zeroing the block l, l' in [4, 6] must break it
    big = mode_list(14)
    hi = np.array([4 <= l <= 6 for (l, m, p) in big])
    xz = xi.copy()
    xz[np.ix_(hi, hi)] = 0.0
    assert _addition_error(xz, 6, 14, xs, xd, pt) > 1e-3
    xr = tr.xi_matrix(14, K, xd - xs, regular=True)
    assert _addition_error(xr, 6, 14, xs, xd, pt, regular_lhs=True) < 1e-11


def _unit(rng):
    v = rng.standard_normal(3)
    return v / np.linalg.norm(v)


def test_printed_forms_fail():
    # R5: printed normalisation is off by sqrt(l'); R6: printed b5 (second 3j with q, not q-1) vanishes
    from oracle.wigner import wigner_3j
    for l, lp, q in [(1, 2, 2), (2, 3, 2), (3, 3, 5)]:
        assert (l + lp + q) % 2 == 1
        assert wigner_3j(l, lp, q, 0, 0, 0) == 0.0
        assert abs(tr.b5(l, 1, lp, 1, q)) > 0


def test_block_symmetries_S1_S2_S3_S4():
    rng = np.random.default_rng(6)
    for lmax in (2, 3, 4, 5, 6):
        L = n_modes(lmax)
        modes = mode_list(lmax)
        d = rng.uniform(0.6, 2.0) * _unit(rng)
        B = tr.block(lmax, K, d, np.zeros(3))
        Bm = tr.block(lmax, K, -d, np.zeros(3))
        Pi = np.diag([(-1.0) ** (l + p) for (l, m, p) in modes])
        assert np.abs(Bm - Pi @ B @ Pi).max() < 1e-13 * np.abs(B).max()            # S1
        perm = np.array([mode_index(l, -m, p, lmax) for (l, m, p) in modes])
        P = np.eye(L)[perm]
        assert np.abs(Bm.T - P @ B @ P).max() < 1e-13 * np.abs(B).max()            # S3
        Rg = tr.block(lmax, K, d, np.zeros(3), regular=True)
        Rgm = tr.block(lmax, K, -d, np.zeros(3), regular=True)
        assert np.abs(Rgm - Rg.conj().T).max() < 1e-13 * np.abs(Rg).max()          # S4: RgA_ij = RgA_ji^H
        Ng, Ngm = (B - Rg) / 1j, (Bm - Rgm) / 1j                                   # A = RgA + i NgA (y_q in place of j_q)
        assert np.abs(Ngm - Ng.conj().T).max() < 1e-13 * np.abs(Ng).max()          # S4b: NgA is Hermitian too, hence
        #      Re(s^H A s) = s^H RgA s for the assembled operator: C_sca needs only the OUTGOING matvec (full-size GPU check)
        # S2: coplanar sparsity counts
        dc = np.array([0.7, -0.4, 0.0])
        Bc = tr.block(lmax, K, dc, np.zeros(3))
        nz = int(np.sum(np.abs(Bc) > 1e-12 * np.abs(Bc).max()))
        if lmax <= 3:
            assert nz == {2: 124, 3: 442}[lmax]
        par = np.array([(-1) ** (l + m + p) for (l, m, p) in modes])
        assert np.all((np.abs(Bc) > 1e-12 * np.abs(Bc).max()) <= (par[:, None] == par[None, :]))
        # axial displacement couples only m = m'
        Ba = tr.block(lmax, K, np.array([0.0, 0.0, 0.9]), np.zeros(3))
        ms = np.array([m for (l, m, p) in modes])
        assert np.all((np.abs(Ba) > 1e-12 * np.abs(Ba).max()) <= (ms[:, None] == ms[None, :]))


def test_blocks_many_equals_literal_block():
    rng = np.random.default_rng(7)
    D = rng.uniform(-2, 2, (6, 3))
    D[0] = [0.5, 0.0, 0.0]
    D[1] = [0.0, 0.0, -0.7]
    for lmax in (1, 2, 3, 5, 6):
        Bm = tr.blocks_many(lmax, K, D)
        for t in range(len(D)):
            B = tr.block(lmax, K, D[t], np.zeros(3))
            assert np.abs(Bm[t] - B).max() < 1e-13 * np.abs(B).max()
        Rm = tr.blocks_many(lmax, K, D, regular=True)
        assert np.abs(Rm[2] - tr.block(lmax, K, D[2], np.zeros(3), regular=True)).max() < 1e-14
