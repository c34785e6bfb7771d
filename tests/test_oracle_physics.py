"""Pins for oracle/tmatrix.py, oracle/incident.py, oracle/system.py, oracle/fields.py, oracle/matvec.py.

Nothing here compares the oracle with itself through the same formula: Mie is checked against an
independently-written logarithmic-derivative form (mpmath), the Rayleigh limit and unitarity; the
plane-wave / Gaussian coefficients by reconstructing the field; the assembled solve by energy
conservation with an independent far-field quadrature, the N=1 limit, a hand-rolled LU and the
forward/adjoint bilinear identity; the C matvec against the dense assembly."""
import os

import mpmath as mp
import numpy as np
import pytest

from oracle import driver, fields, incident, matvec, system, tmatrix, vswf
from oracle.modes import mode_index, mode_list, n_modes
from paper_2107_09879_b200 import workloads as W

K = 2 * np.pi
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _mie_logderiv(l, x, m):
    """Bohren & Huffman Eqs. 4.88 (logarithmic-derivative form), in mpmath: independent of oracle.tmatrix's form."""
    mp.mp.dps = 30
    psi = lambda n, z: z * mp.sqrt(mp.pi / (2 * z)) * mp.besselj(n + 0.5, z)
    xi = lambda n, z: z * mp.sqrt(mp.pi / (2 * z)) * (mp.besselj(n + 0.5, z) + 1j * mp.bessely(n + 0.5, z))
    D = mp.diff(lambda z: mp.log(psi(l, z)), m * x)
    a = ((D / m + l / x) * psi(l, x) - psi(l - 1, x)) / ((D / m + l / x) * xi(l, x) - xi(l - 1, x))
    b = ((D * m + l / x) * psi(l, x) - psi(l - 1, x)) / ((D * m + l / x) * xi(l, x) - xi(l - 1, x))
    return complex(a), complex(b)


def test_mie_against_logderiv_form_unitarity_rayleigh():
    for R in (0.10, 0.2, 0.24):
        t = tmatrix.mie_tmatrix_diag(3, K, R, 4.0)
        assert np.allclose(np.abs(1 + 2 * t), 1.0, atol=1e-13)            # lossless: |S| = 1
        for (l, m, p) in mode_list(3):
            a, b = _mie_logderiv(l, K * R, 2.0)
            ref = -b if p == 0 else -a
            assert abs(t[mode_index(l, m, p, 3)] - ref) < 1e-12 * max(abs(ref), 1e-6)
    # Rayleigh limit: -a_1 -> i (2/3) x^3 (m^2-1)/(m^2+2): electric dipole is p = 1
    x = 1e-3
    t = tmatrix.mie_tmatrix_diag(1, 1.0, x, 4.0)
    ref = 1j * (2.0 / 3.0) * x ** 3 * (4.0 - 1.0) / (4.0 + 2.0)
    assert abs(t[mode_index(1, 0, 1, 1)] - ref) < 1e-5 * abs(ref)
    assert abs(t[mode_index(1, 0, 0, 1)]) < 1e-3 * abs(ref)               # magnetic dipole ~ x^5


def test_plane_wave_reconstruction():
    rng = np.random.default_rng(8)
    for beta, alpha in [(0.0, 0.0), (0.6, 1.1), (2.2, -0.7)]:
        Ab, Aa = 0.7 + 0.2j, -0.3 + 0.5j
        a = incident.plane_wave_coeffs(25, beta, alpha, Ab, Aa)
        x = rng.uniform(-0.25, 0.25, 3)
        E = a @ vswf.vswf_all(25, K, x, regular=True)
        bh = np.array([np.cos(beta) * np.cos(alpha), np.cos(beta) * np.sin(alpha), -np.sin(beta)])
        ah = np.array([-np.sin(alpha), np.cos(alpha), 0.0])
        kv = K * np.array([np.sin(beta) * np.cos(alpha), np.sin(beta) * np.sin(alpha), np.cos(beta)])
        assert np.abs(E - (Ab * bh + Aa * ah) * np.exp(1j * kv @ x)).max() < 1e-12
    # per-scatterer phase of Eq. II6
    pos = rng.uniform(-3, 3, (4, 3))
    p = incident.plane_wave_incident(8, K, pos, 0.6, 1.1, 1.0, 0.0)
    kv = K * np.array([np.sin(0.6) * np.cos(1.1), np.sin(0.6) * np.sin(1.1), np.cos(0.6)])
    for j in range(4):
        E = p[j] @ vswf.vswf_all(8, K, np.array([0.03, -0.02, 0.04]), regular=True)
        bh = np.array([np.cos(0.6) * np.cos(1.1), np.cos(0.6) * np.sin(1.1), -np.sin(0.6)])
        assert np.abs(E - bh * np.exp(1j * kv @ (pos[j] + [0.03, -0.02, 0.04]))).max() < 1e-9


def test_gaussian_beam_reconstruction_and_limits():
    w0, foc = 2.0, np.array([0.1, -0.2, 0.0])
    pos = np.array([[1.3, 0.4, 0.0], [0.1, -0.2, 0.0], [-0.6, 0.9, 0.35]])
    a = incident.gaussian_beam_incident(12, K, pos, foc, w0, 1.0, 0.3j)
    for j in range(3):
        pt = pos[j] + np.array([0.1, 0.05, -0.03])
        E = a[j] @ vswf.vswf_all(12, K, pt - pos[j], regular=True)
        ref = incident.gaussian_beam_field_direct(K, pt, foc, w0, 1.0, 0.3j)      # 2-D quadrature of Eq. II4
        assert np.abs(E - ref).max() < 1e-9
    # on the focal plane the transverse field is the Gaussian profile itself
    pt = np.array([1.4, 0.45, 0.0])
    E = a[0] @ vswf.vswf_all(12, K, pt - pos[0], regular=True)
    g = np.exp(-np.sum((pt - foc)[:2] ** 2) / w0 ** 2)
    assert abs(E[0] - g) < 1e-9 and abs(E[1] - 0.3j * g) < 1e-9
    # w0 -> infinity: plane wave along +z
    big = incident.gaussian_beam_incident(3, K, np.array([[0.3, 0.2, 0.1]]), np.zeros(3), 4000.0, 1.0, 0.0, n_beta=200)
    pw = incident.plane_wave_incident(3, K, np.array([[0.3, 0.2, 0.1]]), 0.0, 0.0, 1.0, 0.0)
    assert np.abs(big - pw).max() < 1e-6


def _farfield_csca(lmax, k, pos, s, n_th=48, n_ph=96):
    """Independent C_sca: integrate |E_sca|^2 r^2 over a large sphere by quadrature."""
    r = 4.0e4
    xg, wg = np.polynomial.legendre.leggauss(n_th)
    ph = 2 * np.pi * np.arange(n_ph) / n_ph
    tot = 0.0
    for ct, wt in zip(xg, wg):
        st = np.sqrt(1 - ct * ct)
        pts = r * np.stack([st * np.cos(ph), st * np.sin(ph), np.full_like(ph, ct)], axis=1)
        E = fields.e_sca(lmax, k, pos, s, pts)
        tot += wt * (2 * np.pi / n_ph) * np.sum(np.abs(E) ** 2) * r * r
    return tot


def test_single_sphere_is_mie_and_textbook_extinction():
    w = dict(W.config(1), pos=np.zeros((1, 3)), type_of=np.zeros(1, dtype=np.int32),
             win_ptr=np.array([0, 1], dtype=np.int32), lmax=3)
    out = driver.solve(w)
    t = tmatrix.mie_tmatrix_diag(3, K, 0.2, 4.0)
    assert np.abs(out["s"][0] - t * out["p"][0]).max() < 1e-15
    cext, csca = fields.cross_sections(3, K, w["pos"], out["s"], out["p"])
    ab = [_mie_logderiv(l, K * 0.2, 2.0) for l in (1, 2, 3)]
    textbook = 2 * np.pi / K ** 2 * sum((2 * l + 1) * (ab[l - 1][0] + ab[l - 1][1]).real for l in (1, 2, 3))
    assert abs(cext - textbook) < 1e-13 and abs(csca - textbook) < 1e-13
    assert abs(_farfield_csca(3, K, w["pos"], out["s"], 16, 32) - textbook) < 1e-6 * textbook


def test_energy_conservation_general_positions_and_farfield():
    w = W.cloud_workload(3, seed=11, lmax=3)
    out = driver.solve(w)
    cext, csca = fields.cross_sections(3, K, w["pos"], out["s"], out["p"])
    # |A|^2 = |A_beta|^2 + |A_alpha|^2 normalises both
    amp2 = abs(w["A_beta"]) ** 2 + abs(w["A_alpha"]) ** 2
    assert abs(cext - csca) < 1e-12 * abs(cext)                      # lossless T: extinction = scattering (R7 sign)
    ff = _farfield_csca(3, K, w["pos"], out["s"])
    assert abs(ff - csca) < 2e-5 * csca                              # formula O9 vs direct far-field quadrature
    assert cext / amp2 > 0


def test_wrong_sign_breaks_energy_conservation():
    w = W.cloud_workload(4, seed=12, lmax=2)
    t, type_of, diag = driver.tmatrices(w)
    p = driver.incident_coeffs(w)
    A = system.assemble_A(2, K, w["pos"])
    Mbad = np.eye(A.shape[0]) + (t[type_of].reshape(-1)[:, None] * A)            # "+xi^T" as printed in Eq. I23
    sbad = np.linalg.solve(Mbad, (t[type_of] * p).reshape(-1)).reshape(p.shape)
    cext, csca = fields.cross_sections(2, K, w["pos"], sbad, p)
    assert abs(cext - csca) > 1e-3 * abs(cext)


def test_two_far_spheres_decouple():
    pos = np.array([[0.0, 0.0, 0.0], [400.0, 90.0, -250.0]])
    w = dict(W.config(1), pos=pos, type_of=np.zeros(2, dtype=np.int32), win_ptr=np.array([0, 2], dtype=np.int32))
    out = driver.solve(w)
    t = tmatrix.mie_tmatrix_diag(2, K, 0.2, 4.0)
    iso = t * out["p"]
    rel = np.abs(out["s"] - iso).max() / np.abs(iso).max()
    assert 1e-6 < rel < 5.0 / (K * np.linalg.norm(pos[1]))          # O(1/kr) correction


def test_cfg1_golden_values():
    """Config 1 (BASELINE.json): values written by tests/golden/make_golden.py from oracle/ only, and the
    independent survey-session values quoted in SURVEY.md 8(c) ("[scratch] reference values for config 1")."""
    w = W.config(1)
    out = driver.solve(w)
    cext, csca = fields.cross_sections(2, K, w["pos"], out["s"], out["p"])
    gold = dict(l.split("=") for l in open(os.path.join(GOLD, "cfg1_scalars.txt")) if "=" in l and not l.startswith("#"))
    assert abs(cext - float(gold["C_ext"])) < 1e-11 and abs(np.linalg.norm(out["s"]) - float(gold["norm_s"])) < 1e-11
    assert abs(cext - 2.85139402475) < 5e-11 and abs(csca - 2.85139402475) < 5e-11     # SURVEY.md:459
    assert abs(np.linalg.norm(out["s"]) - 5.85633350965) < 5e-11                          # SURVEY.md:459
    assert abs(np.linalg.cond(out["M"]) - 12.5) < 0.06                                     # SURVEY.md:459


def test_lu_handrolled_and_adjoint_identity_and_reciprocity():
    w = W.cloud_workload(5, seed=13, lmax=2, full_t=True)
    L = n_modes(2)
    rng = np.random.default_rng(14)
    wv = W.complex_normal((5, L), rng)
    out = driver.solve(w, adjoint_w=wv)
    t, type_of, diag = driver.tmatrices(w)
    b = system.apply_T(t, type_of, out["p"], diag).reshape(-1)
    assert np.abs(system.lu_solve_plain(out["M"], b) - out["s"].reshape(-1)).max() < 1e-12
    # bilinear identity: lambda^T (T p) = w^T s
    assert abs(out["lam"].reshape(-1) @ b - wv.reshape(-1) @ out["s"].reshape(-1)) < 1e-12 * abs(wv.reshape(-1) @ out["s"].reshape(-1))
    # reciprocity for Mie (reciprocal) T: Omega^T = P Omega P, Omega = T^{-1} - A  <=>  (T A)^T-structure: A^T = P A P
    w2 = W.cloud_workload(4, seed=15, lmax=2)
    A = system.assemble_A(2, K, w2["pos"])
    perm1 = np.array([mode_index(l, -m, p, 2) for (l, m, p) in mode_list(2)])
    perm = (np.arange(4)[:, None] * L + perm1[None, :]).reshape(-1)
    assert np.abs(A.T - A[np.ix_(perm, perm)]).max() < 1e-13 * np.abs(A).max()


def test_windows_are_independent():
    w = W.cloud_workload(9, seed=16, lmax=2, n_win=3)
    out = driver.solve(w)
    wp = w["win_ptr"]
    for iw in range(3):
        sl = slice(wp[iw], wp[iw + 1])
        sub = dict(w, pos=w["pos"][sl], radii=w["radii"][sl], type_of=np.arange(wp[iw + 1] - wp[iw], dtype=np.int32),
                   win_ptr=np.array([0, wp[iw + 1] - wp[iw]], dtype=np.int32))
        assert np.abs(driver.solve(sub)["s"] - out["s"][sl]).max() < 1e-13


def test_c_matvec_against_dense():
    rng = np.random.default_rng(17)
    for lmax, n, nw in [(1, 12, 1), (2, 30, 2), (3, 40, 3), (4, 14, 2), (5, 10, 1), (6, 9, 2)]:
        w = W.cloud_workload(n, seed=18 + lmax, lmax=lmax, n_win=nw)
        L = n_modes(lmax)
        x = W.complex_normal((n, L), rng)
        A = system.assemble_A(lmax, K, w["pos"], list(w["win_ptr"]))
        u = (A @ x.reshape(-1)).reshape(n, L)
        u2 = matvec.matvec_rows(lmax, K, w["pos"], x, win_ptr=w["win_ptr"])
        assert np.abs(u - u2).max() < 1e-13 * np.abs(u).max()
        rows = np.array([3, 0, n - 1], dtype=np.int32)
        assert np.abs(matvec.matvec_rows(lmax, K, w["pos"], x, rows=rows, win_ptr=w["win_ptr"]) - u[rows]).max() < 1e-13 * np.abs(u).max()
    # lattice (coplanar, exact pitch multiples) as in the configs
    w = W.config(2, scale=6)
    x = W.complex_normal((36, 30), rng)
    A = system.assemble_A(3, K, w["pos"])
    assert np.abs((A @ x.reshape(-1)).reshape(36, 30) - matvec.matvec_rows(3, K, w["pos"], x)).max() < 1e-12


def test_H_field_is_the_curl_of_E():
    """Pin of oracle/fields.py::zh_sca (reading R10; PAPER.md:284 Eq. I13 with curl Phi_p = k Phi_{1-p}, PAPER.md:230-234
    Eq. I6b): Maxwell's curl E = i omega mu H = i k (Z_b H), with the curl of the ORACLE's own e_sca taken numerically
    (4th-order central differences) near a 3-scatterer cloud.  A wrong sign of the -i, a missing p <-> 1-p swap, or a
    wrong sum fails it."""
    rng = np.random.default_rng(41)
    lmax = 3
    L = n_modes(lmax)
    pos = np.array([[0.0, 0.0, 0.0], [0.7, 0.2, -0.3], [-0.4, 0.8, 0.5]])
    s = W.complex_normal((3, L), rng)
    h = 2e-3

    def curl_E(x):
        J = np.zeros((3, 3), dtype=complex)          # J[a, b] = d E_a / d x_b
        for b in range(3):
            e = np.zeros(3)
            e[b] = h
            f = lambda t: fields.e_sca(lmax, K, pos, s, x + t * e)[0]
            J[:, b] = (8 * (f(1) - f(-1)) - (f(2) - f(-2))) / (12 * h)
        return np.array([J[2, 1] - J[1, 2], J[0, 2] - J[2, 0], J[1, 0] - J[0, 1]])

    swap = np.concatenate([np.arange(L // 2, L), np.arange(0, L // 2)])
    for _ in range(4):
        x = rng.uniform(-1.5, 1.5, 3) + np.array([0.3, -0.2, 1.9])
        zh = fields.zh_sca(lmax, K, pos, s, x)[0]
        ref = curl_E(x) / (1j * K)
        scale = np.abs(ref).max()
        assert np.abs(zh - ref).max() < 1e-6 * scale
        assert np.abs(-zh - ref).max() > 0.5 * scale                      # the +i variant fails
        # without the p <-> 1-p swap (-i sum s Phi_{lmp} = -i E) it fails too
        assert np.abs(-1j * fields.e_sca(lmax, K, pos, s, x)[0] - ref).max() > 1e-2 * scale
        # and it is the same sum as E with the coefficient halves exchanged: Z H[s] = -i E[s with p <-> 1-p]
        assert np.abs(zh + 1j * fields.e_sca(lmax, K, pos, s[:, swap], x)[0]).max() < 1e-13 * scale
