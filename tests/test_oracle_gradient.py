"""Pin of the adjoint sensitivity (Appendix IV, Eqs. IV8-IV9): one adjoint solve reproduces the numerical
derivative of the full solve with respect to every radius."""
import numpy as np

from oracle import gradient, incident
from paper_2107_09879_b200 import workloads as W

K = W.K_B


def test_adjoint_radius_gradient_matches_finite_differences():
    rng = np.random.default_rng(12)
    pos = W.random_cloud(5, seed=4)
    radii = rng.uniform(0.10, 0.22, 5)
    p = incident.plane_wave_incident(2, K, pos, 0.3, 0.8, 1.0, 0.4j)
    v = rng.standard_normal(p.shape) + 1j * rng.standard_normal(p.shape)
    g, s, lam = gradient.adjoint_radius_gradient(2, K, pos, radii, 4.0, p, v)
    for j in range(5):
        fd = gradient.fd_radius(2, K, pos, radii, 4.0, p, v, j)
        assert abs(g[j] - fd) <= 2e-7 * abs(fd)
    # a dropped A s term (using a^(0) only) is caught
    from oracle import tmatrix
    dT = np.stack([gradient.mie_dT_dR(2, K, r, 4.0) for r in radii])
    wrong = np.sum(lam * dT * p, axis=1)
    assert np.abs(wrong - g).max() > 1e-3 * np.abs(g).max()


def test_adjoint_position_gradient_matches_finite_differences():
    rng = np.random.default_rng(21)
    pos = W.random_cloud(4, seed=6)
    radii = rng.uniform(0.12, 0.2, 4)
    inc = lambda q: incident.plane_wave_incident(2, K, q, 0.4, -0.5, 0.7, 0.2j)
    v = rng.standard_normal((4, 16)) + 1j * rng.standard_normal((4, 16))
    g, s, lam = gradient.adjoint_position_gradient(2, K, pos, radii, 4.0, inc, v)
    for (j, a) in ((0, 0), (1, 2), (3, 1)):
        fd = gradient.fd_position(2, K, pos, radii, 4.0, inc, v, j, a)
        assert abs(g[j, a] - fd) <= 1e-6 * np.abs(g).max()
    # exact incident derivative of a plane wave (d a_j / d x_j = i k a_j) instead of its central difference
    kv = K * np.array([np.sin(0.4) * np.cos(-0.5), np.sin(0.4) * np.sin(-0.5), np.cos(0.4)])
    g2, _, _ = gradient.adjoint_position_gradient(2, K, pos, radii, 4.0, inc, v, dinc_fn=lambda q: 1j * kv[None, :, None] * inc(q)[:, None, :])
    assert np.abs(g2 - g).max() <= 1e-8 * np.abs(g).max()


def test_analytic_translation_derivative_matches_central_differences():
    """Pin of oracle/translation.py::d_xi_matrix: the analytic gradient of the translation
    coefficients against 4th-order central differences of xi_matrix itself, for a general displacement, the two polar
    directions (phi undefined, pibar limit), a coplanar one, and the regular (j_q) variant; lmax up to 6 (the paper's
    truncation).  A wrong sign of any of the three spherical components, a missing 1/r or a wrong h_q' fails it."""
    from oracle import translation as tr
    rng = np.random.default_rng(31)
    cases = [(3, rng.uniform(-1, 1, 3) + 0.3), (3, np.array([0.0, 0.0, 0.9])), (3, np.array([0.0, 0.0, -0.7])),
             (3, np.array([0.6, -0.3, 0.0])), (6, np.array([0.5, 0.4, -0.6])), (4, np.array([-0.7, 0.2, 0.0]))]
    h = 1e-4
    for lmax, d in cases:
        for regular in ((False, True) if lmax == 3 else (False,)):
            an = tr.d_xi_matrix(lmax, K, d, regular)
            f = lambda x: tr.xi_matrix(lmax, K, x, regular)
            for al in range(3):
                e = np.zeros(3)
                e[al] = h
                fd = (8 * (f(d + e) - f(d - e)) - (f(d + 2 * e) - f(d - 2 * e))) / (12 * h)
                assert np.abs(an[al] - fd).max() <= 1e-8 * np.abs(fd).max(), (lmax, d, al)
    # d_block: destination rows, source columns, d = x_dst - x_src; moving the SOURCE flips the sign
    xd, xs = np.array([0.2, 0.5, -0.1]), np.array([-0.4, 0.1, 0.6])
    an = tr.d_block(2, K, xd, xs)
    e = np.array([0.0, h, 0.0])
    assert np.abs(an[1] - (tr.block(2, K, xd + e, xs) - tr.block(2, K, xd - e, xs)) / (2 * h)).max() <= 1e-6 * np.abs(an[1]).max()
    assert np.abs(an[1] + (tr.block(2, K, xd, xs + e) - tr.block(2, K, xd, xs - e)) / (2 * h)).max() <= 1e-6 * np.abs(an[1]).max()


def test_shape_parameter_derivative_reduces_to_the_mie_radius_derivative():
    """fd_shape_parameter with spheres as the bodies of revolution = fd_radius with the closed-form Mie T-matrix (two
    independent routes to T: null-field surface integrals vs. Lorenz-Mie)."""
    rng = np.random.default_rng(3)
    pos = W.random_cloud(3, seed=9)
    radii = np.array([0.12, 0.2, 0.16])
    p = incident.plane_wave_incident(2, K, pos, 0.2, 0.1, 1.0, 0.0)
    v = rng.standard_normal(p.shape) + 1j * rng.standard_normal(p.shape)
    fn = lambda r: W.generatrix_sphere(r, 32)                  # noqa: E731
    for j in range(3):
        a = gradient.fd_shape_parameter(2, K, pos, fn, radii, np.arange(3), 4.0, p, v, j, h=1e-6)
        b = gradient.fd_radius(2, K, pos, radii, 4.0, p, v, j, h=1e-6)
        assert abs(a - b) <= 1e-6 * abs(b)
