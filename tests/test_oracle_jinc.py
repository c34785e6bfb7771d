"""Pins of the oracle's jinc sources and Nyquist decomposition (reading R17)."""
import numpy as np
import pytest
from scipy.special import j1

from oracle import incident, vswf

K = 2 * np.pi


def test_jinc_source_reconstruction_closed_form_and_direct_quadrature():
    src = np.array([0.2, -0.1, -1.0])
    pos = np.array([[0.5, 0.3, -1.0], [-0.4, 0.8, 0.6]])
    a = incident.jinc_source_incident(12, K, pos, src, 1.0, 0.4j)
    # on the source plane z = z_0 the transverse field is A^T J_1(k rho)/(k rho)  (Eq. II3 with k_0^2 dropped)
    pt = pos[0] + np.array([0.08, -0.05, 0.0])
    E = a[0] @ vswf.vswf_all(12, K, pt - pos[0], regular=True)
    rho = K * np.hypot(*(pt - src)[:2])
    assert abs(E[0] - j1(rho) / rho) < 1e-9 and abs(E[1] - 0.4j * j1(rho) / rho) < 1e-9
    # off the source plane: direct 2-D quadrature of Eq. II4
    for j in range(2):
        pt = pos[j] + np.array([0.1, 0.05, -0.03])
        E = a[j] @ vswf.vswf_all(12, K, pt - pos[j], regular=True)
        ref = incident.jinc_field_direct(K, pt, src, 1.0, 0.4j)
        assert np.abs(E - ref).max() < 1e-8
    # centre value of the unit source: J_1(x)/x -> 1/2
    c = incident.jinc_source_incident(8, K, src[None, :], src, 1.0, 0.0)
    E0 = c[0] @ vswf.vswf_all(8, K, np.array([1e-3, 0.0, 0.0]), regular=True)
    assert abs(E0[0] - 0.5) < 1e-5


def test_nyquist_decomposition_reproduces_a_band_limited_beam():
    """sum_ij (pi/2) E(x_i, y_j) jinc_ij = E for a field inside the light cone: a Gaussian beam (w0 = 1.2 lambda, spectrum
    < 1e-6 at the light-cone edge) rebuilt from its lambda/2 samples gives the Gaussian-beam coefficients."""
    w0, lmax = 1.2, 3
    pos = np.array([[0.3, -0.2, 0.5], [-0.7, 0.4, 0.0]])
    direct = incident.gaussian_beam_incident(lmax, K, pos, np.zeros(3), w0, 1.0, 0.0)
    src, amp = incident.nyquist_sources(K, (-4.0, 4.0), (-4.0, 4.0), 0.0,
                                        lambda x, y: (np.exp(-(x * x + y * y) / w0 ** 2), np.zeros_like(x)))
    keep = np.abs(amp[:, 0]) > 1e-9
    rebuilt = incident.jinc_sources_incident(lmax, K, pos, src[keep], amp[keep], n_beta=200)
    assert np.abs(rebuilt - direct).max() < 2e-5 * np.abs(direct).max()


def test_nyquist_constant_is_not_one():
    """Without the (pi/2) of reading R17 the reconstruction is off by that factor (pins the constant)."""
    assert incident.nyquist_source_amplitude(1.0) == pytest.approx(np.pi / 2)
