"""Incident-field expansion coefficients a^(0) (TEST INFRASTRUCTURE ONLY - see oracle/__init__.py).

Plane wave: PAPER.md:425-432, Eqs. II6-II7, using the explicit right-hand forms (reading R9b):
    a_{l,m,0}(beta,alpha) = -4 i^l     e^{-i m alpha} c_l [ i m pibar (beta_hat.A) + taubar (alpha_hat.A) ]
    a_{l,m,1}(beta,alpha) = -4 i^{l+1} e^{-i m alpha} c_l [ taubar (beta_hat.A) - i m pibar (alpha_hat.A) ]
    c_l = [2l(l+1)]^{-1/2},  pibar = pibar_l^{|m|}(beta), taubar = taubar_l^{|m|}(beta),
and for a scatterer at x_j the coefficients pick up exp(i k . x_j)  (Eq. II6 with x_0' = x_j, x_0 = origin).

Beam with a given angular spectrum: PAPER.md:441-486, Eqs. II9-II17 (alpha integral in closed form,
Eq. II11; beta integral numeric).  The paper does this for a flat spectrum (jinc source); the
Gaussian beam of BASELINE.json's configs 3 and 4 is reading R9: the same integrand times
    G(beta) = (k w0)^2 / 2 * exp(-(k w0 sin beta)^2 / 4),
i.e. transverse field A^T exp(-|x^T - x_0^T|^2 / w0^2) on the focal plane z = z_0, evanescent part dropped.
"""
from math import sqrt

import numpy as np
from scipy.special import jv

from . import special as sp
from .modes import mode_list, n_modes
from .vswf import cart_to_sph


def plane_wave_coeffs(lmax, beta, alpha, A_beta, A_alpha):
    """Eq. II7 for a plane wave travelling along (beta, alpha) with amplitude
    A = A_beta beta_hat + A_alpha alpha_hat, expanded about the origin.  Shape (L,)."""
    out = np.zeros(n_modes(lmax), dtype=complex)
    for idx, (l, m, p) in enumerate(mode_list(lmax)):
        c = 1.0 / sqrt(2.0 * l * (l + 1))
        pi_ = float(sp.pibar(l, abs(m), beta))
        tau = float(sp.taubar(l, abs(m), beta))
        e = np.exp(-1j * m * alpha)
        if p == 0:
            out[idx] = -4.0 * (1j) ** l * e * c * (1j * m * pi_ * A_beta + tau * A_alpha)
        else:
            out[idx] = -4.0 * (1j) ** (l + 1) * e * c * (tau * A_beta - 1j * m * pi_ * A_alpha)
    return out


def plane_wave_incident(lmax, k, pos, beta, alpha, A_beta, A_alpha):
    """a^(0)_j for every scatterer (Eq. II6): (N, L)."""
    pos = np.asarray(pos, dtype=float)
    a = plane_wave_coeffs(lmax, beta, alpha, A_beta, A_alpha)
    kvec = k * np.array([np.sin(beta) * np.cos(alpha), np.sin(beta) * np.sin(alpha), np.cos(beta)])
    return np.exp(1j * pos @ kvec)[:, None] * a[None, :]


def gamma_m(m, xi, eta, rho):
    """Eq. II11."""
    return ((1j) ** ((m - 1) % 4) * np.exp(-1j * m * xi) / 2.0
            * (np.exp(1j * (xi - eta)) * jv(m - 1, rho) - np.exp(-1j * (xi - eta)) * jv(m + 1, rho)))


def _alpha_integrated(l, m, p, k, rel, beta, Ax, Ay):
    """Right-hand sides of Eq. II15 (p=0) / II17 (p=1) for rel = x_0' - x_0 = scatterer - focus."""
    r0, th0, ph0 = cart_to_sph(rel)
    c = 1.0 / sqrt(2.0 * l * (l + 1))
    pi_ = sp.pibar(l, abs(m), beta)
    tau = sp.taubar(l, abs(m), beta)
    cb, sb = np.cos(beta), np.sin(beta)
    rho = k * r0 * sb * np.sin(th0)
    g0 = gamma_m(m, ph0, 0.0, rho)
    g1 = gamma_m(m, ph0, np.pi / 2, rho)
    ez = np.exp(1j * k * r0 * cb * np.cos(th0))
    if p == 0:
        return (-4.0 * (1j) ** l * ez * sb * c
                * ((1j * m * pi_ * Ax + tau * cb * Ay) * g0 + (1j * m * pi_ * Ay - tau * cb * Ax) * g1))
    return (-4.0 * (1j) ** (l + 1) * ez * sb * c
            * ((tau * Ax - 1j * m * pi_ * Ay * cb) * g0 + (tau * Ay + 1j * m * pi_ * Ax * cb) * g1))


def gaussian_beam_incident(lmax, k, pos, focus, w0, Ax, Ay, n_beta=400):
    """a^(0)_j for a Gaussian beam along +z focused at `focus` (reading R9): (N, L).
    Gauss-Legendre in beta on [0, beta_max], beta_max chosen where G(beta) < 1e-40 (or pi/2)."""
    pos = np.atleast_2d(np.asarray(pos, dtype=float))
    focus = np.asarray(focus, dtype=float)
    kw = k * w0
    smax = min(1.0, 2.0 * sqrt(40.0 * np.log(10.0)) / kw)
    bmax = np.arcsin(smax)
    xg, wg = np.polynomial.legendre.leggauss(n_beta)
    beta = 0.5 * bmax * (xg + 1.0)
    wq = 0.5 * bmax * wg
    G = kw * kw / 2.0 * np.exp(-(kw * np.sin(beta)) ** 2 / 4.0)
    out = np.zeros((pos.shape[0], n_modes(lmax)), dtype=complex)
    for j in range(pos.shape[0]):
        rel = pos[j] - focus
        for idx, (l, m, p) in enumerate(mode_list(lmax)):
            out[j, idx] = np.sum(wq * G * _alpha_integrated(l, m, p, k, rel, beta, Ax, Ay))
    return out


def gaussian_beam_field_direct(k, x, focus, w0, Ax, Ay, n_beta=200, n_alpha=256):
    """Direct 2-D quadrature of Eq. II4 with the Gaussian spectrum (pin for gaussian_beam_incident)."""
    x = np.asarray(x, dtype=float) - np.asarray(focus, dtype=float)
    kw = k * w0
    smax = min(1.0, 2.0 * sqrt(40.0 * np.log(10.0)) / kw)
    bmax = np.arcsin(smax)
    xg, wg = np.polynomial.legendre.leggauss(n_beta)
    beta = 0.5 * bmax * (xg + 1.0)
    wb = 0.5 * bmax * wg
    alpha = 2 * np.pi * np.arange(n_alpha) / n_alpha
    B, Al = np.meshgrid(beta, alpha, indexing="ij")
    G = kw * kw / 2.0 * np.exp(-(kw * np.sin(B)) ** 2 / 4.0)
    kx, ky, kz = k * np.sin(B) * np.cos(Al), k * np.sin(B) * np.sin(Al), k * np.cos(B)
    ph = np.exp(1j * (kx * x[0] + ky * x[1] + kz * x[2]))
    Az = -np.tan(B) * (Ax * np.cos(Al) + Ay * np.sin(Al))
    w = wb[:, None] * (2 * np.pi / n_alpha) * np.sin(B) * np.cos(B) * G * ph / (2 * np.pi)
    return np.array([np.sum(w * Ax), np.sum(w * Ay), np.sum(w * Az)])


# ------------------------------------------------------------------------------------------------ jinc sources (NEXT-1)
def jinc_source_incident(lmax, k, pos, src, Ax, Ay, n_beta=400):
    """a^(0)_j of ONE jinc source: flat angular spectrum inside the light cone, Eq. II3, centred at
    `src` = (x_0, y_0, z_0), transverse amplitude (Ax, Ay).  Eq. II9 with the alpha integral done in closed form
    (Eqs. II15 / II17) and Gauss-Legendre in beta on [0, pi/2] (n_beta nodes: part of the definition, as for reading R9).
    With Eq. II3 (and the k_0^2 of d^2k dropped in Eq. II9) the transverse field on the source plane is
        E^T(x^T, z_0) = A^T J_1(k_0 rho) / (k_0 rho),  rho = |x^T - x_0^T|     (cylindrical J_1; reading R17)."""
    pos = np.atleast_2d(np.asarray(pos, dtype=float))
    src = np.asarray(src, dtype=float)
    xg, wg = np.polynomial.legendre.leggauss(n_beta)
    beta = 0.25 * np.pi * (xg + 1.0)
    wq = 0.25 * np.pi * wg
    out = np.zeros((pos.shape[0], n_modes(lmax)), dtype=complex)
    for j in range(pos.shape[0]):
        rel = pos[j] - src
        for idx, (l, m, p) in enumerate(mode_list(lmax)):
            out[j, idx] = np.sum(wq * _alpha_integrated(l, m, p, k, rel, beta, Ax, Ay))
    return out


def jinc_field_direct(k, x, src, Ax, Ay, n_beta=300, n_alpha=512):
    """Direct 2-D quadrature of Eq. II4 with the flat spectrum (pin for jinc_source_incident), k_0^2 dropped as in II9."""
    x = np.asarray(x, dtype=float) - np.asarray(src, dtype=float)
    xg, wg = np.polynomial.legendre.leggauss(n_beta)
    beta = 0.25 * np.pi * (xg + 1.0)
    wb = 0.25 * np.pi * wg
    alpha = 2 * np.pi * np.arange(n_alpha) / n_alpha
    B, Al = np.meshgrid(beta, alpha, indexing="ij")
    kx, ky, kz = k * np.sin(B) * np.cos(Al), k * np.sin(B) * np.sin(Al), k * np.cos(B)
    ph = np.exp(1j * (kx * x[0] + ky * x[1] + kz * x[2]))
    Az = -np.tan(B) * (Ax * np.cos(Al) + Ay * np.sin(Al))
    w = wb[:, None] * (2 * np.pi / n_alpha) * np.sin(B) * np.cos(B) * ph / (2 * np.pi)
    return np.array([np.sum(w * Ax), np.sum(w * Ay), np.sum(w * Az)])


def nyquist_source_amplitude(E_sample):
    """Amplitude of the jinc source that carries the Nyquist sample E^T(x_i, y_j) (Eq. II1; reading R17).
    For a field band-limited to the light cone and sampled on the square grid of pitch lambda/2 = pi/k_0 the
    reconstruction kernel is the ideal disc low-pass
        f(rho) = (pi/k_0)^2 / (2 pi)^2 * int_{|k|<k_0} e^{i k.rho} d^2k = (pi/2) J_1(k_0 rho)/(k_0 rho),
    i.e. (pi/2) times the unit jinc source of jinc_source_incident (Eq. II1 prints the kernel without the constant)."""
    return 0.5 * np.pi * np.asarray(E_sample)


def nyquist_sources(k, x_range, y_range, z0, field_fn):
    """Sample a transverse field field_fn(x, y) -> (Ex, Ey) on the lambda/2 grid covering the ranges:
    returns (src (S,3), amp (S,2)) with amp the jinc-source amplitudes."""
    h = np.pi / k
    ix = np.arange(int(np.ceil(x_range[0] / h)), int(np.floor(x_range[1] / h)) + 1)
    iy = np.arange(int(np.ceil(y_range[0] / h)), int(np.floor(y_range[1] / h)) + 1)
    X, Y = np.meshgrid(ix * h, iy * h, indexing="xy")
    src = np.stack([X.ravel(), Y.ravel(), np.full(X.size, float(z0))], axis=1)
    Ex, Ey = field_fn(src[:, 0], src[:, 1])
    amp = np.stack([nyquist_source_amplitude(Ex), nyquist_source_amplitude(Ey)], axis=1).astype(complex)
    return src, amp


def jinc_sources_incident(lmax, k, pos, src, amp, n_beta=400):
    """Superposition of jinc sources: sum_s jinc_source_incident(..., src[s], amp[s,0], amp[s,1])."""
    out = np.zeros((np.atleast_2d(pos).shape[0], n_modes(lmax)), dtype=complex)
    for s in range(len(src)):
        out += jinc_source_incident(lmax, k, pos, src[s], amp[s, 0], amp[s, 1], n_beta)
    return out
