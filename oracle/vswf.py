"""Vector spherical wavefunctions (TEST INFRASTRUCTURE ONLY - see oracle/__init__.py).

PAPER.md:213-236, Eqs. I3 and I6:
    phi_{l,m}(k x)   = z_l(kr) Pbar_l^{|m|}(cos theta) exp(i m phi),  z_l = h_l^(1) or j_l (regular, "R")
    Phi_{l,m,p=0}    = [2l(l+1)]^{-1/2} grad(phi_{l,m}) x  x                      (I6a)
    Phi_{l,m,p=1}    = (1/k) curl Phi_{l,m,p=0}                                    (I6b)
Written out in spherical components (theta_hat x r_hat = -phi_hat, phi_hat x r_hat = theta_hat):
    Phi_{l,m,0} = c_l z_l(kr) [ i m pibar theta_hat - taubar phi_hat ] e^{i m phi}
    Phi_{l,m,1} = c_l { l(l+1) z_l(kr)/(kr) Pbar r_hat
                        + [kr z_l(kr)]'/(kr) ( taubar theta_hat + i m pibar phi_hat ) } e^{i m phi}
with c_l = [2l(l+1)]^{-1/2} and pibar, taubar evaluated at |m|.
The p=1 form is pinned numerically against (1/k) curl of the p=0 form in tests/test_oracle_vswf.py.
"""
from math import sqrt

import numpy as np

from . import special as sp
from .modes import mode_list, n_modes


def cart_to_sph(x):
    """x: (..., 3) -> r, theta (polar from +z), phi (azimuth)."""
    x = np.asarray(x, dtype=float)
    r = np.sqrt(np.sum(x * x, axis=-1))
    theta = np.arccos(np.clip(x[..., 2] / np.where(r > 0, r, 1.0), -1.0, 1.0))   # r = 0 -> theta = pi/2, unused
    phi = np.arctan2(x[..., 1], x[..., 0])
    return r, theta, phi


def sph_unit_vectors(theta, phi):
    st, ct, sf, cf = np.sin(theta), np.cos(theta), np.sin(phi), np.cos(phi)
    rh = np.stack([st * cf, st * sf, ct], axis=-1)
    th = np.stack([ct * cf, ct * sf, -st], axis=-1)
    ph = np.stack([-sf, cf, np.zeros_like(st)], axis=-1)
    return rh, th, ph


def vswf(l, m, p, k, x, regular=False):
    """Phi_{l,m,p}(k x) (or R Phi if regular) at points x (..., 3); returns Cartesian (..., 3) complex."""
    r, theta, phi = cart_to_sph(x)
    kr = k * r
    am = abs(m)
    c = 1.0 / sqrt(2.0 * l * (l + 1))
    e = np.exp(1j * m * phi)
    rh, th, ph = sph_unit_vectors(theta, phi)
    pi_ = sp.pibar(l, am, theta)
    tau = sp.taubar(l, am, theta)
    if p == 0:
        z = sp.sph_jn(l, kr) if regular else sp.sph_h1(l, kr)
        f_th = c * z * (1j * m * pi_) * e
        f_ph = c * z * (-tau) * e
        return f_th[..., None] * th + f_ph[..., None] * ph
    z = sp.sph_jn(l, kr) if regular else sp.sph_h1(l, kr)
    zd = sp.sph_jn_rd(l, kr) if regular else sp.sph_h1_rd(l, kr)
    pb = sp.pbar(l, am, np.cos(theta))
    f_r = c * l * (l + 1) * z / kr * pb * e
    f_th = c * zd * tau * e
    f_ph = c * zd * (1j * m * pi_) * e
    return f_r[..., None] * rh + f_th[..., None] * th + f_ph[..., None] * ph


def vswf_all(lmax, k, x, regular=False):
    """All L wavefunctions in flat order (reading R1): returns (L, ..., 3)."""
    return np.stack([vswf(l, m, p, k, x, regular) for (l, m, p) in mode_list(lmax)], axis=0)
