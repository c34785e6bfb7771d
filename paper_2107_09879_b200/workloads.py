"""Seeded synthetic inputs shared by the tests, bench.py and the oracle-side scripts.

This module holds NONE of the method's arithmetic (no special functions, no translation
coefficients, no T-matrix physics, no solver): only geometry, random draws and the bookkeeping
that names BASELINE.json's five configs (recipe: DESIGN.md "Input recipe").
The paper's own workloads are metalens layouts built from the authors' cylinder libraries
(PAPER.md:59, 63, 504), which are not available; these planar sub-wavelength-pitch lattices
stand in for them.  Wavelength 1, k_b = 2*pi, background vacuum.  numpy only.

A workload is a dict:
  lmax, k, pos (N,3) f64, win_ptr (n_win+1,) int32,
  t_kind: "mie_types"  -> radii (n_types,), eps_r, type_of (N,)          [diag T per type]
          "mie_sites"  -> radii (N,), eps_r, type_of = arange(N)         [diag T per site]
          "full_types" -> t_full (n_types, L, L) complex, type_of (N,)   [config 3 / 3b]
  inc_kind: "plane" -> beta, alpha, A_beta, A_alpha
            "gauss" -> focus (n_win,3), w0, Ax, Ay        (per window, +z propagation)
  tol, restart, max_iter, and for config 4 an adjoint weight vector w (N, L).
"""
import numpy as np

K_B = 2.0 * np.pi


def n_modes(lmax):
    return 2 * lmax * (lmax + 2)


def lattice(nx, ny, pitch=0.5, center=(0.0, 0.0), z=0.0):
    """site (ix, iy) -> index iy*nx + ix; centred on `center` in the plane z."""
    ix, iy = np.meshgrid(np.arange(nx), np.arange(ny), indexing="xy")
    x = (ix.ravel() - (nx - 1) / 2.0) * pitch + center[0]
    y = (iy.ravel() - (ny - 1) / 2.0) * pitch + center[1]
    return np.stack([x, y, np.full(x.shape, float(z))], axis=1)


def random_cloud(n, seed, min_sep=0.5, density=0.35, planar=False):
    """Non-lattice positions with a minimum separation (parity only; PAPER.md:375 uses random positions)."""
    rng = np.random.default_rng(seed)
    side = (n / density) ** (1.0 / (2 if planar else 3)) * min_sep * 1.6
    pts = []
    while len(pts) < n:
        c = rng.uniform(-side / 2, side / 2, 3)
        if planar:
            c[2] = 0.0
        if all(np.linalg.norm(c - q) >= min_sep for q in pts):
            pts.append(c)
    return np.array(pts)


def haar_unitary(n, rng):
    """Haar-random unitary: QR of a complex Ginibre matrix with the R-diagonal phase fix (reading R12)."""
    z = (rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))) / np.sqrt(2.0)
    q, r = np.linalg.qr(z)
    d = np.diag(r)
    return q * (d / np.abs(d))[None, :]


def complex_normal(shape, rng):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def config(cfg, scale=None, seed=None):
    """BASELINE.json configs 1..5 (and "3b").  `scale` overrides the lattice side (reduced-size parity
    cases drawn from the same generator); `seed` defaults to the config number."""
    name = str(cfg)
    base = int(name[0])
    rng = np.random.default_rng(base if seed is None else seed)
    w = dict(name=f"cfg{name}" + (f"_n{scale}" if scale else ""), k=K_B, eps_r=4.0)
    if base == 1:
        n = scale or 4
        w.update(lmax=2, pos=lattice(n, n), t_kind="mie_types", radii=np.array([0.2]),
                 type_of=np.zeros(n * n, dtype=np.int32), inc_kind="plane", beta=0.0, alpha=0.0,
                 A_beta=1.0, A_alpha=0.0, tol=1e-10, restart=50, max_iter=2000)
    elif base == 2:
        n = scale or 32
        w.update(lmax=3, pos=lattice(n, n), t_kind="mie_types", radii=0.10 + 0.02 * np.arange(8),
                 type_of=rng.integers(0, 8, n * n).astype(np.int32), inc_kind="plane", beta=0.0, alpha=0.0,
                 A_beta=1.0, A_alpha=0.0, tol=1e-10, restart=50, max_iter=5000)
    elif base == 3:
        n = scale or 100
        L = n_modes(3)
        if name == "3":
            t_full = np.stack([(lambda U: (U @ U.T - np.eye(L)) / 2.0)(haar_unitary(L, rng)) for _ in range(16)])
        else:   # "3b": lossless, symmetric, physical l-envelope (labelled fallback)
            import scipy.linalg as sla
            env = np.array([(1.0, 0.35, 0.05)[l - 1] for p in (0, 1) for l in (1, 2, 3) for m in range(-l, l + 1)])
            t_full = []
            for _ in range(16):
                G = rng.standard_normal((L, L))
                H = env[:, None] * env[None, :] * (G + G.T) / 2.0
                t_full.append((sla.expm(1j * H) - np.eye(L)) / 2.0)
            t_full = np.stack(t_full)
        w.update(lmax=3, pos=lattice(n, n), t_kind="full_types", t_full=t_full,
                 type_of=rng.integers(0, 16, n * n).astype(np.int32), inc_kind="gauss",
                 focus=np.zeros((1, 3)), w0=10.0, Ax=1.0, Ay=0.0, tol=1e-10, restart=50, max_iter=3000)
    elif base == 4:
        n = scale or 64
        n_win = 64 if scale is None else 4
        side = int(round(np.sqrt(n_win)))
        span = n * 0.5 + 4.0
        centers = [((a - (side - 1) / 2.0) * span, (b - (side - 1) / 2.0) * span) for b in range(side) for a in range(side)]
        pos = np.concatenate([lattice(n, n, center=c) for c in centers])
        N = pos.shape[0]
        w.update(lmax=3, pos=pos, win_ptr=(np.arange(n_win + 1) * n * n).astype(np.int32), t_kind="mie_sites",
                 radii=rng.uniform(0.10, 0.24, N), type_of=np.arange(N, dtype=np.int32), inc_kind="gauss",
                 focus=np.array([[c[0], c[1], 0.0] for c in centers]), w0=2.0, Ax=1.0, Ay=0.0,
                 tol=1e-10, restart=50, max_iter=5000)
        w["w_adj"] = complex_normal((N, n_modes(3)), rng)
    elif base == 5:
        n = scale or 200
        w.update(lmax=3, pos=lattice(n, n), t_kind="mie_sites", radii=rng.uniform(0.10, 0.24, n * n),
                 type_of=np.arange(n * n, dtype=np.int32), inc_kind="plane", beta=0.0, alpha=0.0,
                 A_beta=1.0, A_alpha=0.0, tol=1e-8, restart=100, max_iter=20000)
    else:
        raise ValueError(cfg)
    w.setdefault("win_ptr", np.array([0, w["pos"].shape[0]], dtype=np.int32))
    return w


def cloud_workload(n, seed, lmax=3, planar=False, full_t=False, n_win=1):
    """Random non-lattice cloud with Mie sites (or full random-unitary-S types): parity cases only."""
    rng = np.random.default_rng(seed)
    pos = random_cloud(n, seed, planar=planar)
    L = n_modes(lmax)
    w = dict(name=f"cloud{n}_s{seed}", k=K_B, eps_r=4.0, lmax=lmax, pos=pos, inc_kind="plane", beta=0.4, alpha=1.1,
             A_beta=0.8, A_alpha=0.3 - 0.5j, tol=1e-11, restart=60, max_iter=3000)
    if full_t:
        t_full = np.stack([(lambda U: 0.3 * (U @ U.T - np.eye(L)) / 2.0)(haar_unitary(L, rng)) for _ in range(3)])
        w.update(t_kind="full_types", t_full=t_full, type_of=rng.integers(0, 3, n).astype(np.int32))
    else:
        w.update(t_kind="mie_sites", radii=rng.uniform(0.10, 0.24, n), type_of=np.arange(n, dtype=np.int32))
    cuts = np.linspace(0, n, n_win + 1).round().astype(np.int32)
    w["win_ptr"] = cuts
    return w


# ---- surfaces of revolution for the null-field T-matrix ("numerical discretization ... for evaluating
# these surface integrals").  A generatrix is the discretised surface r = r(theta) about the z axis: arrays
# (theta, r, dr, w) with dr = dr/dtheta and Gauss-Legendre weights w in theta, one panel per smooth piece.
# Geometry only: none of the method's arithmetic.

def _panels(edges, n_per_panel):
    x, w = np.polynomial.legendre.leggauss(n_per_panel)
    th, wt = [], []
    for a, b in zip(edges[:-1], edges[1:]):
        th.append(0.5 * (b - a) * x + 0.5 * (a + b))
        wt.append(0.5 * (b - a) * w)
    return np.concatenate(th), np.concatenate(wt)


def generatrix_sphere(radius, n=48, offset=0.0):
    """Sphere of the given radius whose centre sits at z = offset (|offset| < radius), seen from the origin."""
    th, w = _panels([0.0, np.pi], n)
    root = np.sqrt(radius ** 2 - (offset * np.sin(th)) ** 2)
    r = offset * np.cos(th) + root
    dr = -offset * np.sin(th) - offset ** 2 * np.sin(th) * np.cos(th) / root
    return th, r, dr, w


def generatrix_cylinder(radius, height, n_per_panel=48):
    """Finite circular cylinder (the paper's meta-atom shape) centred on the origin, axis z:
    top cap, side wall, bottom cap (three smooth panels)."""
    hh = 0.5 * height
    tc = np.arctan2(radius, hh)
    th, w = _panels([0.0, tc, np.pi - tc, np.pi], n_per_panel)
    r, dr = np.empty_like(th), np.empty_like(th)
    top, bot = th < tc, th > np.pi - tc
    side = ~(top | bot)
    r[top] = hh / np.cos(th[top]);       dr[top] = hh * np.sin(th[top]) / np.cos(th[top]) ** 2
    r[bot] = -hh / np.cos(th[bot]);      dr[bot] = -hh * np.sin(th[bot]) / np.cos(th[bot]) ** 2
    r[side] = radius / np.sin(th[side]); dr[side] = -radius * np.cos(th[side]) / np.sin(th[side]) ** 2
    return th, r, dr, w


def generatrix_spheroid(a_xy, c_z, n=64):
    """Spheroid x^2/a^2 + y^2/a^2 + z^2/c^2 = 1."""
    th, w = _panels([0.0, np.pi], n)
    s, c = np.sin(th), np.cos(th)
    q = (s / a_xy) ** 2 + (c / c_z) ** 2
    r = q ** -0.5
    dr = -0.5 * q ** -1.5 * 2.0 * s * c * (1.0 / a_xy ** 2 - 1.0 / c_z ** 2)
    return th, r, dr, w


def paper_lens(n_side=56, n_types=32, focal_um=25.0):
    """Stand-in for the paper's own single-GPU workload: silicon cylinders (n = 3.48) of height 940 nm
    and radius 50-250 nm on a square lattice of period 1070 nm in air at wavelength 1550 nm; 56 x 56 sites = 60 um x 60 um,
    "the largest single-GPU simulation" (1-1.5 h on a V100).  Lengths in wavelengths.  The paper picks each radius from the
    phase curve of its periodic library (not available); here the hyperbolic lens phase -k (sqrt(rho^2 + f^2) - f) mod 2 pi
    is mapped linearly onto the sorted radius library, which gives the same kind of layout (concentric zones of growing
    radius).  Returns a dict with pos, type_of, radii, height, eps_r, pitch."""
    lam_nm = 1550.0
    pitch, height = 1070.0 / lam_nm, 940.0 / lam_nm
    radii = np.linspace(50.0, 250.0, n_types) / lam_nm
    pos = lattice(n_side, n_side, pitch)
    f = focal_um * 1000.0 / lam_nm
    phase = np.mod(-K_B * (np.sqrt(pos[:, 0] ** 2 + pos[:, 1] ** 2 + f * f) - f), 2.0 * np.pi)
    type_of = np.minimum((phase / (2.0 * np.pi) * n_types).astype(np.int32), n_types - 1)
    return dict(name=f"paper_lens{n_side}", k=K_B, pos=pos, type_of=type_of, radii=radii, height=height, eps_r=3.48 ** 2,
                pitch=pitch, focal=f)
