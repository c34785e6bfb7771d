"""NEXT-4: null-field T-matrices of bodies of revolution on the device (tm_nullfield_tmatrix) against the oracle's literal
two-dimensional surface quadrature (oracle/nullfield.py), and through the coupled solve."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import nullfield as onf, system, tmatrix, incident  # noqa: E402
from paper_2107_09879_b200 import workloads as W  # noqa: E402

K = W.K_B


@pytest.fixture(scope="module")
def tm():
    import torch
    assert torch.cuda.is_available()
    from paper_2107_09879_b200 import libtm
    libtm.lib()
    return libtm


def maxrel(a, b):
    return np.abs(np.asarray(a) - np.asarray(b)).max() / np.abs(b).max()


@pytest.mark.parametrize("lmax", [1, 2, 3, 4, 6])
def test_sphere_is_mie(tm, lmax):
    T = tm.nullfield_tmatrix(lmax, K, 4.0, W.generatrix_sphere(0.2, 48))
    assert maxrel(T, np.diag(tmatrix.mie_tmatrix_diag(lmax, K, 0.2, 4.0))) <= 1e-12


def test_lossy_medium(tm):
    """Complex permittivity (Im eps_r > 0, e^{-i omega t}): complex k_s, Bessel functions of complex argument."""
    eps = 12.0 + 0.8j
    T = tm.nullfield_tmatrix(4, K, eps, W.generatrix_sphere(0.15, 48))
    assert maxrel(T, np.diag(tmatrix.mie_tmatrix_diag(4, K, 0.15, eps))) <= 1e-12
    assert maxrel(T, np.diag(tm.mie_tmatrix(4, K, 0.15, eps))) <= 1e-12
    g = W.generatrix_cylinder(0.1, 0.25, 40)
    assert maxrel(tm.nullfield_tmatrix(5, K, eps, g), onf.nullfield_tmatrix(5, K, eps, g)) <= 1e-9
    g = W.generatrix_spheroid(0.12, 0.18, 64)
    assert maxrel(tm.nullfield_tmatrix(3, K, 2.0 + 3.0j, g), onf.nullfield_tmatrix(3, K, 2.0 + 3.0j, g)) <= 1e-9


@pytest.mark.parametrize("name,lmax,gen", [
    ("cylinder", 3, W.generatrix_cylinder(0.15, 0.3, 32)),
    ("cylinder", 6, W.generatrix_cylinder(0.12, 0.35, 43)),          # 129 nodes: three stages, ragged tail
    ("spheroid", 4, W.generatrix_spheroid(0.15, 0.22, 64)),
    ("offset sphere", 5, W.generatrix_sphere(0.2, 70, offset=0.05)),   # no mirror symmetry: full (l, p) blocks
])
def test_matches_oracle_surface_quadrature(tm, name, lmax, gen):
    T = tm.nullfield_tmatrix(lmax, K, 4.0, gen)
    ref = onf.nullfield_tmatrix(lmax, K, 4.0, gen)
    assert maxrel(T, ref) <= 1e-9


@pytest.mark.parametrize("lmax,lint", [(2, 6), (3, 8), (6, 10), (6, 12), (1, 12)])
def test_internal_truncation(tm, lmax, lint):
    """Expansions inside the method carried to lmax_internal > lmax (blocks up to 24 x 24), block l <= lmax returned; the case
    is the paper's own meta-atom: a silicon cylinder 940 nm tall, radius 205 nm at 1550 nm, where lmax 6 alone is far from
    converged."""
    g = W.generatrix_cylinder(204.84 / 1550, 940.0 / 1550, 48)
    T = tm.nullfield_tmatrix(lmax, K, 3.48 ** 2, g, lmax_internal=lint)
    ref = onf.nullfield_tmatrix(lmax, K, 3.48 ** 2, g, lmax_internal=lint)
    assert maxrel(T, ref) <= 1e-8
    if lmax == 6:
        assert maxrel(T, onf.nullfield_tmatrix(6, K, 3.48 ** 2, g)) > 0.1       # the lmax-6-only result is a different matrix


def test_library_of_shapes_in_one_call(tm):
    radii = [0.10, 0.14, 0.18, 0.22]
    gens = [W.generatrix_cylinder(r, 0.3, 24) for r in radii]
    Ts = tm.nullfield_tmatrix(3, K, 4.0, gens)
    assert Ts.shape == (4, 30, 30)
    for T, g in zip(Ts, gens):
        assert maxrel(T, onf.nullfield_tmatrix(3, K, 4.0, g)) <= 1e-9
        assert maxrel(T, tm.nullfield_tmatrix(3, K, 4.0, g)) == 0.0          # batch = single, bit for bit


def test_invalid_arguments(tm):
    g = W.generatrix_sphere(0.2, 8)
    for bad in ((0, K, 4.0, g), (7, K, 4.0, g), (3, K, -1.0, g), (3, K, 0.0, g), (3, K, 4.0 - 1.0j, g), (3, K, 4.0, (g[0], -g[1], g[2], g[3])),
                (3, K, 4.0, (g[0] + 4.0, g[1], g[2], g[3]))):
        with pytest.raises(tm.TmError):
            tm.nullfield_tmatrix(*bad)
    for li in (2, 13, -1):
        with pytest.raises(tm.TmError):
            tm.nullfield_tmatrix(3, K, 4.0, g, lmax_internal=li)


def test_cylinder_lattice_solve_vs_dense_lu(tm):
    """6x6 lattice of cylinders from a 4-radius library: device T-matrices -> tm_set_tmatrices (full) -> GMRES, against the
    oracle's T-matrices -> dense LU."""
    lmax = 3
    rng = np.random.default_rng(11)
    pos = W.lattice(6, 6)
    radii = [0.10, 0.13, 0.16, 0.19]
    gens = [W.generatrix_cylinder(r, 0.3, 32) for r in radii]
    type_of = rng.integers(0, 4, len(pos)).astype(np.int32)
    t_dev = tm.nullfield_tmatrix(lmax, K, 4.0, gens)
    t_ref = np.stack([onf.nullfield_tmatrix(lmax, K, 4.0, g) for g in gens])
    p = incident.plane_wave_incident(lmax, K, pos, 0.0, 0.0, 1.0, 0.0)
    M = system.assemble_M(lmax, K, pos, t_ref, type_of, False)
    ref = system.solve_forward(M, t_ref, type_of, False, p)
    s = tm.Solver(pos, lmax, K)
    s.set_tmatrices(t_dev, type_of, False)
    s.set_incident_plane(0.0, 0.0, 1.0, 0.0)
    sol, info, rc = s.solve(1e-11, 50, 500)
    assert rc == 0
    assert np.linalg.norm(sol - ref) / np.linalg.norm(ref) <= 1e-9
    s.close()


def test_dtmatrix_against_differences_of_the_oracle(tm):
    """tm_nullfield_dtmatrix (device Richardson difference of four generatrices) vs. the same derivative taken from the ORACLE's
    T-matrices with another step (central difference, h = 1e-5: truncation ~1e-8 relative)."""
    lmax, radii = 3, [0.12, 0.18]
    fn = lambda r: W.generatrix_cylinder(r, 0.3, 32)           # noqa: E731
    dT = tm.nullfield_dtmatrix(lmax, K, 4.0, fn, radii, 2e-3)
    for d, r in zip(dT, radii):
        ref = (onf.nullfield_tmatrix(lmax, K, 4.0, fn(r + 1e-5)) - onf.nullfield_tmatrix(lmax, K, 4.0, fn(r - 1e-5))) / 2e-5
        assert maxrel(d, ref) <= 1e-6


def test_cylinder_radius_gradient_through_the_adjoint_solve(tm):
    """The paper's optimisation chain for its own meta-atoms: cylinder radii -> null-field T and dT/dR on
    the device -> forward + adjoint GMRES -> tm_grad_tmatrix, against central differences of the oracle's dense solve."""
    from oracle import gradient
    lmax = 2
    rng = np.random.default_rng(5)
    pos = W.lattice(4, 4)
    radii = np.array([0.11, 0.15, 0.19])
    fn = lambda r: W.generatrix_cylinder(r, 0.3, 24)           # noqa: E731
    type_of = rng.integers(0, 3, len(pos)).astype(np.int32)
    v = W.complex_normal((len(pos), W.n_modes(lmax)), rng)
    s = tm.Solver(pos, lmax, K)
    s.set_tmatrices(tm.nullfield_tmatrix(lmax, K, 4.0, [fn(r) for r in radii]), type_of, False)
    s.set_incident_plane(0.0, 0.0, 1.0, 0.0)
    sol, _, rc = s.solve(1e-12, 50, 500)
    lam, _, rc2 = s.solve_adjoint(v, 1e-12, 50, 500)
    assert rc == 0 and rc2 == 0
    g_site = s.grad_tmatrix(tm.nullfield_dtmatrix(lmax, K, 4.0, fn, radii, 2e-3), lam, sol)
    p = incident.plane_wave_incident(lmax, K, pos, 0.0, 0.0, 1.0, 0.0)
    for t in range(3):
        g = np.sum(g_site[type_of == t])
        ref = gradient.fd_shape_parameter(lmax, K, pos, fn, radii, type_of, 4.0, p, v, t)
        assert abs(g - ref) <= 1e-6 * abs(ref)
    s.close()
