"""Full-size parity (BASELINE.json sizes, in the launch configuration bench.py times): sampled outputs the oracle can
compute one by one, and properties that hold at any size.  DESIGN.md section 6 / SURVEY.md 8(c) "full-size parity"."""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import matvec as omv  # noqa: E402
from paper_2107_09879_b200 import workloads as W  # noqa: E402

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


@pytest.fixture(scope="module")
def tm():
    import torch
    assert torch.cuda.is_available()
    from paper_2107_09879_b200 import libtm
    libtm.lib()
    return libtm


def rel(a, b):
    return np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(b)


def rand_x(shape, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def sampled_operator_rows(w, x, rows):
    """Oracle rows of y = (I - T A) x for the sampled targets (diag or full T); the oracle's T is evaluated for the
    sampled scatterers only (per-site Mie for 2.6e5 sites through scipy would take hours)."""
    from oracle import tmatrix
    u = omv.matvec_rows(w["lmax"], w["k"], w["pos"], x, rows=rows, win_ptr=w["win_ptr"])
    type_of = np.asarray(w["type_of"])
    if w["t_kind"] in ("mie_types", "mie_sites"):
        t_rows = np.stack([tmatrix.mie_tmatrix_diag(w["lmax"], w["k"], w["radii"][type_of[r]], w["eps_r"]) for r in rows])
        tu = t_rows * u
    else:
        tu = np.einsum("nab,nb->na", np.asarray(w["t_full"])[type_of[rows]], u)
    return x[rows] - tu


@pytest.mark.parametrize("cfg,prec,tol,n_rows", [(2, "fp64", 1e-12, 64), (3, "fp64", 1e-12, 16), (3, "fp32", 2e-5, 16),
                                                 (4, "fp64", 1e-12, 24), (5, "fp64", 1e-12, 8)])
def test_operator_rows_at_full_size(tm, cfg, prec, tol, n_rows):
    w = W.config(cfg)
    N, L = w["pos"].shape[0], W.n_modes(w["lmax"])
    x = rand_x((N, L), 100 + cfg)
    s = tm.solver_for_workload(w, precision=tm.TM_FP32 if prec == "fp32" else tm.TM_FP64)
    assert s.get_kernel() == tm.TM_KERNEL_COPLANAR
    y = s.matvec(x, 0)
    rng = np.random.default_rng(200 + cfg)
    rows = np.sort(rng.choice(N, n_rows, replace=False)).astype(np.int32)
    rows[0], rows[-1] = 0, N - 1                          # first and last scatterer (tile / chunk edges)
    ref = sampled_operator_rows(w, x, rows)
    assert rel(y[rows], ref) <= tol
    # transpose consistency at full size: z^T (M x) = (M^T z)^T x  (bilinear, no conjugation)
    z = rand_x((N, L), 300 + cfg)
    yt = s.matvec(z, 1)
    lhs, rhs = np.sum(z * y), np.sum(yt * x)
    assert abs(lhs - rhs) <= (1e-10 if prec == "fp64" else 1e-3) * abs(lhs)
    s.close()


def test_cfg2_full_solve_vs_dense_lu_golden(tm):
    """Config 2 at full size: GPU GMRES(50) to 1e-10 against the oracle's dense LU (tests/golden/make_golden.py cfg2)."""
    path = os.path.join(GOLD, "cfg2_solution.npy")
    if not os.path.exists(path):
        pytest.skip("golden file not generated (python tests/golden/make_golden.py cfg2)")
    ref = np.load(path)
    w = W.config(2)
    s = tm.solver_for_workload(w)
    sol, info, rc = s.solve(w["tol"], w["restart"], w["max_iter"])
    assert rc == 0 and info[0].rel_residual <= w["tol"]
    assert rel(sol, ref) <= 1e-9
    s.close()


@pytest.mark.parametrize("cfg,scale", [(2, None), (5, 64)])
def test_energy_conservation_of_the_gpu_solution(tm, cfg, scale):
    """Property that holds at any size (no oracle values): lossless Mie spheres under a unit plane wave scatter exactly what they
    extinguish, C_ext = -(pi/k^2) Re p^H s = C_sca = (pi/k^2) (|s|^2 + Re s^H A s)  (Re s^H A s = s^H RgA s
    because the Neumann part of A is Hermitian, identity S4b pinned in tests/test_oracle_vswf_translation.py).  The operator
    product A s is the GPU all-pairs kernel; a wrong block, sign or missing pair breaks the balance at O(1)."""
    w = W.config(cfg, scale=scale)
    s = tm.solver_for_workload(w)
    sol, info, rc = s.solve(1e-10, w["restart"], 4000)
    assert rc == 0
    p = s.get_incident()
    u = s.matvec(sol, transpose=2)                                   # u = A s
    c_ext = -(np.pi / w["k"] ** 2) * np.real(np.vdot(p, sol))
    c_sca = (np.pi / w["k"] ** 2) * (np.real(np.vdot(sol, sol)) + np.real(np.vdot(sol, u)))
    assert c_ext > 0 and abs(c_ext - c_sca) <= 1e-8 * c_ext
    s.close()


def test_cfg4_windows_are_independent_at_full_size(tm):
    """One 64x64 window solved alone vs. inside the 64-window batch: a few GMRES cycles give identical iterates."""
    w = W.config(4)
    lo, hi = int(w["win_ptr"][5]), int(w["win_ptr"][6])
    s = tm.solver_for_workload(w)
    sol, info, rc = s.solve(1e-3, 20, 20)
    w1 = dict(w, pos=w["pos"][lo:hi], win_ptr=np.array([0, hi - lo], dtype=np.int32), radii=w["radii"][lo:hi],
              type_of=np.arange(hi - lo, dtype=np.int32), focus=w["focus"][5:6])
    s1 = tm.solver_for_workload(w1)
    sol1, info1, rc1 = s1.solve(1e-3, 20, 20)
    assert rel(sol1, sol[lo:hi]) <= 1e-10
    assert info1[0].iterations == info[5].iterations
    s.close(); s1.close()


def test_sym3d_kernel_on_a_large_3d_cloud(tm):
    """Generated 3-D kernel at scale (2e4 scatterers in a slab: 157 target tiles, many source chunks): sampled oracle rows."""
    rng = np.random.default_rng(91)
    n = 20000
    side = 40.0
    # jittered grid in a slab of thickness 3 wavelengths: minimum separation stays > 0.3
    g = int(np.ceil(np.sqrt(n / 3)))
    ix, iy, iz = np.meshgrid(np.arange(g), np.arange(g), np.arange(3), indexing="ij")
    pos = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1)[:n].astype(float)
    pos[:, :2] *= side / g
    pos += rng.uniform(-0.1, 0.1, pos.shape)
    x = rand_x((n, 30), 92)
    s = tm.Solver(pos, 3, W.K_B)
    assert s.get_kernel() == tm.TM_KERNEL_SYM3D
    u = s.matvec(x, transpose=2)
    rows = np.sort(rng.choice(n, 12, replace=False)).astype(np.int32)
    rows[0], rows[-1] = 0, n - 1
    ref = omv.matvec_rows(3, W.K_B, pos, x, rows=rows)
    assert rel(u[rows], ref) <= 1e-12
    s.close()
