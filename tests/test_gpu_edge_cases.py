"""GPU edge cases: degenerate sizes, empty / single-scatterer windows, zero right-hand side, extreme solver options,
maximum lmax of each kernel.  Every result is compared with the oracle."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import driver, matvec as omv, tmatrix  # noqa: E402
from paper_2107_09879_b200 import workloads as W  # noqa: E402


@pytest.fixture(scope="module")
def tm():
    import torch
    assert torch.cuda.is_available()
    from paper_2107_09879_b200 import libtm
    libtm.lib()
    return libtm


from parity_metric import rel, rel_solve  # noqa: E402,F401  (L2 AND per-(l,p)-block / per-point max error; solutions: L2 AND max norm)


def rand_x(shape, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def test_single_scatterer_is_mie(tm):
    """N = 1: A = 0, so s = T p exactly (closed-form Mie response) and GMRES stops after one step."""
    pos = np.array([[0.3, -0.2, 0.1]])
    for lmax in (1, 2, 3):
        s = tm.Solver(pos, lmax, W.K_B)
        t = tm.mie_tmatrix(lmax, W.K_B, 0.2, 4.0)
        s.set_tmatrices(t[None, :], np.zeros(1, dtype=np.int32), True)
        s.set_incident_plane(0.3, 0.7, 1.0, 0.5j)
        sol, info, rc = s.solve(1e-12, 10, 10)
        ref = tmatrix.mie_tmatrix_diag(lmax, W.K_B, 0.2, 4.0) * s.get_incident()[0]
        assert rc == 0 and info[0].iterations <= 1 and rel_solve(sol[0], ref) <= 1e-13
        assert np.all(s.matvec(rand_x((1, s.L), 1), transpose=2) == 0)
        s.close()


def test_empty_and_singleton_windows(tm):
    """win_ptr with an empty window and a one-scatterer window between two real ones."""
    w = W.cloud_workload(41, seed=9, lmax=2, planar=True)
    wp = np.array([0, 20, 20, 21, 41], dtype=np.int32)
    w["win_ptr"] = wp
    ref = driver.solve(w)
    s = tm.solver_for_workload(w)
    sol, info, rc = s.solve(1e-11, 30, 500)
    assert rc == 0 and len(info) == 4 and info[1].iterations == 0 and info[1].converged
    assert rel_solve(sol, ref["s"]) <= 1e-9
    x = rand_x(sol.shape, 3)
    assert rel(s.matvec(x, 2), omv.matvec_rows(2, w["k"], w["pos"], x, win_ptr=wp)) <= 1e-12
    s.close()


def test_zero_incident_gives_zero_solution(tm):
    w = W.config(1)
    s = tm.solver_for_workload(w)
    s.set_incident_coeffs(np.zeros((16, 16), dtype=np.complex128))
    sol, info, rc = s.solve(1e-10, 20, 100)
    assert rc == 0 and info[0].converged and info[0].iterations == 0 and np.all(sol == 0)
    lam, info2, rc2 = s.solve_adjoint(np.zeros((16, 16), dtype=np.complex128), 1e-10, 20, 100)
    assert rc2 == 0 and np.all(lam == 0)
    s.close()


def test_short_and_long_restart_agree(tm):
    """GMRES(8) with many restarts and unrestarted GMRES reach the same solution."""
    w = W.config(1)
    ref = driver.solve(w)
    s = tm.solver_for_workload(w)
    a, ia, rca = s.solve(1e-10, 300, 300)
    b, ib, rcb = s.solve(1e-10, 8, 20000)
    assert rca == 0 and ia[0].restarts == 1 and rel_solve(a, ref["s"]) <= 1e-9
    assert rcb == 0 and ib[0].iterations > ia[0].iterations and rel_solve(b, ref["s"]) <= 1e-9
    with pytest.raises(tm.TmError):
        s.solve(1e-10, 301, 10)                       # restart above the supported maximum
    with pytest.raises(tm.TmError):
        s.solve(0.0, 10, 10)
    s.close()


@pytest.mark.parametrize("lmax", [5, 6])
def test_table_kernel_at_maximum_lmax(tm, lmax):
    """lmax = 6 is the paper's own truncation: L = 96, table-driven kernel, 3 rows per lane."""
    pos = W.random_cloud(12, seed=60 + lmax)
    x = rand_x((12, W.n_modes(lmax)), lmax)
    s = tm.Solver(pos, lmax, W.K_B)
    s.set_kernel(tm.TM_KERNEL_GENERAL)
    assert s.get_kernel() == tm.TM_KERNEL_GENERAL
    assert rel(s.matvec(x, 2), omv.matvec_rows(lmax, W.K_B, pos, x)) <= 1e-12
    with pytest.raises(tm.TmError):
        s.set_kernel(tm.TM_KERNEL_SYM3D)
    s.close()


def test_lmax6_solve_small(tm):
    w = W.cloud_workload(8, seed=66, lmax=6, planar=True)
    ref = driver.solve(w)
    s = tm.solver_for_workload(w)
    assert s.get_kernel() == tm.TM_KERNEL_COPLANAR       # planar: four-sector generated kernel for lmax > 3
    p = s.get_incident()
    assert rel(p, ref["p"]) <= 1e-13
    sol, info, rc = s.solve(1e-11, 60, 600)
    assert rc == 0 and rel_solve(sol, ref["s"]) <= 1e-9
    s.close()


def test_far_apart_and_close_pairs(tm):
    """k r from 1.9 (nearly touching small spheres) to 6e4 (phase accuracy at long range)."""
    pos = np.array([[0.0, 0.0, 0.0], [0.3, 0.0, 0.0], [9000.0, 4000.0, 0.0], [0.0, 0.31, 0.0]])
    x = rand_x((4, 30), 8)
    ref = omv.matvec_rows(3, W.K_B, pos, x)
    s = tm.Solver(pos, 3, W.K_B)
    assert rel(s.matvec(x, 2), ref) <= 1e-11             # k r = 6e4: 6e4 * 1.1e-16 phase rounding on both sides
    s.close()


def test_adjoint_radius_sensitivities(tm):
    """NEXT-2 (geometry half): dJ/dR_j for every scatterer from ONE adjoint solve (PAPER.md Eqs. IV8-IV9) against the oracle's
    adjoint formula (tight) and the oracle's finite differences of the dense solve (the plain definition)."""
    from oracle import gradient, incident
    rng = np.random.default_rng(12)
    pos = W.random_cloud(6, seed=41)
    radii = rng.uniform(0.10, 0.22, 6)
    lmax = 2
    p = incident.plane_wave_incident(lmax, W.K_B, pos, 0.3, 0.8, 1.0, 0.4j)
    v = rand_x(p.shape, 13)
    g_ref, s_ref, lam_ref = gradient.adjoint_radius_gradient(lmax, W.K_B, pos, radii, 4.0, p, v)
    s = tm.Solver(pos, lmax, W.K_B)
    T = np.stack([tm.mie_tmatrix(lmax, W.K_B, r, 4.0) for r in radii])
    dT = np.stack([tm.mie_tmatrix_dR(lmax, W.K_B, r, 4.0) for r in radii])
    assert rel(dT, np.stack([gradient.mie_dT_dR(lmax, W.K_B, r, 4.0) for r in radii])) <= 1e-8
    s.set_tmatrices(T, np.arange(6, dtype=np.int32), True)
    s.set_incident_plane(0.3, 0.8, 1.0, 0.4j)
    sol, _, rc = s.solve(1e-12, 60, 600)
    lam, _, rc2 = s.solve_adjoint(v, 1e-12, 60, 600)
    assert rc == 0 and rc2 == 0
    g = s.grad_tmatrix(dT, lam, sol)
    assert rel(g, g_ref) <= 1e-8
    for j in (0, 3):
        fd = gradient.fd_radius(lmax, W.K_B, pos, radii, 4.0, p, v, j)
        assert abs(g[j] - fd) <= 1e-6 * abs(fd)
    s.close()


@pytest.mark.parametrize("lmax,n,planar", [(2, 5, False), (2, 5, True), (3, 6, True), (4, 4, False), (6, 3, True)])
def test_adjoint_position_sensitivities(tm, lmax, n, planar):
    """NEXT-2 (position half): dJ/dx_{j,alpha} for every scatterer and direction from ONE adjoint solve (Eqs. IV3-IV9) with the
    ANALYTIC derivative of the translation operator (dA/dd = k D A^ext: two all-pairs products at lmax + 1),
    3-D clouds and planar layouts (the z-derivative of a planar layout stays on the coplanar kernel), up to the paper's
    lmax = 6, against the oracle's chain-rule derivative (oracle/translation.py: d_xi_matrix) and, for one component, against
    central differences of the oracle's whole dense solve."""
    from oracle import gradient, incident
    rng = np.random.default_rng(22 + lmax)
    beta, alpha = 0.4, -0.5
    kv = W.K_B * np.array([np.sin(beta) * np.cos(alpha), np.sin(beta) * np.sin(alpha), np.cos(beta)])
    pos = W.random_cloud(n, seed=8 + lmax, planar=planar)
    radii = rng.uniform(0.12, 0.2, n)
    L = W.n_modes(lmax)
    inc = lambda q: incident.plane_wave_incident(lmax, W.K_B, q, beta, alpha, 0.7, 0.2j)
    dinc = lambda q: 1j * kv[None, :, None] * inc(q)[:, None, :]
    v = rand_x((n, L), 23)
    g_ref, s_ref, lam_ref = gradient.adjoint_position_gradient(lmax, W.K_B, pos, radii, 4.0, inc, v, dinc_fn=dinc)
    s = tm.Solver(pos, lmax, W.K_B)
    T = np.stack([tm.mie_tmatrix(lmax, W.K_B, r, 4.0) for r in radii])
    s.set_tmatrices(T, np.arange(n, dtype=np.int32), True)
    s.set_incident_plane(beta, alpha, 0.7, 0.2j)
    kern = s.get_kernel()
    sol, _, rc = s.solve(1e-13, 80, 800)
    lam, _, rc2 = s.solve_adjoint(v, 1e-13, 80, 800)
    p = s.get_incident()
    dp = 1j * kv[None, :, None] * p[:, None, :]                     # plane wave: d p_j / d x_j = i k p_j
    g = s.grad_positions(lam, sol, dp=dp)
    assert s.get_kernel() == kern
    assert np.abs(g - g_ref).max() <= 1e-9 * np.abs(g_ref).max()
    # the gradient kernels alone, on the ORACLE's solutions (no GMRES error in the comparison)
    g0 = s.grad_positions(lam_ref, s_ref, dp=dp)
    assert np.abs(g0 - g_ref).max() <= 1e-11 * np.abs(g_ref).max()
    assert np.abs(s.grad_positions(lam_ref, s_ref, dp=dp) - g0).max() == 0.0      # second call (cached context): same bits
    if lmax <= 3:
        fd = gradient.fd_position(lmax, W.K_B, pos, radii, 4.0, inc, v, 2, 2)
        assert abs(g[2, 2] - fd) <= 1e-6 * np.abs(g_ref).max()
    s.close()


def test_fp32_precision_floor_stops_the_restart_loop(tm):
    """A tolerance below what an fp32 operator can reach: the solver must notice (estimated residual met, true residual
    stuck) and return the soft status after a few cycles instead of burning max_iter."""
    w = W.config(2, scale=12)
    ref = driver.solve(w)
    s = tm.solver_for_workload(w, precision=tm.TM_FP32)
    sol, info, rc = s.solve(1e-9, 50, 100000)
    assert rc == tm.TM_NOT_CONVERGED and info[0].rel_residual < 1e-5
    assert info[0].matvecs < 3000                        # not the 100000-iteration budget
    assert rel_solve(sol, ref["s"]) <= 1e-4
    s.close()


@pytest.mark.parametrize("lmax", [4, 5, 6])
def test_four_sector_coplanar_kernel(tm, lmax):
    """lmax 4..6 on planar layouts (lmax = 6 is the paper's truncation): several 128-target tiles with a ragged tail,
    source chunks, ragged windows, against the oracle and against the table-driven kernel; fp32 too."""
    pos = W.lattice(13, 11 if lmax == 6 else 14)
    pos = pos + np.random.default_rng(lmax).uniform(-0.05, 0.05, pos.shape) * [1, 1, 0]      # not a perfect lattice
    N, L = pos.shape[0], W.n_modes(lmax)
    wp = np.array([0, 40, 41, N], dtype=np.int32)
    x = rand_x((N, L), 70 + lmax)
    ref = omv.matvec_rows(lmax, W.K_B, pos, x, win_ptr=wp)
    s = tm.Solver(pos, lmax, W.K_B, win_ptr=wp)
    assert s.get_kernel() == tm.TM_KERNEL_COPLANAR
    u = s.matvec(x, transpose=2)
    assert rel(u, ref) <= 1e-12 and np.all(u[40] == 0)
    s.set_kernel(tm.TM_KERNEL_GENERAL)
    assert rel(s.matvec(x, transpose=2), u) <= 1e-12
    s.close()
    s = tm.Solver(pos, lmax, W.K_B, win_ptr=wp, precision=tm.TM_FP32)
    assert rel(s.matvec(x, transpose=2), ref) <= 2e-5
    s.close()


@pytest.mark.parametrize("lmax", [4, 6])
def test_incident_and_fields_at_high_lmax(tm, lmax):
    """Beam / jinc expansion and field evaluation for lmax up to 6 (the paper's truncation)."""
    from oracle import fields, incident
    pos = W.random_cloud(6, seed=50 + lmax)
    s = tm.Solver(pos, lmax, W.K_B)
    focus = np.array([[0.2, -0.1, 0.3]])
    s.set_incident_gauss(focus, 2.0, 0.8, 0.3 - 0.4j)
    ref = incident.gaussian_beam_incident(lmax, W.K_B, pos, focus[0], 2.0, 0.8, 0.3 - 0.4j)
    assert rel(s.get_incident(), ref) <= 1e-10
    src = np.array([[0.5, 0.5, -2.0], [-1.0, 0.2, -2.0]])
    amp = np.array([[1.0, 0.2j], [0.3, -0.7]])
    s.set_incident_jinc(src, amp)
    assert rel(s.get_incident(), incident.jinc_sources_incident(lmax, W.K_B, pos, src, amp)) <= 1e-10
    coef = rand_x((6, W.n_modes(lmax)), lmax)
    pts = np.random.default_rng(lmax).uniform(-4, 4, (40, 3))
    pts = pts[np.linalg.norm(pts[:, None, :] - pos[None], axis=2).min(axis=1) > 0.4]
    assert rel(s.fields(pts, coef, tm.TM_FIELD_E_SCA), fields.e_sca(lmax, W.K_B, pos, coef, pts)) <= 1e-12
    assert rel(s.fields(pts, coef, tm.TM_FIELD_H_SCA), fields.zh_sca(lmax, W.K_B, pos, coef, pts)) <= 1e-12
    s.close()


def test_mixed_precision_iterative_refinement(tm):
    """TM_MIXED: fp32 Krylov cycles, fp64 iterate / right-hand side / true residual: fp64-level parity with the oracle.
    Covers the cooperative path (small), diagonal and full T, windows, forward and adjoint."""
    w = W.config(2, scale=12)
    ref = driver.solve(w)
    s = tm.solver_for_workload(w, precision=tm.TM_MIXED)
    sol, info, rc = s.solve(1e-10, 50, 5000)
    assert rc == 0 and info[0].rel_residual <= 1e-10 and rel_solve(sol, ref["s"]) <= 1e-9
    x = rand_x(sol.shape, 5)                              # everything outside the solves runs in fp64
    assert rel(s.matvec(x, 0), (ref["M"] @ x.reshape(-1)).reshape(x.shape)) <= 1e-12
    s.close()
    w = W.config(4, scale=6)
    ref = driver.solve(w, adjoint_w=w["w_adj"])
    s = tm.solver_for_workload(w, precision=tm.TM_MIXED)
    sol, info, rc = s.solve(1e-11, 50, 5000)
    lam, info2, rc2 = s.solve_adjoint(w["w_adj"], 1e-11, 50, 5000)
    assert rc == 0 and rc2 == 0 and rel_solve(sol, ref["s"]) <= 1e-9 and rel_solve(lam, ref["lam"]) <= 1e-9
    s.close()
    w = W.config("3b", scale=8)
    ref = driver.solve(w)
    s = tm.solver_for_workload(w, precision=tm.TM_MIXED)
    sol, info, rc = s.solve(1e-11, 50, 5000)
    assert rc == 0 and rel_solve(sol, ref["s"]) <= 1e-9
    s.close()


def test_incident_field_at_detector_points(tm):
    """TM_FIELD_E_INC: plane wave (closed form), Gaussian beams and jinc sources (direct 2-D quadrature of Eq. II4 in the
    oracle), all sources of all windows summed."""
    from oracle import incident
    pos = W.random_cloud(6, seed=71)
    pts = np.random.default_rng(72).uniform(-2, 2, (9, 3))
    s = tm.Solver(pos, 2, W.K_B, win_ptr=np.array([0, 2, 6], dtype=np.int32))
    with pytest.raises(tm.TmError) as e:
        s.fields(pts, None, tm.TM_FIELD_E_INC)
    assert e.value.code == tm.TM_E_STATE
    beta, alpha, Ab, Aa = 0.5, -0.7, 0.8, 0.3 - 0.4j
    s.set_incident_plane(beta, alpha, Ab, Aa)
    kv = W.K_B * np.array([np.sin(beta) * np.cos(alpha), np.sin(beta) * np.sin(alpha), np.cos(beta)])
    bh = np.array([np.cos(beta) * np.cos(alpha), np.cos(beta) * np.sin(alpha), -np.sin(beta)])
    ah = np.array([-np.sin(alpha), np.cos(alpha), 0.0])
    ref = (Ab * bh + Aa * ah)[None, :] * np.exp(1j * pts @ kv)[:, None]
    assert rel(s.fields(pts, None, tm.TM_FIELD_E_INC), ref) <= 1e-13
    focus = np.array([[0.2, -0.1, -0.5], [-0.6, 0.4, -0.5]])
    s.set_incident_gauss(focus, 1.5, 0.8, 0.3 - 0.4j)
    ref = np.array([sum(incident.gaussian_beam_field_direct(W.K_B, p, f, 1.5, 0.8, 0.3 - 0.4j, n_beta=300, n_alpha=512) for f in focus)
                    for p in pts])
    assert rel(s.fields(pts, None, tm.TM_FIELD_E_INC), ref) <= 1e-8
    src = np.array([[0.5, 0.5, -1.0], [-1.0, 0.2, -1.0], [0.0, 0.0, -1.0]])
    amp = np.array([[1.0, 0.2j], [0.3, -0.7], [0.5j, 0.1]])
    s.set_incident_jinc(src, amp, np.array([0, 1, 3], dtype=np.int32))
    ref = np.array([sum(incident.jinc_field_direct(W.K_B, p, src[i], amp[i, 0], amp[i, 1]) for i in range(3)) for p in pts])
    assert rel(s.fields(pts, None, tm.TM_FIELD_E_INC), ref) <= 1e-7
    s.close()


@pytest.mark.parametrize("precision", ["fp64", "mixed"])
def test_warm_start(tm, precision):
    """tm_solve_opts.warm_start (optimisation loop): starting from the exact solution takes no Arnoldi
    step; starting from the solution of a slightly different design takes fewer steps than a cold start and reaches the
    same solution (oracle: dense LU of the perturbed design); the adjoint solve honours it too."""
    prec = tm.TM_FP64 if precision == "fp64" else tm.TM_MIXED
    w = W.cloud_workload(40, seed=11, lmax=2, planar=True)
    ref = driver.solve(w)
    s = tm.solver_for_workload(w, precision=prec)
    cold, ic, rc = s.solve(1e-10, 30, 2000)
    assert rc == 0 and rel_solve(cold, ref["s"]) <= 1e-9
    again = cold.copy()
    again, ia, rc = s.solve(1e-10, 30, 2000, out=again, warm_start=True)
    assert rc == 0 and ia[0].iterations == 0 and ia[0].rel_residual <= 1e-10 and rel_solve(again, ref["s"]) <= 1e-9
    # design step: every radius grows by 0.5 %
    w2 = dict(w)
    w2["radii"] = np.asarray(w["radii"]) * 1.005
    ref2 = driver.solve(w2)
    T2 = np.stack([tm.mie_tmatrix(w["lmax"], w["k"], r, w["eps_r"]) for r in w2["radii"]])
    s.set_tmatrices(T2, np.asarray(w["type_of"], dtype=np.int32), True)
    cold2, ic2, rc = s.solve(1e-10, 30, 2000)
    assert rc == 0 and rel_solve(cold2, ref2["s"]) <= 1e-9
    warm2 = cold.copy()
    warm2, iw2, rc = s.solve(1e-10, 30, 2000, out=warm2, warm_start=True)
    assert rc == 0 and rel_solve(warm2, ref2["s"]) <= 1e-9
    assert iw2[0].iterations < ic2[0].iterations
    # adjoint
    wv = rand_x(cold.shape, 5)
    lam, il, rc = s.solve_adjoint(wv, 1e-10, 30, 2000)
    lam2 = lam.copy()
    lam2, il2, rc2 = s.solve_adjoint(wv, 1e-10, 30, 2000, out=lam2, warm_start=True)
    assert rc == 0 and rc2 == 0 and il2[0].iterations == 0 and rel_solve(lam2, lam) <= 1e-9
    s.close()


def test_cuda_graph_cycles_equal_launch_by_launch_cycles(tm):
    """Window-sized problems replay a full restart cycle as one CUDA graph: same kernels, same arguments, so the
    iterates must equal - bit for bit - those of the launch-by-launch path (the library's timing mode), forward and transposed,
    also after the T-matrices were replaced (the captured nodes bake the T pointer: the cache key must notice) and in TM_MIXED."""
    w = W.config(2, scale=14)
    for prec in (tm.TM_FP64, tm.TM_MIXED):
        s = tm.solver_for_workload(w, precision=prec)
        wv = rand_x((196, 30), 5)
        s.kernel_time(reset=-1)                                          # production mode: graphs
        a, ia, rca = s.solve(1e-10, 12, 600)                             # several cycles of restart 12
        la, _, _ = s.solve_adjoint(wv, 1e-10, 12, 600)
        a2, _, _ = s.solve(1e-10, 12, 600)                               # replay of the cached graph
        s.kernel_time(reset=True)                                        # timing mode: launch by launch
        b, ib, rcb = s.solve(1e-10, 12, 600)
        lb, _, _ = s.solve_adjoint(wv, 1e-10, 12, 600)
        assert rca == 0 and rcb == 0 and ia[0].iterations == ib[0].iterations and ia[0].restarts > 2
        assert np.array_equal(a, b) and np.array_equal(a, a2) and np.array_equal(la, lb)
        s.kernel_time(reset=-1)
        # new T-matrices on the same context
        w2 = dict(w, radii=np.asarray(w["radii"]) * 0.9)
        T2 = np.stack([tm.mie_tmatrix(3, W.K_B, r, 4.0) for r in w2["radii"]])
        s.set_tmatrices(T2, w["type_of"], True)
        c, _, rcc = s.solve(1e-11, 12, 900)
        assert rcc == 0 and rel_solve(c, driver.solve(w2)["s"]) <= 1e-9
        s.close()


def test_solve_multi_equals_separate_solves_and_the_oracle(tm):
    """tm_solve_multi (NEXT-3: several right-hand sides on one geometry, solved together as replicated windows): same solutions and
    iteration counts as separate solves, forward and adjoint, two windows, also after the T-matrices were replaced (the auxiliary
    context must re-clone them) and in TM_MIXED; right-hand side 0 against the oracle's dense LU."""
    w = W.cloud_workload(40, seed=77, lmax=3, n_win=2)
    ref = driver.solve(w)
    for prec in (tm.TM_FP64, tm.TM_MIXED):
        s = tm.solver_for_workload(w, precision=prec)
        P = [s.get_incident().copy()]
        for (b, a, Ab, Aa) in ((0.0, 0.0, 0.0, 1.0), (0.7, 2.0, 0.3, 1.0 - 0.5j)):
            s.set_incident_plane(b, a, Ab, Aa)
            P.append(s.get_incident().copy())
        P = np.stack(P)
        sep, its = [], []
        for r in range(3):
            s.set_incident_coeffs(P[r])
            sol, info, rc = s.solve(1e-11, 40, 2000)
            assert rc == 0
            sep.append(sol.copy()); its.append([i.iterations for i in info])
        out, info, rc = s.solve_multi(P, 1e-11, 40, 2000)
        assert rc == 0 and out.shape == (3, 40, 30)
        for r in range(3):
            assert rel_solve(out[r], sep[r]) <= 1e-12
            assert [i.iterations for i in info[r]] == its[r]
        assert rel_solve(out[0], ref["s"]) <= 1e-9
        # adjoint right-hand sides
        Wv = rand_x((2, 40, 30), 78)
        lam, _, rc = s.solve_multi(Wv, 1e-11, 40, 2000, adjoint=True)
        assert rc == 0
        for r in range(2):
            l1, _, _ = s.solve_adjoint(Wv[r], 1e-11, 40, 2000)
            assert rel_solve(lam[r], l1) <= 1e-12
        # new T-matrices: the cached auxiliary context must pick them up
        w2 = dict(w, radii=np.asarray(w["radii"]) * 0.93)
        s.set_tmatrices(np.stack([tm.mie_tmatrix(3, W.K_B, r, 4.0) for r in w2["radii"]]), w["type_of"], True)
        out2, _, rc = s.solve_multi(P[:1], 1e-11, 40, 2000)              # and another n_rhs
        assert rc == 0 and rel_solve(out2[0], driver.solve(w2)["s"]) <= 1e-9
        s.close()
