"""T-matrix look-up table on the device (tm_ttable_interp, reading R20) against oracle/ttable.py, and through the
coupled solve: radius gradient of an objective whose T-matrices come from the interpolated table."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import incident, system, tmatrix, ttable  # noqa: E402
from paper_2107_09879_b200 import workloads as W  # noqa: E402

K = W.K_B
NODES = np.array([0.05, 0.08, 0.10, 0.13, 0.17, 0.19, 0.24, 0.25])          # not equidistant


@pytest.fixture(scope="module")
def tm():
    import torch
    assert torch.cuda.is_available()
    from paper_2107_09879_b200 import libtm
    libtm.lib()
    return libtm


def maxrel(a, b):
    return np.abs(np.asarray(a) - np.asarray(b)).max() / np.abs(b).max()


# Tolerances: T is a 4-term sum of weights |w_a| <= ~1.3 times table entries, the weights themselves 3 products and a division
# (kernel: one reciprocal of the denominator product; oracle: product of three ratios) - a few ulp each -> 1e-14 expected, 1e-13
# required; the derivative weights are sums of products of mixed sign divided by the same denominators -> 1e-12 required.
@pytest.mark.parametrize("shape", [(30,), (16, 16), (7,), (30, 30), (257,)])
def test_interpolation_matches_the_oracle_host_and_device_arrays(tm, shape):
    import torch
    rng = np.random.default_rng(11)
    tab = rng.standard_normal((len(NODES),) + shape) + 1j * rng.standard_normal((len(NODES),) + shape)
    p = np.concatenate([NODES, 0.5 * (NODES[:-1] + NODES[1:]), rng.uniform(NODES[0], NODES[-1], 1003)])      # ragged: 1018 sites
    T_ref, dT_ref = ttable.interp_table(NODES, tab, p)
    T, dT = tm.ttable_interp(NODES, tab, p)
    assert T.shape == T_ref.shape and dT.shape == dT_ref.shape
    assert maxrel(T, T_ref) <= 1e-13 and maxrel(dT, dT_ref) <= 1e-12
    # per-site bound too (no site hides behind the largest one)
    ax = tuple(range(1, T.ndim))
    assert (np.abs(T - T_ref).max(axis=ax) <= 1e-13 * np.abs(tab).max()).all()
    # device arrays in place, value only
    Td, none = tm.ttable_interp(torch.from_numpy(NODES).cuda(), torch.from_numpy(tab).cuda(), torch.from_numpy(p).cuda(), deriv=False)
    assert none is None and np.array_equal(Td.cpu().numpy(), T)
    # mixed: host table, device parameters
    Tm, dTm = tm.ttable_interp(NODES, tab, torch.from_numpy(p).cuda())
    assert np.array_equal(Tm.cpu().numpy(), T) and np.array_equal(dTm.cpu().numpy(), dT)


def test_minimal_table_and_single_site(tm):
    rng = np.random.default_rng(12)
    tab = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    nodes = np.array([0.1, 0.2, 0.25, 0.4])
    for p in (0.1, 0.22, 0.4):
        T, dT = tm.ttable_interp(nodes, tab, np.array([p]))
        T_ref, dT_ref = ttable.interp_table(nodes, tab, [p])
        assert maxrel(T, T_ref) <= 1e-13 and maxrel(dT, dT_ref) <= 1e-12


def test_rejects_what_the_table_does_not_cover(tm):
    tab = np.zeros((len(NODES), 2), dtype=complex)
    for bad in (NODES[0] - 1e-9, NODES[-1] + 1e-9, np.nan):
        with pytest.raises(tm.TmError) as e:
            tm.ttable_interp(NODES, tab, np.array([0.1, bad, 0.2]))
        assert e.value.code == tm.TM_E_INVALID
    with pytest.raises(tm.TmError):
        tm.ttable_interp(NODES[:3], tab[:3], np.array([0.07]))
    with pytest.raises(tm.TmError):
        tm.ttable_interp(NODES[::-1].copy(), tab, np.array([0.07]))


def test_full_size_table_of_the_paper_lens(tm):
    """The paper's setting: lmax 6 full T-matrices (96 x 96) for every scatterer of the 56 x 56 lens from a 64-node radius table;
    sampled sites against the oracle, every site against two properties that hold at any size (the weights sum to one: a
    table that is constant in p is returned unchanged with zero derivative; linear in p: exact)."""
    import torch
    rng = np.random.default_rng(13)
    L, n_tab, n_out = 96, 64, 3136
    nodes = np.linspace(0.05, 0.25, n_tab)
    base = rng.standard_normal((L, L)) + 1j * rng.standard_normal((L, L))
    slope = rng.standard_normal((L, L)) + 1j * rng.standard_normal((L, L))
    tab = torch.from_numpy(np.stack([base + x * slope for x in nodes])).cuda()
    p = rng.uniform(0.05, 0.25, n_out)
    T, dT = tm.ttable_interp(torch.from_numpy(nodes).cuda(), tab, torch.from_numpy(p).cuda())
    torch.cuda.synchronize()
    pd = torch.from_numpy(p).cuda()[:, None, None]
    exact = torch.from_numpy(base).cuda()[None] + pd * torch.from_numpy(slope).cuda()[None]
    assert float((T - exact).abs().max()) <= 1e-12 * float(exact.abs().max())
    assert float((dT - torch.from_numpy(slope).cuda()[None]).abs().max()) <= 1e-9 * float(np.abs(slope).max())
    # a random table on sampled sites against the oracle
    tab2 = rng.standard_normal((n_tab, L, L)) + 1j * rng.standard_normal((n_tab, L, L))
    T2, dT2 = tm.ttable_interp(torch.from_numpy(nodes).cuda(), torch.from_numpy(tab2).cuda(), torch.from_numpy(p).cuda())
    pick = rng.choice(n_out, 40, replace=False)
    T_ref, dT_ref = ttable.interp_table(nodes, tab2, p[pick])
    assert maxrel(T2[torch.from_numpy(pick).cuda()].cpu().numpy(), T_ref) <= 1e-13
    assert maxrel(dT2[torch.from_numpy(pick).cuda()].cpu().numpy(), dT_ref) <= 1e-12


def test_radius_gradient_through_the_interpolated_table(tm):
    """PAPER.md:560 end to end: table of T(R) -> interpolated T_j, dT_j/dR on the device -> forward + adjoint solve ->
    tm_grad_tmatrix; against central differences of the oracle's dense solve with the oracle's interpolation of the oracle's
    table (the derivative of the INTERPOLATED model: exact to the difference's O(h^2) inside a piece)."""
    lmax = 2
    rng = np.random.default_rng(14)
    pos = W.lattice(4, 3)
    n = len(pos)
    nodes = np.linspace(0.08, 0.24, 17)
    radii = rng.uniform(0.1, 0.22, n)
    radii = nodes[np.searchsorted(nodes, radii) - 1] + rng.uniform(0.3, 0.7, n) * (nodes[1] - nodes[0])      # well inside a piece
    v = W.complex_normal((n, W.n_modes(lmax)), rng)
    tab_gpu = np.stack([tm.mie_tmatrix(lmax, K, r, 4.0) for r in nodes])
    T, dT = tm.ttable_interp(nodes, tab_gpu, radii)
    s = tm.Solver(pos, lmax, K)
    s.set_tmatrices(T, np.arange(n, dtype=np.int32), True)
    s.set_incident_plane(0.3, 0.2, 1.0, 0.5j)
    sol, _, rc = s.solve(1e-12, 40, 400)
    lam, _, rc2 = s.solve_adjoint(v, 1e-12, 40, 400)
    assert rc == 0 and rc2 == 0
    g = s.grad_tmatrix(dT, lam, sol)
    s.close()
    tab_or = np.stack([tmatrix.mie_tmatrix_diag(lmax, K, r, 4.0) for r in nodes])
    p_inc = incident.plane_wave_incident(lmax, K, pos, 0.3, 0.2, 1.0, 0.5j)
    type_of = np.arange(n)

    def J(rr):
        t, _ = ttable.interp_table(nodes, tab_or, rr)
        M = system.assemble_M(lmax, K, pos, t, type_of, True)
        return np.sum(v * system.solve_forward(M, t, type_of, True, p_inc))
    h = 1e-6
    for j in (0, 5, n - 1):
        rp, rm = radii.copy(), radii.copy()
        rp[j] += h
        rm[j] -= h
        ref = (J(rp) - J(rm)) / (2 * h)
        assert abs(g[j] - ref) <= 1e-6 * abs(ref)
