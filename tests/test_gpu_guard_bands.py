"""Memory-safety evidence without compute-sanitizer (closed on this GPU pool): every caller-owned DEVICE buffer of the path - inputs,
outputs and the Krylov workspace, sized exactly as tm_workspace_bytes says - sits inside a larger tensor whose margins hold a sentinel
pattern; after incident expansion, forward / adjoint solves, operator applications, field evaluation, the sensitivities and the
allocation-free field entry point on RAGGED shapes (windows that are no multiple of a tile, a one-scatterer window, a point count
that is no multiple of a block) the margins must be untouched and the interiors must agree with host-buffer runs of the same calls.
The library's INTERNAL device buffers get the same treatment through tm_debug_guards (include/tm.h), switched on for this module:
every block its allocator hands out (positions, tables, chunk partials, Krylov state, the auxiliary contexts of tm_grad_positions
and tm_solve_multi, quadrature scratch of the beam expansions) carries sentinel margins that are compared on free and on query."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2107_09879_b200 import workloads as W  # noqa: E402

GUARD = 4096          # bytes on each side


@pytest.fixture(scope="module")
def tm():
    import torch
    assert torch.cuda.is_available()
    from paper_2107_09879_b200 import libtm
    libtm.lib()
    return libtm


@pytest.fixture(autouse=True)
def internal_guards(tm):
    bad0, n0 = tm.debug_guards(1)
    yield
    import os
    bad, n = tm.debug_guards(-1 if os.environ.get("TM_DEBUG_GUARDS") == "1" else 0)      # (conftest.py keeps them on for the session)
    assert n > n0, "no internal block was guarded"
    assert bad == bad0 == 0, f"{bad} damaged margin(s) around internal device buffers"


class Guarded:
    """A device buffer of `nbytes` bytes with sentinel margins; .view(dtype, shape) gives the interior as a tensor."""

    def __init__(self, nbytes):
        import torch
        pad = (-nbytes) % 256
        self.raw = torch.full((GUARD + nbytes + pad + GUARD,), 0xA5, dtype=torch.uint8, device="cuda")
        self.nbytes, self.pad = nbytes, pad

    def view(self, dtype, shape):
        return self.raw[GUARD:GUARD + self.nbytes].view(dtype).reshape(shape)

    def interior_bytes(self):
        return self.raw[GUARD:GUARD + self.nbytes]

    def intact(self):
        import torch
        lo, hi = self.raw[:GUARD], self.raw[GUARD + self.nbytes:]
        return bool(torch.all(lo == 0xA5)) and bool(torch.all(hi == 0xA5))


@pytest.mark.parametrize("lmax,planar,prec", [(3, True, "fp64"), (3, False, "fp64"), (6, True, "fp64"), (5, False, "mixed"), (2, True, "fp32")])
def test_no_write_outside_caller_buffers(tm, lmax, planar, prec):
    import torch
    rng = np.random.default_rng(900 + lmax)
    n = 167                                                    # prime: no multiple of 32 / 64 / 128 / 256
    w = W.cloud_workload(n, seed=90 + lmax, lmax=lmax, planar=planar, n_win=1)
    wp = np.array([0, 1, 70, n], dtype=np.int32)               # one-scatterer window + ragged windows
    L = W.n_modes(lmax)
    precision = {"fp64": tm.TM_FP64, "fp32": tm.TM_FP32, "mixed": tm.TM_MIXED}[prec]
    tol = 1e-5 if prec == "fp32" else 1e-9
    restart, max_iter = 37, 600
    s = tm.Solver(w["pos"], lmax, W.K_B, win_ptr=wp, precision=precision)
    T = np.stack([tm.mie_tmatrix(lmax, W.K_B, r, 4.0) for r in w["radii"]])
    s.set_tmatrices(T, w["type_of"], True)
    s.set_incident_plane(0.4, 1.1, 0.8, 0.3 - 0.5j)
    # host-buffer reference run of the same calls
    ref_s, _, rc = s.solve(tol, restart, max_iter)
    wv = rng.standard_normal((n, L)) + 1j * rng.standard_normal((n, L))
    ref_l, _, rc2 = s.solve_adjoint(wv, tol, restart, max_iter)
    assert rc == 0 and rc2 == 0
    pts = rng.uniform(-6, 6, (77, 3)) + np.array([0.0, 0.0, 12.0])
    ref_E = s.fields(pts, ref_s)
    ref_y = s.matvec(wv, 1)
    # guarded device buffers
    g_ws = Guarded(s.workspace_bytes(restart))
    s.set_workspace(g_ws.raw[GUARD:GUARD + g_ws.nbytes + g_ws.pad])          # 256-byte aligned interior (torch allocations are 512-aligned)
    g = {k: Guarded(b) for k, b in dict(s=n * L * 16, lam=n * L * 16, w=n * L * 16, y=n * L * 16, p=n * L * 16, pts=77 * 24,
                                        E=77 * 48, E2=77 * 48, pos=n * 24, gx=n * 48).items()}
    d_s, d_lam, d_w = g["s"].view(torch.complex128, (n, L)), g["lam"].view(torch.complex128, (n, L)), g["w"].view(torch.complex128, (n, L))
    d_y, d_p = g["y"].view(torch.complex128, (n, L)), g["p"].view(torch.complex128, (n, L))
    d_pts, d_E, d_E2 = g["pts"].view(torch.float64, (77, 3)), g["E"].view(torch.complex128, (77, 3)), g["E2"].view(torch.complex128, (77, 3))
    d_pos, d_gx = g["pos"].view(torch.float64, (n, 3)), g["gx"].view(torch.complex128, (n, 3))
    d_w.copy_(torch.from_numpy(wv)); d_pts.copy_(torch.from_numpy(pts)); d_pos.copy_(torch.from_numpy(w["pos"]))
    s.set_incident_plane(0.4, 1.1, 0.8, 0.3 - 0.5j)
    s.get_incident(out=d_p)
    _, _, rc = s.solve(tol, restart, max_iter, out=d_s)
    _, _, rc2 = s.solve_adjoint(d_w, tol, restart, max_iter, out=d_lam)
    s.matvec(d_w, 1, out=d_y)
    s.fields(d_pts, d_s, tm.TM_FIELD_E_SCA, out=d_E)
    s.grad_positions(d_lam, d_s, out=d_gx)
    tm.fields_static(lmax, W.K_B, d_pos, d_s, d_pts, tm.TM_FIELD_E_SCA, out=d_E2, stream=None)
    torch.cuda.synchronize()
    assert rc == 0 and rc2 == 0
    for name, buf in list(g.items()) + [("workspace", g_ws)]:
        assert buf.intact(), f"write outside the caller's {name} buffer"
    # inputs are not modified
    assert np.array_equal(d_w.cpu().numpy(), wv) and np.array_equal(d_pts.cpu().numpy(), pts)
    # and the device-buffer results are those of the host-buffer run
    etol = 2e-4 if prec == "fp32" else 1e-8
    assert np.abs(d_s.cpu().numpy() - ref_s).max() <= etol * np.abs(ref_s).max()
    assert np.abs(d_lam.cpu().numpy() - ref_l).max() <= etol * np.abs(ref_l).max()
    assert np.abs(d_y.cpu().numpy() - ref_y).max() <= (1e-5 if prec == "fp32" else 1e-12) * np.abs(ref_y).max()
    assert np.abs(d_E.cpu().numpy() - ref_E).max() <= etol * np.abs(ref_E).max()
    assert np.abs(d_E2.cpu().numpy() - d_E.cpu().numpy()).max() <= 1e-12 * np.abs(ref_E).max()
    # several right-hand sides at once (tm_solve_multi): guarded stack of inputs and outputs
    g_r, g_o = Guarded(3 * n * L * 16), Guarded(3 * n * L * 16)
    d_r, d_o = g_r.view(torch.complex128, (3, n, L)), g_o.view(torch.complex128, (3, n, L))
    rhs = rng.standard_normal((3, n, L)) + 1j * rng.standard_normal((3, n, L))
    d_r.copy_(torch.from_numpy(rhs))
    _, _, rc3 = s.solve_multi(d_r, tol, restart, max_iter, out=d_o)
    torch.cuda.synchronize()
    assert rc3 == 0 and g_r.intact() and g_o.intact() and g_ws.intact()
    assert np.array_equal(d_r.cpu().numpy(), rhs)
    # beam expansions (quadrature scratch) and the incident field at the detector points
    s.set_incident_gauss(np.tile(np.array([0.3, -0.2, 0.1]), (3, 1)), 1.5, 1.0, 0.2j)
    s.get_incident(out=d_p)
    s.fields(d_pts, None, tm.TM_FIELD_E_INC, out=d_E)
    src = rng.uniform(-2, 2, (9, 3)); src[:, 2] = -3.0
    s.set_incident_jinc(src, rng.standard_normal((9, 2)) + 0j, src_ptr=[0, 2, 5, 9])
    s.get_incident(out=d_p)
    torch.cuda.synchronize()
    assert g["p"].intact() and g["E"].intact() and g["pts"].intact()
    bad, _ = tm.debug_guards()
    assert bad == 0
    s.close()


def test_guard_detects_a_stray_write(tm):
    """Negative control of the checker itself: one byte past either end is seen."""
    pos = np.zeros((2, 3)); pos[1, 0] = 1.0
    tm.Solver(pos, 1, W.K_B).close()                 # (something for the module's internal-guard fixture to count)
    g = Guarded(1000)
    assert g.intact()
    g.raw[GUARD - 1] = 0
    assert not g.intact()
    g.raw[GUARD - 1] = 0xA5
    g.raw[GUARD + 1000] = 1
    assert not g.intact()
