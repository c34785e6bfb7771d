"""tm_fields_static: the allocation-free entry point (static device scratch, include/tm.h) against the existing tm_fields path.

Collected LAST on purpose (the suite runs with `pytest -x`): a failure here must not hide other tests.  Passes alone in a fresh
process and after the other tests: the first call resolves the static array's address itself (cudaGetSymbolAddress, once per
device), and every call overwrites the part of the shared array it reads, so earlier contents do not matter."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2107_09879_b200 import workloads as W  # noqa: E402
from parity_metric import rel  # noqa: E402


@pytest.fixture(scope="module")
def tm():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2107_09879_b200 import libtm
    libtm.lib()
    return libtm


def test_fields_static_matches_tm_fields_on_two_calls_in_a_row(tm):
    import torch
    rng = np.random.default_rng(71)
    lmax, n = 3, 150
    L = W.n_modes(lmax)
    pos = W.random_cloud(n, seed=72)
    pts = rng.uniform(-6.0, 6.0, (700, 3)) + np.array([0.0, 0.0, 9.0])        # ragged tail of the 128-point blocks
    s1 = rng.standard_normal((n, L)) + 1j * rng.standard_normal((n, L))
    s2 = rng.standard_normal((n, L)) + 1j * rng.standard_normal((n, L))
    ctx = tm.Solver(pos, lmax, W.K_B)
    ref_E = ctx.fields(pts, s1, tm.TM_FIELD_E_SCA)                           # existing path (context scratch)
    ref_H = ctx.fields(pts, s2, tm.TM_FIELD_H_SCA)
    ctx.close()
    d_pos, d_pts = torch.from_numpy(pos).cuda(), torch.from_numpy(pts).cuda()
    d_s1, d_s2 = torch.from_numpy(s1).cuda(), torch.from_numpy(s2).cuda()
    out1 = torch.empty((pts.shape[0], 3), dtype=torch.complex128, device="cuda")
    out2 = torch.empty_like(out1)
    torch.cuda.synchronize()
    st = torch.cuda.current_stream().cuda_stream
    tm.fields_static_setup()
    # two calls in a row on one stream, sharing the static array: E of s1, then Z H of s2 (different data, different branch)
    tm.fields_static(lmax, W.K_B, d_pos, d_s1, d_pts, tm.TM_FIELD_E_SCA, out=out1, stream=st)
    tm.fields_static(lmax, W.K_B, d_pos, d_s2, d_pts, tm.TM_FIELD_H_SCA, out=out2, stream=st)
    torch.cuda.synchronize()
    assert rel(out1.cpu().numpy(), ref_E) <= 1e-12
    assert rel(out2.cpu().numpy(), ref_H) <= 1e-12
    # and once more the first one: the array now holds the second call's partial sums
    tm.fields_static(lmax, W.K_B, d_pos, d_s1, d_pts, tm.TM_FIELD_E_SCA, out=out2, stream=st)
    torch.cuda.synchronize()
    assert torch.equal(out1, out2)


def test_fields_static_lmax6_and_many_points(tm):
    """The paper's truncation and a point set large enough that the static array, not the heuristic, fixes the chunk count."""
    import torch
    rng = np.random.default_rng(73)
    lmax, n = 6, 70
    L = W.n_modes(lmax)
    pos = W.random_cloud(n, seed=74)
    pts = rng.uniform(-8.0, 8.0, (40000, 3)) + np.array([0.0, 0.0, 12.0])
    s = rng.standard_normal((n, L)) + 1j * rng.standard_normal((n, L))
    ctx = tm.Solver(pos, lmax, W.K_B)
    ref = ctx.fields(pts, s, tm.TM_FIELD_E_SCA)
    ctx.close()
    out = tm.fields_static(lmax, W.K_B, torch.from_numpy(pos).cuda(), torch.from_numpy(s).cuda(), torch.from_numpy(pts).cuda())
    torch.cuda.synchronize()
    assert rel(out.cpu().numpy(), ref) <= 1e-12


def test_fields_static_rejects_what_does_not_fit(tm):
    import torch
    pos = torch.zeros((2, 3), dtype=torch.float64, device="cuda")
    pos[1, 0] = 1.0
    s = torch.zeros((2, 6), dtype=torch.complex128, device="cuda")
    big = torch.ones((65537, 3), dtype=torch.float64, device="cuda")
    with pytest.raises(tm.TmError) as e:
        tm.fields_static(1, W.K_B, pos, s, big)
    assert e.value.code == tm.TM_E_INVALID and "65536" in str(e.value)
    with pytest.raises(tm.TmError) as e:                                      # host pointers are refused: nothing is copied
        tm.fields_static(1, W.K_B, pos, s, torch.ones((4, 3), dtype=torch.float64))
    assert e.value.code == tm.TM_E_INVALID
    ok = tm.fields_static(1, W.K_B, pos, s, big[:65536])                      # the stated maximum itself is served
    torch.cuda.synchronize()
    assert ok.shape == (65536, 3) and bool(torch.all(ok == 0))
