"""GPU: jinc-source expansion against the oracle, and the Nyquist window decomposition
against the undistributed solve (padding convergence, Fig. 1b in spirit)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import incident  # noqa: E402
from paper_2107_09879_b200 import workloads as W  # noqa: E402


@pytest.fixture(scope="module")
def tm():
    import torch
    assert torch.cuda.is_available()
    from paper_2107_09879_b200 import libtm
    libtm.lib()
    return libtm


from parity_metric import rel, rel_solve  # noqa: E402,F401  (L2 AND per-(l,p)-block / per-point max error; solutions: L2 AND max norm)


def test_jinc_incident_matches_oracle(tm):
    rng = np.random.default_rng(5)
    pos = W.random_cloud(14, seed=31)
    wp = np.array([0, 6, 14], dtype=np.int32)
    src = np.concatenate([rng.uniform(-2, 2, (5, 2)), np.full((5, 1), -1.5)], axis=1)
    src[1, :2] = pos[2, :2]                                   # a source straight below a scatterer (rho_T = 0)
    amp = rng.standard_normal((5, 2)) + 1j * rng.standard_normal((5, 2))
    sp = np.array([0, 2, 5], dtype=np.int32)
    s = tm.Solver(pos, 3, W.K_B, win_ptr=wp)
    s.set_incident_jinc(src, amp, sp)
    ref = np.concatenate([incident.jinc_sources_incident(3, W.K_B, pos[wp[i]:wp[i + 1]], src[sp[i]:sp[i + 1]], amp[sp[i]:sp[i + 1]])
                          for i in range(2)])
    assert rel(s.get_incident(), ref) <= 1e-11
    # samples instead of amplitudes: the library applies the Nyquist factor of reading R17 (oracle: incident.nyquist_sources)
    s.set_incident_jinc(src, amp, sp, samples=True)
    assert rel(s.get_incident(), 0.5 * np.pi * ref) <= 1e-11
    s.close()


def test_nyquist_decomposed_beam_equals_direct_beam_and_padding_converges(tm):
    from paper_2107_09879_b200 import nyquist
    w = W.config(2, scale=24)                                  # 24 x 24 lattice, 12 x 12 wavelengths, Mie library
    w0 = 1.5
    gauss = lambda x, y: (np.exp(-(x * x + y * y) / w0 ** 2), np.zeros_like(x))
    src, amp, gi = nyquist.jinc_sources(w["k"], (-6, 6), (-6, 6), 0.0, gauss, drop_below=1e-7)
    g = np.linspace(-5, 5, 9)
    pts = np.array([[a, b, 4.0] for a in g for b in g])
    # (1) undistributed: all sources, all scatterers == direct Gaussian-beam drive (Nyquist theorem, reading R17)
    E_full, info = nyquist.simulate(w, src, amp, gi, None, 0.0, pts, tol=1e-9)
    assert info["rc"] == 0 and info["n_windows"] == 1
    s = tm.Solver(w["pos"], w["lmax"], w["k"])
    T = np.stack([tm.mie_tmatrix(w["lmax"], w["k"], r, w["eps_r"]) for r in w["radii"]])
    s.set_tmatrices(T, w["type_of"], True)
    s.set_incident_gauss(np.zeros((1, 3)), w0, 1.0, 0.0)
    sol, _, rc = s.solve(1e-9, 50, 5000)
    E_direct = s.fields(pts, sol)
    s.close()
    assert rc == 0 and rel(E_full, E_direct) <= 1e-4
    # (2) distributed: groups of 6 x 6 samples (3 x 3 wavelengths), growing padding -> converges to the full solve
    errs = []
    for pad in (0.5, 2.0, 4.0):
        E, inf = nyquist.simulate(w, src, amp, gi, 6, pad, pts, tol=1e-9)
        assert inf["rc"] == 0 and inf["n_windows"] > 1
        errs.append(rel(E, E_full))
    # (resonant, strongly coupled lattice: the truncation error falls slowly - measured 0.26 / 0.18 / 0.11)
    assert errs[0] > errs[1] > errs[2] and errs[2] < 0.6 * errs[0], errs
    # windows that contain everything reproduce the full solve exactly (linearity: fields of the groups add up)
    E_big, _ = nyquist.simulate(w, src, amp, gi, 6, 30.0, pts, tol=1e-10)
    assert rel(E_big, E_full) <= 1e-6
