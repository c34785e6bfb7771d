"""Host logic of the Nyquist window decomposition: CPU only, no device calls."""
import numpy as np

from paper_2107_09879_b200 import nyquist, workloads as W

K = W.K_B


def test_sample_grid_is_the_half_wavelength_lattice():
    xs, ys = nyquist.sample_grid(K, (-2.0, 2.0), (-1.0, 1.26))
    assert np.allclose(np.diff(xs), 0.5) and np.allclose(np.diff(ys), 0.5)
    assert xs[0] == -2.0 and xs[-1] == 2.0 and ys[0] == -1.0 and ys[-1] == 1.0
    assert np.allclose(xs / 0.5, np.round(xs / 0.5))          # x_i = i lambda/2 (origin on the grid)


def test_sources_carry_pi_over_two_times_the_sample():
    src, amp, gi = nyquist.jinc_sources(K, (-1, 1), (-1, 1), -0.5, lambda x, y: (1.0 + 0 * x, 2j * np.ones_like(y)))
    assert src.shape == (25, 3) and np.all(src[:, 2] == -0.5)
    assert np.allclose(amp[:, 0], 1.0) and np.allclose(amp[:, 1], 2j)       # samples; the (pi/2) of reading R17 is the library's
    assert gi.min() == 0 and gi.max() == 4


def test_plan_and_batch_bookkeeping():
    pos = W.lattice(20, 20)                                   # 10 x 10 wavelengths
    src, amp, gi = nyquist.jinc_sources(K, (-5, 5), (-5, 5), 0.0, lambda x, y: (np.exp(-(x * x + y * y) / 9.0), 0 * x))
    plans = nyquist.plan_windows(pos, src, gi, group=6, padding=1.5)
    allsrc = np.concatenate([p[0] for p in plans])
    assert np.array_equal(np.sort(allsrc), np.arange(src.shape[0]))            # every source in exactly one window
    for sidx, scat in plans:
        lo, hi = src[sidx, :2].min(axis=0) - 1.5, src[sidx, :2].max(axis=0) + 1.5
        inside = np.all((pos[:, :2] >= lo - 1e-12) & (pos[:, :2] <= hi + 1e-12), axis=1)
        assert np.array_equal(np.nonzero(inside)[0], scat)
        assert np.ptp(gi[sidx, 0]) < 6 and np.ptp(gi[sidx, 1]) < 6
    b = nyquist.build_batch(pos, src, amp, plans)
    nw = len(b["win_ptr"]) - 1
    assert nw == len(plans) and b["win_ptr"][-1] == b["pos"].shape[0] == b["scat_index"].size
    assert b["src_ptr"][-1] == src.shape[0] and len(b["src_ptr"]) == nw + 1
    assert b["pos"].shape[0] > pos.shape[0]                                    # padding duplicates scatterers
    assert np.array_equal(b["pos"], pos[b["scat_index"]])
    # larger padding -> every window grows
    plans2 = nyquist.plan_windows(pos, src, gi, group=6, padding=3.0)
    assert all(p2[1].size >= p1[1].size for p1, p2 in zip(plans, plans2))
