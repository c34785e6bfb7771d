"""Pins of oracle/ttable.py (T-matrix look-up table, reading R20) against what the mathematics fixes."""
import numpy as np
import pytest

from oracle import gradient, tmatrix, ttable

NODES = np.array([0.05, 0.08, 0.10, 0.13, 0.17, 0.19, 0.24, 0.25])          # not equidistant


def _cubic_table(rng, shape):
    c = rng.standard_normal((4,) + shape) + 1j * rng.standard_normal((4,) + shape)
    f = lambda x: c[0] + c[1] * x + c[2] * x ** 2 + c[3] * x ** 3            # noqa: E731
    df = lambda x: c[1] + 2 * c[2] * x + 3 * c[3] * x ** 2                   # noqa: E731
    return f, df


def test_cubics_are_reproduced_exactly_with_their_derivative_in_every_interval():
    rng = np.random.default_rng(1)
    f, df = _cubic_table(rng, (3, 3))
    tab = np.stack([f(x) for x in NODES])
    p = np.concatenate([[NODES[0], NODES[-1]], 0.5 * (NODES[:-1] + NODES[1:]), NODES[1:-1], rng.uniform(NODES[0], NODES[-1], 20)])
    T, dT = ttable.interp_table(NODES, tab, p)
    for j, pj in enumerate(p):
        assert np.abs(T[j] - f(pj)).max() <= 1e-13 * np.abs(f(pj)).max()
        assert np.abs(dT[j] - df(pj)).max() <= 1e-11 * np.abs(df(pj)).max()


def test_nodes_return_the_table_entries():
    rng = np.random.default_rng(2)
    tab = rng.standard_normal((len(NODES), 5)) + 1j * rng.standard_normal((len(NODES), 5))
    T, _ = ttable.interp_table(NODES, tab, NODES)
    assert np.abs(T - tab).max() <= 1e-14


def test_quartic_remainder_fixes_the_stencil():
    """f = x^4: f - P_3 = f''''/4! prod_b (p - x_b) = prod_b (p - x_b) over the four nodes USED; with the stencil of R20 that
    is nodes i-1..i+2 around the interval (clamped at the ends).  A stencil shifted by one node changes the value."""
    tab = (NODES ** 4).astype(complex)[:, None]
    n = len(NODES)
    for i in range(n - 1):
        p = 0.3 * NODES[i] + 0.7 * NODES[i + 1]
        i0 = min(max(i - 1, 0), n - 4)
        expected = p ** 4 - np.prod(p - NODES[i0:i0 + 4])
        T, dT = ttable.interp_table(NODES, tab, [p])
        assert abs(T[0, 0] - expected) <= 1e-15
        # the derivative of the remainder: d/dp prod_b (p - x_b) = sum_c prod_{b != c} (p - x_b)
        drem = sum(np.prod([p - NODES[i0 + b] for b in range(4) if b != c]) for c in range(4))
        assert abs(dT[0, 0] - (4 * p ** 3 - drem)) <= 1e-13
        for shift in (-1, 1):
            j0 = i0 + shift
            if 0 <= j0 <= n - 4:
                assert abs(T[0, 0] - (p ** 4 - np.prod(p - NODES[j0:j0 + 4]))) > 1e-9


def test_equals_a_library_polynomial_through_the_same_four_nodes():
    rng = np.random.default_rng(3)
    tab = rng.standard_normal(len(NODES)) + 1j * rng.standard_normal(len(NODES))
    for p in rng.uniform(NODES[0], NODES[-1], 12):
        i0 = ttable.stencil_start(NODES, p)
        x = NODES[i0:i0 + 4]
        cr, ci = np.polyfit(x - x[0], tab[i0:i0 + 4].real, 3), np.polyfit(x - x[0], tab[i0:i0 + 4].imag, 3)
        val = np.polyval(cr, p - x[0]) + 1j * np.polyval(ci, p - x[0])
        der = np.polyval(np.polyder(cr), p - x[0]) + 1j * np.polyval(np.polyder(ci), p - x[0])
        T, dT = ttable.interp_table(NODES, tab[:, None], [p])
        assert abs(T[0, 0] - val) <= 1e-11 and abs(dT[0, 0] - der) <= 1e-9


def test_weights_sum_to_one_and_derivative_weights_to_zero():
    rng = np.random.default_rng(4)
    for p in rng.uniform(NODES[0], NODES[-1], 10):
        i0 = ttable.stencil_start(NODES, p)
        w, dw = ttable.lagrange_weights(NODES[i0:i0 + 4], p)
        assert abs(w.sum() - 1) <= 1e-13 and abs(dw.sum()) <= 1e-10


def test_converges_to_the_mie_tmatrix_at_fourth_order_and_its_derivative_at_third():
    """The table of Lorenz-Mie T(R) (eps_r = 4, lmax 2), sup norm over 151 radii: halving the node spacing divides the
    interpolation error by ~16 and the derivative's by ~8 (cubic interpolation)."""
    lmax, k, eps = 2, 2 * np.pi, 4.0
    probe = np.linspace(0.1, 0.2, 151)
    exact = np.stack([tmatrix.mie_tmatrix_diag(lmax, k, r, eps) for r in probe])
    dexact = np.stack([gradient.mie_dT_dR(lmax, k, r, eps, h=1e-3) for r in probe])
    errs, derrs = [], []
    for n in (33, 65, 129):
        nodes = np.linspace(0.05, 0.25, n)
        tab = np.stack([tmatrix.mie_tmatrix_diag(lmax, k, r, eps) for r in nodes])
        T, dT = ttable.interp_table(nodes, tab, probe)
        errs.append(np.abs(T - exact).max())
        derrs.append(np.abs(dT - dexact).max())
    assert 11 <= errs[0] / errs[1] <= 20 and 11 <= errs[1] / errs[2] <= 20
    assert 6.5 <= derrs[0] / derrs[1] <= 10.5 and 6.5 <= derrs[1] / derrs[2] <= 10.5
    assert errs[2] <= 1e-6


def test_outside_the_table_and_bad_tables_raise():
    tab = np.zeros((len(NODES), 2), dtype=complex)
    for p in (NODES[0] - 1e-9, NODES[-1] + 1e-9, np.nan):
        with pytest.raises(ValueError):
            ttable.interp_table(NODES, tab, [p])
    with pytest.raises(ValueError):
        ttable.interp_table(NODES[:3], tab[:3], [0.07])
    with pytest.raises(ValueError):
        ttable.interp_table(NODES[::-1], tab, [0.07])
