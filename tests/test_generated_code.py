"""CPU pins of the PRODUCT's build-time generated code against the oracle (no GPU needed):
the straight-line coplanar pair code is compiled as host C++ (tests/hostcheck_coplanar.cpp) and the general-kernel
term tables are evaluated with numpy; both must reproduce the oracle's translation block (PAPER.md Eqs. I16-I21)."""
import os
import re
import subprocess

import numpy as np
import pytest

from oracle import special as sp, translation as tr
from oracle.modes import mode_list, n_modes
from oracle.vswf import cart_to_sph

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GEN = os.path.join(ROOT, "paper_2107_09879_b200", "csrc", "generated")
K = 2 * np.pi


@pytest.mark.parametrize("lmax", [1, 2, 3])
def test_generated_coplanar_pair_code_matches_oracle_block(lmax, tmp_path):
    exe = str(tmp_path / f"hostcheck{lmax}")
    subprocess.check_call(["g++", "-O1", f"-DLMAX={lmax}", "-o", exe, os.path.join(ROOT, "tests", "hostcheck_coplanar.cpp")])
    rng = np.random.default_rng(40 + lmax)
    L = n_modes(lmax)
    for d in ([0.5, 0.0], [0.0, -0.5], [-1.7, 2.9], rng.uniform(-40, 40, 2), rng.uniform(-3, 3, 2)):
        x = rng.standard_normal(L) + 1j * rng.standard_normal(L)
        inp = f"{float(d[0])!r} {float(d[1])!r}\n" + "\n".join(f"{float(z.real)!r} {float(z.imag)!r}" for z in x) + "\n"
        out = subprocess.run([exe], input=inp, capture_output=True, text=True, check=True).stdout
        u = np.array([complex(*map(float, ln.split())) for ln in out.strip().splitlines()])
        ref = tr.block(lmax, K, np.array([d[0], d[1], 0.0]), np.zeros(3)) @ x
        assert np.abs(u - ref).max() <= 2e-13 * np.abs(ref).max()


@pytest.mark.parametrize("lmax", [1, 2, 3])
def test_generated_3d_pair_code_matches_oracle_block(lmax, tmp_path):
    exe = str(tmp_path / f"hostcheck3d{lmax}")
    subprocess.check_call(["g++", "-O1", f"-DLMAX={lmax}", "-o", exe, os.path.join(ROOT, "tests", "hostcheck_general3d.cpp")])
    rng = np.random.default_rng(50 + lmax)
    L = n_modes(lmax)
    for d in ([0.3, -0.4, 0.8], [0.0, 0.0, 1.2], [0.0, 0.0, -0.7], [1.0, 0.5, 0.0], rng.uniform(-30, 30, 3), rng.uniform(-3, 3, 3)):
        x = rng.standard_normal(L) + 1j * rng.standard_normal(L)
        inp = " ".join(repr(float(v)) for v in d) + "\n" + "\n".join(f"{float(z.real)!r} {float(z.imag)!r}" for z in x) + "\n"
        out = subprocess.run([exe], input=inp, capture_output=True, text=True, check=True).stdout
        u = np.array([complex(*map(float, ln.split())) for ln in out.strip().splitlines()])
        ref = tr.block(lmax, K, np.array(d, dtype=float), np.zeros(3)) @ x
        assert np.abs(u - ref).max() <= 2e-13 * np.abs(ref).max()


@pytest.mark.parametrize("lmax", [4, 5, 6])
def test_generated_four_sector_coplanar_code_matches_oracle_block(lmax, tmp_path):
    exe = str(tmp_path / f"hostcheck4_{lmax}")
    subprocess.check_call(["g++", "-O0", f"-DLMAX={lmax}", "-o", exe, os.path.join(ROOT, "tests", "hostcheck_coplanar4.cpp")])
    rng = np.random.default_rng(60 + lmax)
    L = n_modes(lmax)
    for d in ([0.5, 0.0], [0.0, -0.5], rng.uniform(-20, 20, 2)):
        x = rng.standard_normal(L) + 1j * rng.standard_normal(L)
        inp = f"{float(d[0])!r} {float(d[1])!r}\n" + "\n".join(f"{float(z.real)!r} {float(z.imag)!r}" for z in x) + "\n"
        out = subprocess.run([exe], input=inp, capture_output=True, text=True, check=True).stdout
        u = np.array([complex(*map(float, ln.split())) for ln in out.strip().splitlines()])
        ref = tr.block(lmax, K, np.array([d[0], d[1], 0.0]), np.zeros(3)) @ x
        assert np.abs(u - ref).max() <= 5e-13 * np.abs(ref).max()


def _parse_table(text, name, conv):
    m = re.search(name + r"\[\d+\] = \{(.*?)\};", text, flags=re.S)
    return [conv(t) for t in m.group(1).replace("\n", " ").split(",") if t.strip()]


@pytest.mark.parametrize("lmax", [1, 2, 3, 4])
def test_generated_general_term_table_matches_oracle_block(lmax):
    text = open(os.path.join(GEN, "tm_tables_gen.h")).read()
    tag = f"L{lmax}"
    rp = _parse_table(text, f"tm_rowptr_{tag}", int)
    col = _parse_table(text, f"tm_col_{tag}", int)
    qq = _parse_table(text, f"tm_q_{tag}", int)
    ip = _parse_table(text, f"tm_ipow_{tag}", int)
    val = _parse_table(text, f"tm_val_{tag}", float)
    modes = mode_list(lmax)
    L = n_modes(lmax)
    d = np.array([0.7, -1.3, 0.45])
    r, th, ph = cart_to_sph(d)
    h = [sp.sph_h1(q, K * r) for q in range(2 * lmax + 1)]
    B = np.zeros((L, L), dtype=complex)
    for b in range(L):
        for t in range(rp[b], rp[b + 1]):
            a = col[t]
            mu = modes[a][1] - modes[b][1]
            B[b, a] += (1j) ** ip[t] * val[t] * h[qq[t]] * sp.pbar(qq[t], abs(mu), np.cos(th)) * np.exp(1j * mu * ph)
    ref = tr.block(lmax, K, d, np.zeros(3))
    assert np.abs(B - ref).max() <= 1e-13 * np.abs(ref).max()


def _load_generator():
    import importlib.util
    spec = importlib.util.spec_from_file_location("tm_gen_tables", os.path.join(ROOT, "paper_2107_09879_b200", "csrc", "gen_tables.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def test_frame_rotation_is_a_quarter_turn():
    """The generator's frame change F' -> F'' (z'' = pair axis): real, orthogonal (all Ybar_lm have the same norm), four
    applications give the identity, and it carries the direction x' onto z'': Ybar_l0 of the pole is the only non-zero
    harmonic there, so column m' must reproduce Ybar_{l,m'}(x') = Pbar_l^{|m'|}(0) up to the pole value sqrt((2l+1)/2)."""
    g = _load_generator()
    for l in (1, 2, 3, 6):
        D = np.array(g.frame_rotation(l).tolist(), dtype=float)
        n = 2 * l + 1
        assert np.abs(D @ D.T - np.eye(n)).max() < 1e-14
        assert np.abs(np.linalg.matrix_power(D, 4) - np.eye(n)).max() < 1e-13
        pole = np.sqrt((2 * l + 1) / 2.0)
        for j, m in enumerate(range(-l, l + 1)):
            want = float(sp.pbar(l, abs(m), 0.0))
            assert abs(D[l, j] * pole - want) < 1e-14          # row m'' = 0


@pytest.mark.parametrize("lmax", [1, 2, 3])
def test_axial_factorisation_reproduces_the_oracle_block(lmax):
    """u = A x for an in-plane pair through the generator's factorisation  K_q = Gout Z''_q G  (numpy evaluation of the
    returned sparse factors, both halves, with the kernel's +- staging and phase rotation) against the oracle block."""
    g = _load_generator()
    md = g.modes(lmax)
    idx = {t: i for i, t in enumerate(md)}
    L = len(md)
    rng = np.random.default_rng(70 + lmax)
    ipow = np.array([1j ** p for (_, _, p) in md])
    for d in ([0.5, 0.0], [-1.7, 2.9], rng.uniform(-6, 6, 2)):
        x = rng.standard_normal(L) + 1j * rng.standard_normal(L)
        r = float(np.hypot(d[0], d[1]))
        phi = float(np.arctan2(d[1], d[0]))
        hq = np.array([complex(sp.sph_h1(q, K * r)) for q in range(2 * lmax + 1)])
        xt = ipow * x * np.exp(1j * np.array([m for (_, m, _) in md]) * phi)        # x~' = e^{i m phi} i^p x
        ut = np.zeros(L, dtype=complex)
        for (slots, slots2, G, entries, Gout) in g.coplanar_axial(lmax):
            n = len(slots)
            xs = np.array([xt[idx[(l, am, p)]] + {"0": 0, "+": 1, "-": -1}[k] * xt[idx[(l, -am, p)]] for (l, am, p, k) in slots])
            w = np.array([sum(float(v) * xs[c] for (c, v) in row) for row in G])
            t = np.zeros(n, dtype=complex)
            for (i, j), lst in entries.items():
                t[i] += sum(float(v) * hq[q] for (q, v) in lst) * w[j]
            u = np.array([sum(float(v) * t[c] for (c, v) in row) for row in Gout])
            for k_, (l, am, p, kind) in enumerate(slots):
                if kind == "0":
                    ut[idx[(l, 0, p)]] += u[k_]
                else:
                    sg = 1 if kind == "+" else -1
                    ut[idx[(l, am, p)]] += 0.5 * u[k_]
                    ut[idx[(l, -am, p)]] += 0.5 * sg * u[k_]
        u_full = np.conj(ipow) * np.exp(-1j * np.array([m for (_, m, _) in md]) * phi) * ut
        ref = tr.block(lmax, K, np.array([d[0], d[1], 0.0]), np.zeros(3)) @ x
        assert np.abs(u_full - ref).max() <= 2e-13 * np.abs(ref).max()


@pytest.mark.parametrize("lmax", [1, 2, 3, 5])
def test_generated_gradient_tables_match_oracle_derivative(lmax):
    """The product's analytic position derivative  dA/dd_alpha = k D^alpha A^ext  (gen_tables.py: gradient_entries; one
    all-pairs product at lmax + 1 and a constant sparse matrix) against the oracle's chain-rule derivative of Eq. I17
    (oracle/translation.py: d_block, itself pinned by central differences): two independent routes to the same matrix."""
    text = open(os.path.join(GEN, "tm_tables_gen.h")).read()
    tag = f"L{lmax}"
    al = _parse_table(text, f"tm_grad_alpha_{tag}", int)
    row = _parse_table(text, f"tm_grad_row_{tag}", int)
    col = _parse_table(text, f"tm_grad_col_{tag}", int)
    re_ = _parse_table(text, f"tm_grad_re_{tag}", float)
    im_ = _parse_table(text, f"tm_grad_im_{tag}", float)
    L, Le = n_modes(lmax), n_modes(lmax + 1)
    D = np.zeros((3, L, Le), dtype=complex)
    for a, r, c, x, y in zip(al, row, col, re_, im_):
        D[a, r, c] += x + 1j * y
    ext = mode_list(lmax + 1)
    cols = np.array([ext.index(t) for t in mode_list(lmax)])           # the lmax modes inside the lmax + 1 ordering
    rng = np.random.default_rng(80 + lmax)
    for d in (rng.uniform(-2, 2, 3), np.array([0.7, -0.2, 0.0]), np.array([0.0, 0.0, 0.9])):
        Aext = tr.block(lmax + 1, K, d, np.zeros(3))[:, cols]          # rows l' <= lmax + 1, source columns l <= lmax
        ref = tr.d_block(lmax, K, d, np.zeros(3))
        for a in range(3):
            got = K * D[a] @ Aext
            assert np.abs(got - ref[a]).max() <= 1e-12 * np.abs(ref[a]).max(), (lmax, a)


@pytest.mark.parametrize("lmax", [1, 2, 3, 4, 6])
def test_generated_rotation_based_3d_pair_code_matches_oracle_block(lmax, tmp_path):
    """Generated rotation - axial translation - rotation code for arbitrary pair directions (tm_rot3d_gen.cuh, the AUTO kernel
    of non-planar layouts at every lmax) compiled as host C++: u = A_ji x against the oracle block, including pairs along
    +-z (theta = 0, pi: phi undefined), in the plane, along -x (phi = pi) and far apart (k r ~ 200)."""
    exe = str(tmp_path / f"hostcheck_rot3d_{lmax}")
    subprocess.check_call(["g++", "-O0" if lmax > 4 else "-O1", f"-DLMAX={lmax}", "-o", exe, os.path.join(ROOT, "tests", "hostcheck_rot3d.cpp")])
    rng = np.random.default_rng(50 + lmax)
    L = n_modes(lmax)
    for d in ([0.3, -0.4, 0.8], [0.0, 0.0, 1.2], [0.0, 0.0, -0.7], [1.0, 0.5, 0.0], [-0.6, 0.0, 0.0], rng.uniform(-30, 30, 3), rng.uniform(-3, 3, 3)):
        x = rng.standard_normal(L) + 1j * rng.standard_normal(L)
        inp = " ".join(repr(float(v)) for v in d) + "\n" + "\n".join(f"{float(z.real)!r} {float(z.imag)!r}" for z in x) + "\n"
        out = subprocess.run([exe], input=inp, capture_output=True, text=True, check=True).stdout
        u = np.array([complex(*map(float, ln.split())) for ln in out.strip().splitlines()])
        ref = tr.block(lmax, K, np.array(d, dtype=float), np.zeros(3)) @ x
        assert np.abs(u - ref).max() <= 2e-13 * np.abs(ref).max()


@pytest.mark.parametrize("lmax", [4, 5, 6])
def test_generated_warp_split_3d_pair_code_matches_oracle_block(lmax, tmp_path):
    """Generated warp-split rotation-based code (tm_rot3d_ws_gen.cuh: the AUTO kernel of non-planar layouts at lmax 4..6) compiled as
    host C++ - phase A, phase B in place, then every owner part's phase C and unmix - against the oracle block, including pairs along
    +-z, in the plane, along -x and far apart."""
    exe = str(tmp_path / f"hostcheck_rot3d_ws_{lmax}")
    subprocess.check_call(["g++", "-O0", f"-DLMAX={lmax}", "-o", exe, os.path.join(ROOT, "tests", "hostcheck_rot3d_ws.cpp")])
    rng = np.random.default_rng(50 + lmax)
    L = n_modes(lmax)
    for d in ([0.3, -0.4, 0.8], [0.0, 0.0, 1.2], [0.0, 0.0, -0.7], [1.0, 0.5, 0.0], [-0.6, 0.0, 0.0], rng.uniform(-30, 30, 3), rng.uniform(-3, 3, 3)):
        x = rng.standard_normal(L) + 1j * rng.standard_normal(L)
        inp = " ".join(repr(float(v)) for v in d) + "\n" + "\n".join(f"{float(z.real)!r} {float(z.imag)!r}" for z in x) + "\n"
        out = subprocess.run([exe], input=inp, capture_output=True, text=True, check=True).stdout
        u = np.array([complex(*map(float, ln.split())) for ln in out.strip().splitlines()])
        ref = tr.block(lmax, K, np.array(d, dtype=float), np.zeros(3)) @ x
        assert np.abs(u - ref).max() <= 2e-13 * np.abs(ref).max()
