#!/usr/bin/env python3
"""Build-time generator for the constant part of the translation (addition-theorem) operator.

Product-side code: shares nothing with oracle/ (own Wigner-3j, own Legendre values).  It restates
PAPER.md:299-327 (Eqs. I16-I19) with the readings R3-R8 of DESIGN.md:

  [A_ji]_{b,a} = e^{i(m_a-m_b)phi} sum_q c(q;a->b) h_q^(1)(k r) Pbar_q^{|m_a-m_b|}(cos theta),
  (r, theta, phi) = x_j - x_i,   a = source mode (l,m,p), b = destination mode (l',m',p'),
  c = a5(l,m|l',m'|q) for p = p', b5(l,m|l',m'|q) for p != p'.

Outputs (written next to this file, under generated/):
  tm_tables_gen.h        sparse (row, col, q, value, is_imag) term lists for lmax = 1..6
                         (general 3-D kernel; value already includes nothing angle-dependent)
  tm_coplanar_gen.cuh    straight-line device code for the coplanar (theta = pi/2) specialisation,
                         lmax = 1..3, in the "tilde" basis x~ = i^p x where every coefficient is real,
                         split into the two mirror-parity halves (-1)^{l+m+p} = +-1 that coplanar
                         translations do not mix (structural identity S2).

Run:  python gen_tables.py            (build.py runs it when generated/ is missing or stale)
"""
import os
import sys
from fractions import Fraction
from math import comb, factorial

import mpmath as mp

mp.mp.dps = 40
HERE = os.path.dirname(os.path.abspath(__file__))
OUT = os.path.join(HERE, "generated")


# ----------------------------------------------------------------------------- mode bookkeeping
def n_modes(lmax):
    return 2 * lmax * (lmax + 2)


def modes(lmax):
    """flat order idx = p*(L/2) + l(l+1) - 1 + m  (reading R1, part of the ABI)."""
    return [(l, m, p) for p in (0, 1) for l in range(1, lmax + 1) for m in range(-l, l + 1)]


# ----------------------------------------------------------------------------- Wigner 3j
_w3j_cache = {}


def w3j(j1, j2, j3, m1, m2, m3):
    """Exact-rational Racah sum in binomial form; returns an mpf.
    (j1 j2 j3; m1 m2 m3) = (-1)^{j1-j2-m3} sqrt(D) sum_t (-1)^t / (t! (j3-j2+t+m1)! ...)"""
    key = (j1, j2, j3, m1, m2, m3)
    if key in _w3j_cache:
        return _w3j_cache[key]
    val = mp.mpf(0)
    if m1 + m2 + m3 == 0 and abs(j1 - j2) <= j3 <= j1 + j2 and abs(m1) <= j1 and abs(m2) <= j2 and abs(m3) <= j3:
        J = j1 + j2 + j3
        # squared prefactor as an exact fraction
        d2 = Fraction(factorial(J - 2 * j1) * factorial(J - 2 * j2) * factorial(J - 2 * j3), factorial(J + 1))
        d2 *= (factorial(j1 + m1) * factorial(j1 - m1) * factorial(j2 + m2) * factorial(j2 - m2)
               * factorial(j3 + m3) * factorial(j3 - m3))
        lo = max(0, j2 - j3 - m1, j1 - j3 + m2)
        hi = min(j1 + j2 - j3, j1 - m1, j2 + m2)
        s = Fraction(0)
        for t in range(lo, hi + 1):
            s += Fraction((-1) ** t, factorial(t) * factorial(j3 - j2 + t + m1) * factorial(j3 - j1 + t - m2)
                          * factorial(j1 + j2 - j3 - t) * factorial(j1 - t - m1) * factorial(j2 - t + m2))
        val = (-1) ** ((j1 - j2 - m3) % 2) * mp.sqrt(mp.mpf(d2.numerator) / mp.mpf(d2.denominator)) \
            * (mp.mpf(s.numerator) / mp.mpf(s.denominator))
    _w3j_cache[key] = val
    return val


# ----------------------------------------------------------------------------- Eq. I18 (repairs R5, R6)
def _iphase(l, m, lp, mp_, q):
    """(exponent of i) mod 4 of i^{|m-m'|-|m|-|m'|+l'-l+q} (-1)^{m-m'}."""
    e = abs(m - mp_) - abs(m) - abs(mp_) + lp - l + q + 2 * ((m - mp_) % 2)
    return e % 4


def _nrm(l, lp):
    return mp.sqrt(mp.mpf((2 * l + 1) * (2 * lp + 1)) / (2 * l * (l + 1) * lp * (lp + 1)))


def coupling(l, m, p, lp, mp_, pp, q):
    """-> (ipow, real magnitude incl. sign) with c = i^ipow * value; value = 0 when the term is absent."""
    if q < abs(m - mp_) or q > l + lp:
        return 0, mp.mpf(0)
    if p == pp:
        if q < abs(l - lp):
            return 0, mp.mpf(0)
        v = ((l * (l + 1) + lp * (lp + 1) - q * (q + 1)) * mp.sqrt(2 * q + 1) * _nrm(l, lp)
             * w3j(l, lp, q, m, -mp_, mp_ - m) * w3j(l, lp, q, 0, 0, 0))
    else:
        if q < abs(l - lp) + 1:
            return 0, mp.mpf(0)
        rad = (l + lp + 1 + q) * (l + lp + 1 - q) * (q + l - lp) * (q - l + lp) * (2 * q + 1)
        if rad <= 0:
            return 0, mp.mpf(0)
        v = mp.sqrt(rad) * _nrm(l, lp) * w3j(l, lp, q, m, -mp_, mp_ - m) * w3j(l, lp, q - 1, 0, 0, 0)
    return _iphase(l, m, lp, mp_, q), v


# ----------------------------------------------------------------------------- Pbar_q^mu(0), no Condon-Shortley phase (R2)
def pbar_at_zero(q, mu):
    if (q - mu) % 2:
        return mp.mpf(0)
    k = (q - mu) // 2
    # mu-th derivative at 0 of P_q(x) = 2^-q sum_k (-1)^k C(q,k) C(2q-2k,q) x^{q-2k}
    d = Fraction((-1) ** k * comb(q, k) * comb(2 * q - 2 * k, q) * factorial(mu), 2 ** q)
    n2 = Fraction((2 * q + 1) * factorial(q - mu), 2 * factorial(q + mu))
    return mp.mpf(d.numerator) / mp.mpf(d.denominator) * mp.sqrt(mp.mpf(n2.numerator) / mp.mpf(n2.denominator))


def lit(v):
    return repr(float(v))


# ----------------------------------------------------------------------------- general 3-D term lists
def general_terms(lmax):
    """[(b, a, q, ipow, value)] sorted by destination row b, then source column a, then q."""
    md = modes(lmax)
    out = []
    for b, (lp, mp_, pp) in enumerate(md):
        for a, (l, m, p) in enumerate(md):
            for q in range(0, 2 * lmax + 1):
                ip, v = coupling(l, m, p, lp, mp_, pp, q)
                if v != 0:
                    out.append((b, a, q, ip, v))
    return out


def emit_tables(lmaxes, path):
    with open(path, "w") as f:
        f.write("// GENERATED by gen_tables.py - do not edit.  Sparse constant part of Eqs. I16-I18 (PAPER.md:299-323).\n")
        f.write("// term t of row b (row_ptr[b] <= t < row_ptr[b+1]): A[b][col[t]] += i^ipow[t] * val[t] * h_q[t] * Pbar_q[t]^{|m_col - m_b|}\n")
        f.write("#pragma once\n#include <cstdint>\n\n")
        f.write("struct TmTermTable { int lmax; int n_terms; const int* row_ptr; const uint8_t* col; const uint8_t* q; const uint8_t* ipow; const double* val; };\n\n")
        for lmax in lmaxes:
            terms = general_terms(lmax)
            L = n_modes(lmax)
            rp = [0] * (L + 1)
            for t in terms:
                rp[t[0] + 1] += 1
            for b in range(L):
                rp[b + 1] += rp[b]
            tag = f"L{lmax}"
            f.write(f"static const int tm_rowptr_{tag}[{L + 1}] = {{{', '.join(map(str, rp))}}};\n")
            f.write(f"static const uint8_t tm_col_{tag}[{len(terms)}] = {{{', '.join(str(t[1]) for t in terms)}}};\n")
            f.write(f"static const uint8_t tm_q_{tag}[{len(terms)}] = {{{', '.join(str(t[2]) for t in terms)}}};\n")
            f.write(f"static const uint8_t tm_ipow_{tag}[{len(terms)}] = {{{', '.join(str(t[3]) for t in terms)}}};\n")
            f.write(f"static const double tm_val_{tag}[{len(terms)}] = {{\n")
            for s in range(0, len(terms), 6):
                f.write("  " + ", ".join(lit(t[4]) for t in terms[s:s + 6]) + ",\n")
            f.write("};\n\n")
            print(f"lmax={lmax}: L={L} general terms={len(terms)}", file=sys.stderr)
        emit_gradient_tables(f, [l for l in lmaxes if l + 1 in lmaxes])
        f.write(f"static const int tm_max_table_lmax = {max(lmaxes)};\n")
        f.write("static const TmTermTable tm_term_tables[] = {\n")
        for lmax in lmaxes:
            tag = f"L{lmax}"
            f.write(f"  {{{lmax}, (int)(sizeof(tm_col_{tag})), tm_rowptr_{tag}, tm_col_{tag}, tm_q_{tag}, tm_ipow_{tag}, tm_val_{tag}}},\n")
        f.write("};\n")


# ----------------------------------------------------------------------------- gradient of the translation operator
def gradient_entries(lmax):
    """Constant matrices of the analytic position derivative (PAPER.md:517-546 Eqs. IV2-IV6, :560 "can be computed
    analytically").  The regular wavefunctions obey  d/dx_alpha RPhi_b = k sum_b' D^alpha[b', b] RPhi_b'  with
    D^alpha = (1/k) d RgA(eps)/d eps_alpha at eps = 0, and only the q = 1 term of Eq. I17 is linear in eps:
        j_1(k eps) Pbar_1^0(cos theta) -> (k/3) sqrt(3/2) eps_z ,   j_1(k eps) Pbar_1^1 e^{+-i phi} -> (k/3) (sqrt(3)/2) (eps_x +- i eps_y).
    Differentiating  Phi_a(x - x_i) = sum_b A_ba(x_j - x_i) RPhi_b(x - x_j)  with respect to x_j gives
        d A(d) / d d_alpha = k D^alpha A^ext(d),
    A^ext = the translation operator with destination rows up to lmax + 1: the derivative of the operator is ONE ordinary
    all-pairs product at lmax + 1 followed by a constant sparse matrix per direction.
    Returns [(alpha, row b' in modes(lmax), col b in modes(lmax+1), complex value D^alpha[b', b])]."""
    md, mde = modes(lmax), modes(lmax + 1)
    cz = mp.sqrt(mp.mpf(3) / 2) / 3
    cx = mp.sqrt(mp.mpf(3)) / 2 / 3
    out = []
    for bp, (lp, mp_, pp) in enumerate(md):            # destination b'
        for b, (l, m, p) in enumerate(mde):             # source b
            ip, v = coupling(l, m, p, lp, mp_, pp, 1)
            if v == 0:
                continue
            c = (mp.mpc(0, 1) ** ip) * v
            mu = m - mp_
            if mu == 0:
                out.append((2, bp, b, c * cz))
            elif abs(mu) == 1:
                out.append((0, bp, b, c * cx))
                out.append((1, bp, b, c * cx * mp.mpc(0, mu)))
    return out


def emit_gradient_tables(f, lmaxes):
    f.write("// Gradient of the translation operator (gen_tables.py: gradient_entries):  dA/dd_alpha = k D^alpha A^ext,\n")
    f.write("// entry e: D^{alpha[e]}[row[e] (flat index at lmax), col[e] (flat index at lmax + 1)] = (re[e], im[e]).\n")
    f.write("struct TmGradTable { int lmax; int n; const uint8_t* alpha; const uint8_t* row; const uint8_t* col; const double* re; const double* im; };\n")
    for lmax in lmaxes:
        ent = gradient_entries(lmax)
        tag = f"L{lmax}"
        f.write(f"static const uint8_t tm_grad_alpha_{tag}[{len(ent)}] = {{{', '.join(str(e[0]) for e in ent)}}};\n")
        f.write(f"static const uint8_t tm_grad_row_{tag}[{len(ent)}] = {{{', '.join(str(e[1]) for e in ent)}}};\n")
        f.write(f"static const uint8_t tm_grad_col_{tag}[{len(ent)}] = {{{', '.join(str(e[2]) for e in ent)}}};\n")
        f.write(f"static const double tm_grad_re_{tag}[{len(ent)}] = {{{', '.join(lit(mp.re(e[3])) for e in ent)}}};\n")
        f.write(f"static const double tm_grad_im_{tag}[{len(ent)}] = {{{', '.join(lit(mp.im(e[3])) for e in ent)}}};\n")
        print(f"lmax={lmax}: gradient entries={len(ent)}", file=sys.stderr)
    f.write("static const TmGradTable tm_grad_tables[] = {\n")
    for lmax in lmaxes:
        tag = f"L{lmax}"
        f.write(f"  {{{lmax}, (int)(sizeof(tm_grad_alpha_{tag})), tm_grad_alpha_{tag}, tm_grad_row_{tag}, tm_grad_col_{tag}, tm_grad_re_{tag}, tm_grad_im_{tag}}},\n")
    f.write("};\n\n")


# ----------------------------------------------------------------------------- coplanar specialisation
def coplanar_rows(lmax):
    """Real coefficients of the tilde-basis coplanar operator.
    K[b][q] = [(a, value)] with  u~'_b = sum_q h_q sum_a value * x~'_a,
    x~'_a = e^{i m_a phi} i^{p_a} x_a,   u_b = (-i)^{p_b} e^{-i m_b phi} u~'_b."""
    md = modes(lmax)
    L = len(md)
    K = [[[] for _ in range(2 * lmax + 1)] for _ in range(L)]
    for b, (lp, mp_, pp) in enumerate(md):
        for a, (l, m, p) in enumerate(md):
            for q in range(0, 2 * lmax + 1):
                ip, v = coupling(l, m, p, lp, mp_, pp, q)
                if v == 0:
                    continue
                v = v * pbar_at_zero(q, abs(m - mp_))
                if v == 0:
                    continue
                tot = (ip + (pp - p)) % 4              # i^{p_b - p_a} * i^ipow must be real
                assert tot % 2 == 0, (b, a, q, ip)
                assert (l + m + p) % 2 == (lp + mp_ + pp) % 2, "mirror parity must be conserved (S2)"
                K[b][q].append((a, v if tot == 0 else -v))
    return K


def coplanar_sym(lmax):
    """The coplanar operator in the pair frame, reduced by BOTH mirror symmetries of a pair:
      * z -> -z  (structural identity S2): modes split into the halves (-1)^{l+m+p} = +-1;
      * y' -> -y' in the frame whose x' axis is the pair axis: K_q[(l',-m',p'),(l,-m,p)] = +-K_q[(l',m',p'),(l,m,p)]
        (+ for p = p', - for p != p'), so in the basis x^+- = x'_{l,m,p} +- x'_{l,-m,p} (m > 0) each half splits
        again into two sectors that do not couple.
    Returns per half: slots [(l, am, p, kind)], kind in '0+-', and Knew[q][row_slot] = [(col_slot, value)]."""
    md = modes(lmax)
    L = len(md)
    idx = {t: i for i, t in enumerate(md)}
    rows = coplanar_rows(lmax)
    nq = 2 * lmax + 1
    Kd = [[[mp.mpf(0)] * L for _ in range(L)] for _ in range(nq)]
    for b in range(L):
        for q in range(nq):
            for (a, v) in rows[b][q]:
                Kd[q][b][a] += v
    out = []
    for h in (0, 1):
        slots = []
        for p in (0, 1):
            for l in range(1, lmax + 1):
                for am in range(0, l + 1):
                    if (l + am + p) % 2 != h:
                        continue
                    if am == 0:
                        slots.append((l, 0, p, "0"))
                    else:
                        slots.append((l, am, p, "+"))
                        slots.append((l, am, p, "-"))
        n = len(slots)
        # S: new = S x' ; Sinv: x' = Sinv new
        S = [[mp.mpf(0)] * L for _ in range(n)]
        Sinv = [[mp.mpf(0)] * n for _ in range(L)]
        for k, (l, am, p, kind) in enumerate(slots):
            if kind == "0":
                S[k][idx[(l, 0, p)]] = mp.mpf(1)
                Sinv[idx[(l, 0, p)]][k] = mp.mpf(1)
            else:
                sg = 1 if kind == "+" else -1
                S[k][idx[(l, am, p)]] = mp.mpf(1)
                S[k][idx[(l, -am, p)]] = mp.mpf(sg)
                Sinv[idx[(l, am, p)]][k] = mp.mpf(1) / 2
                Sinv[idx[(l, -am, p)]][k] = mp.mpf(sg) / 2
        Knew = []
        for q in range(nq):
            per_row = []
            for r in range(n):
                terms = []
                for c in range(n):
                    v = mp.mpf(0)
                    for b in range(L):
                        if S[r][b] == 0:
                            continue
                        for a in range(L):
                            if Sinv[a][c] != 0 and Kd[q][b][a] != 0:
                                v += S[r][b] * Kd[q][b][a] * Sinv[a][c]
                    if abs(v) > mp.mpf(10) ** -30:
                        terms.append((c, v))
                per_row.append(terms)
            Knew.append(per_row)
        out.append((slots, Knew))
    return out


# ----------------------------------------------------------------------------- coplanar: rotation - axial translation - rotation
# In the pair frame F' (x' along the pair, z' the layout normal) the translation mixes all m.  In the frame F'' whose z''
# axis is the pair axis (x'' = -z', y'' = y', z'' = x': F' turned by +90 degrees about y') it is diagonal in m'' (theta = 0:
# Pbar_q^mu(1) = 0 for mu > 0 in Eq. I16).  The frame change acts on the coefficients of every (l, p) with the same real
# (2l+1) x (2l+1) matrix Dl, because Phi_{l,m,p} are built from Ybar_{l,m} = Pbar_l^{|m|}(cos theta) e^{i m phi} by
# coordinate-free operators.  Dl is obtained numerically (40 digits) from its definition
#   Ybar_{l,m'}(direction in F') = sum_{m''} Dl[m'', m'] Ybar_{l,m''}(same direction in F''),
# so no phase convention enters; coplanar_axial() asserts K_q = D^-1 Z_q D for every q against coplanar_rows().
def pbar_general(l, m, x):
    """Pbar_l^m(x), m >= 0, no Condon-Shortley phase (R2): sqrt((2l+1)/2 (l-m)!/(l+m)!) (1-x^2)^{m/2} d^m P_l/dx^m."""
    s = mp.mpf(0)
    for k in range(0, l // 2 + 1):
        e = l - 2 * k
        if e - m < 0:
            continue
        c = Fraction((-1) ** k * comb(l, k) * comb(2 * l - 2 * k, l), 2 ** l) * Fraction(factorial(e), factorial(e - m))
        s += mp.mpf(c.numerator) / mp.mpf(c.denominator) * mp.mpf(x) ** (e - m)
    n2 = Fraction((2 * l + 1) * factorial(l - m), 2 * factorial(l + m))
    return s * mp.sqrt(1 - mp.mpf(x) ** 2) ** m * mp.sqrt(mp.mpf(n2.numerator) / mp.mpf(n2.denominator))


_rot_cache = {}


def frame_rotation(l):
    """Dl (real, (2l+1) x (2l+1), rows m'' = -l..l, columns m' = -l..l) for F' -> F''."""
    if l in _rot_cache:
        return _rot_cache[l]
    N = 2 * l + 1
    pts = []
    for i in range(N + 3):          # fixed, well spread directions (golden-angle spiral)
        z = mp.mpf(2 * i + 1) / (N + 3) - 1
        ph = i * mp.pi * (3 - mp.sqrt(5))
        r = mp.sqrt(1 - z * z)
        pts.append((r * mp.cos(ph), r * mp.sin(ph), z))

    def ybar(m, v):
        return pbar_general(l, abs(m), v[2]) * mp.e ** (1j * m * mp.atan2(v[1], v[0]))
    Yp = mp.matrix(len(pts), N)
    Ypp = mp.matrix(len(pts), N)
    for i, v in enumerate(pts):
        vpp = (-v[2], v[1], v[0])
        for j, m in enumerate(range(-l, l + 1)):
            Yp[i, j] = ybar(m, v)
            Ypp[i, j] = ybar(m, vpp)
    D = mp.inverse(Ypp[:N, :]) * Yp[:N, :]
    assert mp.norm(Ypp * D - Yp) < mp.mpf(10) ** -30, "frame rotation: projection does not reproduce the extra directions"
    assert max(abs(mp.im(D[i, j])) for i in range(N) for j in range(N)) < mp.mpf(10) ** -30
    D = D.apply(mp.re)
    _rot_cache[l] = D
    return D


_axial_cache = {}


def _axial_operators(lmax):
    """(Rm, Rinv, Z, all2, S2, S2inv, pm_matrices) of one lmax: block rotation, tilde-basis axial operator per q, F'' slots."""
    if lmax in _axial_cache:
        return _axial_cache[lmax]
    md = modes(lmax)
    L = len(md)
    nq = 2 * lmax + 1
    idx = {t: i for i, t in enumerate(md)}
    eps = mp.mpf(10) ** -30
    Rm = mp.matrix(L, L)
    for p in (0, 1):
        for l in range(1, lmax + 1):
            D = frame_rotation(l)
            for i, m2 in enumerate(range(-l, l + 1)):
                for j, m1 in enumerate(range(-l, l + 1)):
                    Rm[idx[(l, m2, p)], idx[(l, m1, p)]] = D[i, j]
    Rinv = mp.inverse(Rm)
    # tilde-basis axial operator (theta = 0): only m_a = m_b, Pbar_q^0(1) = sqrt((2q+1)/2)
    Z = [mp.matrix(L, L) for _ in range(nq)]
    for b, (lp, mp_, pp) in enumerate(md):
        for a, (l, m, p) in enumerate(md):
            if m != mp_:
                continue
            for q in range(nq):
                ip, v = coupling(l, m, p, lp, mp_, pp, q)
                if v == 0:
                    continue
                tot = (ip + (pp - p)) % 4
                assert tot % 2 == 0
                v = v * mp.sqrt(mp.mpf(2 * q + 1) / 2)
                Z[q][b, a] = v if tot == 0 else -v
    rows = coplanar_rows(lmax)
    for q in range(nq):                      # the identity the whole factorisation rests on
        Kd = mp.matrix(L, L)
        for b in range(L):
            for (a, v) in rows[b][q]:
                Kd[b, a] += v
        assert mp.norm(Kd - Rinv * Z[q] * Rm) < eps, "rotation - axial translation - rotation identity violated"

    def pm_matrices(slots):
        S = mp.matrix(len(slots), L)
        Sinv = mp.matrix(L, len(slots))
        for k, (l, am, p, kind) in enumerate(slots):
            if kind == "0":
                S[k, idx[(l, 0, p)]] = 1
                Sinv[idx[(l, 0, p)], k] = 1
            else:
                sg = 1 if kind == "+" else -1
                S[k, idx[(l, am, p)]] = 1
                S[k, idx[(l, -am, p)]] = sg
                Sinv[idx[(l, am, p)], k] = mp.mpf(1) / 2
                Sinv[idx[(l, -am, p)], k] = mp.mpf(sg) / 2
        return S, Sinv
    all2 = []
    for p in (0, 1):
        for l in range(1, lmax + 1):
            for am in range(0, l + 1):
                all2 += [(l, 0, p, "0")] if am == 0 else [(l, am, p, "+"), (l, am, p, "-")]
    S2, S2inv = pm_matrices(all2)
    Zc = [S2 * Z[q] * S2inv for q in range(nq)]
    _axial_cache[lmax] = (Rm, Rinv, Zc, all2, S2, S2inv, pm_matrices)
    return _axial_cache[lmax]


def axial_factorise(lmax, slots, Kdirect):
    """Factorisation  K_q = Gout Z''_q G  of the pair-frame operator restricted to the +- slots `slots` (a subspace the
    operator does not leave).  Kdirect(q) -> {(row, col): value} is the direct operator, used only for the final check.
    Returns (slots, slots2, G, entries, Gout):
      slots2  the F'' slots (l, |m''|, p, kind) reached from this subspace (same count)
      G       rows over slots2: [(col slot, value)]        x'' = G x'
      entries {(row2, col2): [(q, value)]}                 u''_row = sum_col (sum_q value h_q) x''_col   (same |m''| only)
      Gout    rows over slots: [(col2, value)]             u' = Gout u''"""
    Rm, Rinv, Zc, all2, S2, S2inv, pm_matrices = _axial_operators(lmax)
    L = len(all2)
    nq = 2 * lmax + 1
    eps = mp.mpf(10) ** -30
    n = len(slots)
    S, Sinv = pm_matrices(slots)
    Gf = S2 * Rm * Sinv                  # L x n
    sel = [r for r in range(L) if any(abs(Gf[r, c]) > eps for c in range(n))]
    assert len(sel) == n, "the subspace must map onto as many F'' slots"
    sel.sort(key=lambda r: (all2[r][1], r))          # group by |m''|
    pos = {r: i for i, r in enumerate(sel)}
    Go_f = S * Rinv * S2inv              # n x L
    G = [[(c, Gf[r, c]) for c in range(n) if abs(Gf[r, c]) > eps] for r in sel]
    Gout = [[(j, Go_f[i, r]) for j, r in enumerate(sel) if abs(Go_f[i, r]) > eps] for i in range(n)]
    entries = {}
    for q in range(nq):
        for i, r in enumerate(sel):
            for c in range(L):
                if abs(Zc[q][r, c]) > eps:
                    assert c in pos and all2[c][1] == all2[r][1], "axial operator must stay inside the subspace and inside |m''|"
                    entries.setdefault((i, pos[c]), []).append((q, Zc[q][r, c]))
    Gm = mp.matrix(n, n)
    Gom = mp.matrix(n, n)
    for i, row in enumerate(G):
        for (c, v) in row:
            Gm[i, c] = v
    for i, row in enumerate(Gout):
        for (c, v) in row:
            Gom[i, c] = v
    for q in range(nq):                  # end-to-end check against the direct operator
        M = mp.matrix(n, n)
        for (i, j), lst in entries.items():
            for (qq, v) in lst:
                if qq == q:
                    M[i, j] = v
        Kq = mp.matrix(n, n)
        for (r, c), v in Kdirect(q).items():
            Kq[r, c] = v
        assert mp.norm(Kq - Gom * M * Gm) < eps, "factorised operator differs from the direct one"
    return slots, [all2[r] for r in sel], G, entries, Gout


def coplanar_axial(lmax):
    """Per z-mirror half of coplanar_sym(): the factorisation of axial_factorise()."""
    out = []
    for (slots, Knew) in coplanar_sym(lmax):
        out.append(axial_factorise(lmax, slots, lambda q, Knew=Knew: {(r, c): v for r in range(len(Knew[q])) for (c, v) in Knew[q][r]}))
    return out


def coplanar_sectors_axial(lmax):
    """Per sector of coplanar_sectors(): the factorisation of axial_factorise()."""
    out = {}
    for z, (slots, rows) in coplanar_sectors(lmax).items():
        out[z] = axial_factorise(lmax, slots, lambda q, rows=rows: {(r, c): v for r in range(len(rows)) for (c, v) in rows[r][q]})
    return out


COPLANAR_AXIAL = True      # False: direct pair-frame operator (sum over (row, col, q) terms), the round's first version


def emit_axial_core(f, fac, sync_tag=None, hooks=False):
    """Straight-line code  u' = Gout (sum_q h_q Z''_q) G x'  for one half; x' in xr{k}/xi{k}, result in ur{k}/ui{k}.
    hooks: emit `hk.template at<K>();` after the frame change (K = 0) and after every row of the axial translation (K = 1 ..):
    places where the calling kernel may put independent work of its own (k_allpairs_coplanar: the set-up of the NEXT pair) into
    the middle of this straight-line code; a no-op functor leaves the code as it was.
    sync_tag: emit TM_PHASE_SYNC(tag, k) after the frame change (k = 0) and after every |m''| block of the axial translation
    (k = 1, 2, ...): block-wide barriers that keep the warps of a block inside one phase of the straight-line code, so that
    the phase - not the whole loop body - has to fit the 32 KB instruction cache (lmax >= 5; a no-op elsewhere).
    Returns (FP instructions, flop)."""
    slots, slots2, G, entries, Gout = fac
    n = len(slots)
    inst = flop = 0

    # x'' = G x'
    f.write("  // frame change F' -> F'' (z'' = pair axis)\n")
    for i, row in enumerate(G):
        for part in ("r", "i"):
            expr = None
            for t, (c, v) in enumerate(row):
                if t == 0:
                    if abs(v) == 1:
                        expr = f"{'-' if v < 0 else ''}x{part}{c}"
                    else:
                        expr = f"R({lit(v)}) * x{part}{c}"
                        inst += 1
                        flop += 1
                else:
                    expr = f"fma(R({lit(v)}), x{part}{c}, {expr})"
                    inst += 1
                    flop += 2
            f.write(f"  const R w{part}{i} = {expr};\n")
    # axial translation, one |m''| block after the other; identical radial sums are formed once
    if sync_tag is not None:
        f.write(f"  TM_PHASE_SYNC({sync_tag}, 0);\n")
    if hooks:
        f.write("  hk.template at<0>();\n")
    f.write("  // axial translation along z'': diagonal in m''\n")
    known = {}
    by_row = {}
    n_sync = 1
    for (i, j), lst in sorted(entries.items()):
        by_row.setdefault(i, []).append((j, lst))
    for i in range(n):
        if sync_tag is not None and i > 0 and slots2[i][1] != slots2[i - 1][1]:
            f.write(f"  TM_PHASE_SYNC({sync_tag}, {n_sync});\n")
            n_sync += 1
        first = True
        for (j, lst) in by_row.get(i, []):
            s0 = 1 if lst[0][1] > 0 else -1
            key = tuple((q, mp.nstr(s0 * v, 30)) for (q, v) in lst)
            if key not in known:
                e = len(known)
                known[key] = e
                for part, hh in (("r", "hr"), ("i", "hi")):
                    expr = None
                    for t, (q, v) in enumerate(lst):
                        vv = s0 * v
                        if t == 0 and abs(vv) == 1:
                            expr = f"{'-' if vv < 0 else ''}{hh}[{q}]"
                        elif t == 0:
                            expr = f"R({lit(vv)}) * {hh}[{q}]"
                            inst += 1
                            flop += 1
                        else:
                            expr = f"fma(R({lit(vv)}), {hh}[{q}], {expr})"
                            inst += 1
                            flop += 2
                    f.write(f"  const R e{part}{e} = {expr};\n")
            e = known[key]
            sg = "" if s0 > 0 else "-"
            ng = "-" if s0 > 0 else ""
            if first:
                f.write(f"  R tr{i} = {sg}er{e} * wr{j}; tr{i} = fma({ng}ei{e}, wi{j}, tr{i}); "
                        f"R ti{i} = {sg}er{e} * wi{j}; ti{i} = fma({sg}ei{e}, wr{j}, ti{i});\n")
                inst += 4
                flop += 6
                first = False
            else:
                f.write(f"  tr{i} = fma({sg}er{e}, wr{j}, tr{i}); tr{i} = fma({ng}ei{e}, wi{j}, tr{i}); "
                        f"ti{i} = fma({sg}er{e}, wi{j}, ti{i}); ti{i} = fma({sg}ei{e}, wr{j}, ti{i});\n")
                inst += 4
                flop += 8
        assert not first, "every F'' slot receives something"
        if hooks:
            f.write(f"  hk.template at<{i + 1}>();\n")
    # u' = Gout u''
    if sync_tag is not None:
        f.write(f"  TM_PHASE_SYNC({sync_tag}, {n_sync});\n")
    f.write("  // frame change back F'' -> F'\n")
    for r, row in enumerate(Gout):
        for part in ("r", "i"):
            expr = None
            for t, (c, v) in enumerate(row):
                if t == 0:
                    if abs(v) == 1:
                        expr = f"{'-' if v < 0 else ''}t{part}{c}"
                    else:
                        expr = f"R({lit(v)}) * t{part}{c}"
                        inst += 1
                        flop += 1
                else:
                    expr = f"fma(R({lit(v)}), t{part}{c}, {expr})"
                    inst += 1
                    flop += 2
            f.write(f"  const R u{part}{r} = {expr};\n")
    return inst, flop, len(known), sum(len(k) for k in known)


def emit_coplanar(lmaxes, path):
    with open(path, "w") as f:
        f.write("// GENERATED by gen_tables.py - do not edit.\n")
        f.write("// Coplanar (theta = pi/2) translation apply, one z-mirror-parity half per call: phase rotation onto the pair frame,\n")
        f.write("// fixed real frame change onto the pair AXIS, m''-diagonal axial translation, and back (gen_tables.py: coplanar_axial).\n")
        f.write("// Interface and +- bases as in the direct version: pair frame, one z-mirror-parity half per call, reduced by\n")
        f.write("// the pair's y'-mirror symmetry (DESIGN.md, kernel K2c).  Basis of a half (\"slots\"): for every (l, |m|, p):\n")
        f.write("// d^0 = x~_{l,0,p};  d^+- = x~_{l,m,p} +- x~_{l,-m,p}  (x~ = i^p x), staged by the kernel with the tables below.\n")
        f.write("// xs: interleaved (re,im) d-values of this half; cm/sm: cos/sin(m phi); hr/hi: Re/Im h_q^(1)(kr);\n")
        f.write("// ar/ai: accumulators A^0, A^+- = u~_{l,m,p} +- u~_{l,-m,p} of this half (unmixed once at the end).\n")
        f.write("// tm_cop_pair_*_hk: the same code with hook points hk.at<K>() (after the frame change: K = 0; after row K - 1 of the axial\n")
        f.write("// translation: K = 1 ..) where the caller may place independent work; TmCopNoHook leaves the code as it is.\n#pragma once\n\n")
        f.write("struct TmCopNoHook { template <int K> __device__ __forceinline__ void at() const {} };\n\n")
        for lmax in lmaxes:
            md = modes(lmax)
            idx = {t: i for i, t in enumerate(md)}
            sym = coplanar_sym(lmax)
            axial = coplanar_axial(lmax) if COPLANAR_AXIAL else None
            cost = [0, 0]
            for h in (0, 1):
                slots, Knew = sym[h]
                n = len(slots)
                nq = 2 * lmax + 1
                nterm = nrowq = 0
                f.write(f"// lmax={lmax} half={h}: slots (l,|m|,p,kind) {[(l, am, p, k) for (l, am, p, k) in slots]}\n")
                f.write("template <typename R, typename HK>\n__device__ __forceinline__ void "
                        f"tm_cop_pair_L{lmax}_H{h}_hk(const R* __restrict__ xs, const R* cm, const R* sm, const R* hr, const R* hi, R* ar, R* ai, const HK& hk) {{\n")
                # input phase rotation in the +- basis
                k = 0
                n_pairs = n_zero = 0
                while k < n:
                    l, am, p, kind = slots[k]
                    if kind == "0":
                        f.write(f"  const R xr{k} = xs[{2 * k}], xi{k} = xs[{2 * k + 1}];\n")
                        n_zero += 1
                        k += 1
                    else:       # slots k (+) and k+1 (-):  x^+ = c d^+ + i s d^- ,  x^- = c d^- + i s d^+
                        kp, km = k, k + 1
                        f.write(f"  const R xr{kp} = xs[{2 * kp}] * cm[{am}] - xs[{2 * km + 1}] * sm[{am}], "
                                f"xi{kp} = xs[{2 * kp + 1}] * cm[{am}] + xs[{2 * km}] * sm[{am}];\n")
                        f.write(f"  const R xr{km} = xs[{2 * km}] * cm[{am}] - xs[{2 * kp + 1}] * sm[{am}], "
                                f"xi{km} = xs[{2 * km + 1}] * cm[{am}] + xs[{2 * kp}] * sm[{am}];\n")
                        n_pairs += 1
                        k += 2

                core = None
                if COPLANAR_AXIAL:
                    core = emit_axial_core(f, axial[h], hooks=True)

                def row_code(r):
                    nonlocal nterm, nrowq
                    if COPLANAR_AXIAL:
                        return
                    f.write(f"    R ur{r} = R(0), ui{r} = R(0);\n")
                    first_q = True
                    for q in range(nq):
                        terms = Knew[q][r]
                        if not terms:
                            continue
                        nrowq += 1
                        for t, (c, v) in enumerate(terms):
                            nterm += 1
                            if t == 0:
                                f.write(f"    yr = R({lit(v)}) * xr{c}; yi = R({lit(v)}) * xi{c};\n")
                            else:
                                f.write(f"    yr = fma(R({lit(v)}), xr{c}, yr); yi = fma(R({lit(v)}), xi{c}, yi);\n")
                        if first_q:
                            f.write(f"    ur{r} = hr[{q}] * yr; ur{r} = fma(-hi[{q}], yi, ur{r}); ui{r} = hr[{q}] * yi; ui{r} = fma(hi[{q}], yr, ui{r});\n")
                            first_q = False
                        else:
                            f.write(f"    ur{r} = fma(hr[{q}], yr, ur{r}); ur{r} = fma(-hi[{q}], yi, ur{r}); ui{r} = fma(hr[{q}], yi, ui{r}); ui{r} = fma(hi[{q}], yr, ui{r});\n")

                k = 0
                while k < n:
                    l, am, p, kind = slots[k]
                    f.write("  {\n" if COPLANAR_AXIAL else "  {\n    R yr, yi;\n")
                    if kind == "0":
                        row_code(k)
                        f.write(f"    ar[{k}] += ur{k}; ai[{k}] += ui{k};\n")
                        k += 1
                    else:       # A^+ += c u^+ - i s u^- ;  A^- += c u^- - i s u^+
                        kp, km = k, k + 1
                        row_code(kp)
                        row_code(km)
                        f.write(f"    ar[{kp}] = fma(ur{kp}, cm[{am}], ar[{kp}]); ar[{kp}] = fma(ui{km}, sm[{am}], ar[{kp}]);\n")
                        f.write(f"    ai[{kp}] = fma(ui{kp}, cm[{am}], ai[{kp}]); ai[{kp}] = fma(-ur{km}, sm[{am}], ai[{kp}]);\n")
                        f.write(f"    ar[{km}] = fma(ur{km}, cm[{am}], ar[{km}]); ar[{km}] = fma(ui{kp}, sm[{am}], ar[{km}]);\n")
                        f.write(f"    ai[{km}] = fma(ui{km}, cm[{am}], ai[{km}]); ai[{km}] = fma(-ur{kp}, sm[{am}], ai[{km}]);\n")
                        k += 2
                    f.write("  }\n")
                f.write("}\n")
                f.write("template <typename R>\n__device__ __forceinline__ void "
                        f"tm_cop_pair_L{lmax}_H{h}(const R* __restrict__ xs, const R* cm, const R* sm, const R* hr, const R* hi, R* ar, R* ai) {{\n"
                        f"  tm_cop_pair_L{lmax}_H{h}_hk<R, TmCopNoHook>(xs, cm, sm, hr, hi, ar, ai, TmCopNoHook());\n}}\n")
                # executed FP work per pair-half (generated code only; geometry/Hankel not counted):
                #   first term of a (row,q): 2 MUL, other terms 2 FMA; per (row,q): 4 FMA (first q of a row: 2 MUL + 2 FMA);
                #   input rotation per +- pair: 4 MUL + 4 FMA; output per pair: 8 FMA; m = 0 rows: 2 ADD
                inst = 2 * nterm + 4 * nrowq + 8 * n_pairs + 8 * n_pairs + 2 * n_zero
                flop = (2 * nrowq + 4 * (nterm - nrowq)) + (8 * nrowq - 2 * n) + (4 + 8) * n_pairs + 16 * n_pairs + 2 * n_zero
                if COPLANAR_AXIAL:      # frame changes + radial sums + m''-diagonal apply, plus the phase rotations in and out
                    inst = core[0] + 16 * n_pairs + 2 * n_zero
                    flop = core[1] + (4 + 8) * n_pairs + 16 * n_pairs + 2 * n_zero
                    print(f"lmax={lmax} half={h}: n={n} axial: {core[2]} distinct radial sums ({core[3]} terms) "
                          f"-> {inst} FP instructions, {flop} flop per pair-half", file=sys.stderr)
                else:
                    print(f"lmax={lmax} half={h}: n={n} sym terms={nterm} (row,q) combos={nrowq} "
                          f"-> {inst} FP instructions, {flop} flop per pair-half", file=sys.stderr)
                cost[0] += inst
                cost[1] += flop
                # staging tables: d_k = x~[sa] + ss * x~[sb]
                sa, sb, ss = [], [], []
                for (l, am, p, kind) in slots:
                    sa.append(idx[(l, am, p)])
                    sb.append(idx[(l, -am, p)])
                    ss.append({"0": 0, "+": 1, "-": -1}[kind])
                f.write(f"__device__ __constant__ int tm_cop_sa_L{lmax}_H{h}[{n}] = {{{', '.join(map(str, sa))}}};\n")
                f.write(f"__device__ __constant__ int tm_cop_sb_L{lmax}_H{h}[{n}] = {{{', '.join(map(str, sb))}}};\n")
                f.write(f"__device__ __constant__ int tm_cop_ss_L{lmax}_H{h}[{n}] = {{{', '.join(map(str, ss))}}};\n")
                # unmix: u~_{l,+-m,p} = (A^+ +- A^-)/2, then u = (-i)^p u~
                f.write("template <typename R, typename C>\n__device__ __forceinline__ void "
                        f"tm_cop_unmix_L{lmax}_H{h}(const R* ar, const R* ai, C* out) {{\n")
                half_l = len(md) // 2
                k = 0
                while k < n:
                    l, am, p, kind = slots[k]

                    def store(i_flat, re, im):
                        if i_flat >= half_l:      # p = 1: multiply by -i
                            f.write(f"  out[{i_flat}].re = {im}; out[{i_flat}].im = -({re});\n")
                        else:
                            f.write(f"  out[{i_flat}].re = {re}; out[{i_flat}].im = {im};\n")
                    if kind == "0":
                        store(idx[(l, 0, p)], f"ar[{k}]", f"ai[{k}]")
                        k += 1
                    else:
                        kp, km = k, k + 1
                        store(idx[(l, am, p)], f"R(0.5) * (ar[{kp}] + ar[{km}])", f"R(0.5) * (ai[{kp}] + ai[{km}])")
                        store(idx[(l, -am, p)], f"R(0.5) * (ar[{kp}] - ar[{km}])", f"R(0.5) * (ai[{kp}] - ai[{km}])")
                        k += 2
                f.write("}\n")
            f.write(f"#define TM_COP_NH_L{lmax} {len(md) // 2}\n")
            f.write(f"#define TM_COP_FPINST_L{lmax} {cost[0]}   // FP instructions per ordered pair (both halves)\n")
            f.write(f"#define TM_COP_FLOP_L{lmax} {cost[1]}     // flop per ordered pair (FMA = 2)\n\n")


# ----------------------------------------------------------------------------- general 3-D, symmetric-basis code
def general_sym(lmax):
    """3-D operator in the frame rotated about z so that the pair lies in the x'z plane (phi = 0):
         u'_b = sum_a sum_q c~_q(b,a) h_q(kr) Pbar_q^{|m_a-m_b|}(cos theta) x'_a      (c~ real in the tilde basis)
    The pair lies in the mirror plane y' = 0, so c~_q((l',-m',p'),(l,-m,p)) = +-c~_q((l',m',p'),(l,m,p)) and the +- basis
    of coplanar_sym splits the L modes into two uncoupled SECTORS of L/2:
         sector 0 = {p=0: '0','+'; p=1: '-'},   sector 1 = {p=0: '-'; p=1: '0','+'}.
    Returns per sector: slots [(l, am, p, kind)] and rows[r][q] = [(c, [(mu, kappa)])]:
         u^new_r = sum_q h_q sum_c ( sum_mu kappa Pbar_q^mu ) x^new_c ."""
    md = modes(lmax)
    idx = {t: i for i, t in enumerate(md)}
    nq = 2 * lmax + 1
    C = {}
    for (b, a, q, ip, v) in general_terms(lmax):
        (lp, mp_, pp), (l, m, p) = md[b], md[a]
        tot = (ip + (pp - p)) % 4
        assert tot % 2 == 0
        C[(b, a, q)] = v if tot == 0 else -v
    sectors = [[], []]
    for p in (0, 1):
        for l in range(1, lmax + 1):
            for am in range(0, l + 1):
                for kind in (["0"] if am == 0 else ["+", "-"]):
                    in0 = (p == 0 and kind in "0+") or (p == 1 and kind == "-")
                    sectors[0 if in0 else 1].append((l, am, p, kind))
    out = []
    for sec in sectors:
        n = len(sec)
        rows = [[[] for _ in range(nq)] for _ in range(n)]
        for r, (lr, mr, pr, kr) in enumerate(sec):
            rws = [(idx[(lr, mr, pr)], 1)] if kr == "0" else [(idx[(lr, mr, pr)], 1), (idx[(lr, -mr, pr)], 1 if kr == "+" else -1)]
            for c, (lc, mc, pc, kc) in enumerate(sec):
                cls = ([(idx[(lc, mc, pc)], mp.mpf(1))] if kc == "0" else
                       [(idx[(lc, mc, pc)], mp.mpf(1) / 2), (idx[(lc, -mc, pc)], (mp.mpf(1) if kc == "+" else -mp.mpf(1)) / 2)])
                acc = {}
                for (b, sb) in rws:
                    for (a, sa) in cls:
                        mu = abs(md[a][1] - md[b][1])
                        for q in range(nq):
                            if (b, a, q) in C:
                                acc[(q, mu)] = acc.get((q, mu), mp.mpf(0)) + sb * sa * C[(b, a, q)]
                for q in range(nq):
                    lst = [(mu, v) for (qq, mu), v in sorted(acc.items()) if qq == q and abs(v) > mp.mpf(10) ** -30]
                    if lst:
                        rows[r][q].append((c, lst))
        # the other sector must not couple (checked through the full matrix): every (b,a,q) term is consumed above
        out.append((sec, rows))
    return out


def emit_general_sym(lmaxes, path):
    with open(path, "w") as f:
        f.write("// GENERATED by gen_tables.py - do not edit.\n")
        f.write("// General 3-D translation apply in the frame rotated about z onto the pair's azimuth, one y'-mirror SECTOR per call\n")
        f.write("// (DESIGN.md, kernel K2s).  Slots as in tm_coplanar_gen.cuh; Pq_mu = Pbar_q^mu(cos theta), normalised, no Condon-Shortley phase.\n#pragma once\n\n")
        for lmax in lmaxes:
            md = modes(lmax)
            idx = {t: i for i, t in enumerate(md)}
            nq = 2 * lmax + 1
            cost = [0, 0]
            for sct, (slots, rows) in enumerate(general_sym(lmax)):
                n = len(slots)
                f.write(f"// lmax={lmax} sector={sct}: slots (l,|m|,p,kind) {slots}\n")
                f.write("// q-outer order: Pbar_q^mu is produced level by level (recurrence in q) and dies after its level, so the\n")
                f.write("// live state is x^new, the row sums u and two Legendre levels (no spills at 255 registers).\n")
                f.write("template <typename R, int AS>\n__device__ __forceinline__ void "
                        f"tm_g3d_pair_L{lmax}_S{sct}(const R* __restrict__ xs, const R* cm, const R* sm, const R* hr, const R* hi, R ct, R st, R* ar, R* ai) {{\n")
                k = 0
                n_pairs = n_zero = 0
                while k < n:
                    l, am, p, kind = slots[k]
                    if kind == "0":
                        f.write(f"  const R xr{k} = xs[{2 * k}], xi{k} = xs[{2 * k + 1}];\n")
                        n_zero += 1
                    else:
                        f.write(f"  const R xr{k} = xs[{2 * k}] * cm[{am}] - xs[{2 * (n + k) + 1}] * sm[{am}], "
                                f"xi{k} = xs[{2 * k + 1}] * cm[{am}] + xs[{2 * (n + k)}] * sm[{am}];\n")
                        n_pairs += 1
                    k += 1
                for r in range(n):
                    f.write(f"  R ur{r} = R(0), ui{r} = R(0);\n")
                nterm = nrc = nrowq = 0
                for q in range(nq):
                    f.write("  {\n")
                    # Legendre level q: P{q}_{mu}, mu = 0..q
                    for mu in range(0, q + 1):
                        if q == 0:
                            f.write(f"    const R P0_0 = R({lit(mp.sqrt(mp.mpf(1) / 2))});\n")
                        elif mu == q:
                            f.write(f"    const R P{q}_{mu} = R({lit(mp.sqrt(mp.mpf(2 * mu + 1) / (2 * mu)))}) * st * P{q - 1}_{mu - 1};\n")
                        elif mu == q - 1:
                            f.write(f"    const R P{q}_{mu} = R({lit(mp.sqrt(mp.mpf(2 * mu + 3)))}) * ct * P{q - 1}_{mu};\n")
                        else:
                            a_ = mp.sqrt(mp.mpf(4 * q * q - 1) / (q * q - mu * mu))
                            b_ = mp.sqrt(mp.mpf((q - 1) ** 2 - mu * mu) / (4 * (q - 1) ** 2 - 1))
                            f.write(f"    const R P{q}_{mu} = R({lit(a_)}) * (ct * P{q - 1}_{mu} - R({lit(b_)}) * P{q - 2}_{mu});\n")
                    f.write("    R zr, zi, rho;\n")
                    for r in range(n):
                        ent = rows[r][q]
                        if not ent:
                            continue
                        nrowq += 1
                        for t, (c, lst) in enumerate(ent):
                            nrc += 1
                            expr = None
                            for (mu, v) in lst:
                                nterm += 1
                                expr = f"R({lit(v)}) * P{q}_{mu}" if expr is None else f"fma(R({lit(v)}), P{q}_{mu}, {expr})"
                            f.write(f"    rho = {expr};\n")
                            if t == 0:
                                f.write(f"    zr = rho * xr{c}; zi = rho * xi{c};\n")
                            else:
                                f.write(f"    zr = fma(rho, xr{c}, zr); zi = fma(rho, xi{c}, zi);\n")
                        f.write(f"    ur{r} = fma(hr[{q}], zr, ur{r}); ur{r} = fma(-hi[{q}], zi, ur{r}); ui{r} = fma(hr[{q}], zi, ui{r}); ui{r} = fma(hi[{q}], zr, ui{r});\n")
                    # nested scopes keep level q-1 and q-2 visible: close nothing here (levels are declared in nested blocks)
                # output rotation: this sector's u^new_r feeds A^own (cos) and the PARTNER sector's accumulator (sin):
                #   A^+ += c u^+ - i s u^- ;  A^- += c u^- - i s u^+   -> ar/ai hold [own n slots | partner n slots]
                for r in range(n):
                    l, am, p, kind = slots[r]
                    if kind == "0":
                        f.write(f"    ar[{r} * AS] += ur{r}; ai[{r} * AS] += ui{r};\n")
                    else:
                        f.write(f"    ar[{r} * AS] = fma(ur{r}, cm[{am}], ar[{r} * AS]); ai[{r} * AS] = fma(ui{r}, cm[{am}], ai[{r} * AS]);\n")
                        f.write(f"    ar[{n + r} * AS] = fma(ui{r}, sm[{am}], ar[{n + r} * AS]); ai[{n + r} * AS] = fma(-ur{r}, sm[{am}], ai[{n + r} * AS]);\n")
                f.write("  " + "}" * nq + "\n}\n")
                inst = nterm + 2 * nrc + 4 * nrowq + 4 * n_pairs + 4 * n_pairs + 2 * n_zero
                flop = (2 * nterm - nrc) + (4 * nrc - 2 * nrowq) + 8 * nrowq + 6 * n_pairs + 8 * n_pairs + 2 * n_zero
                cost[0] += inst
                cost[1] += flop
                print(f"lmax={lmax} sector={sct}: n={n} terms={nterm} (row,col,q)={nrc} (row,q)={nrowq} -> {inst} FP instructions, {flop} flop",
                      file=sys.stderr)
                # staging tables for this sector: own slots then partner slots (kind flipped; '0' has no partner -> itself, unused)
                sa, sb, ss = [], [], []
                for (l, am, p, kind) in slots:
                    sa.append(idx[(l, am, p)]); sb.append(idx[(l, -am, p)]); ss.append({"0": 0, "+": 1, "-": -1}[kind])
                for (l, am, p, kind) in slots:
                    sa.append(idx[(l, am, p)]); sb.append(idx[(l, -am, p)]); ss.append({"0": 0, "+": -1, "-": 1}[kind])
                f.write(f"__device__ __constant__ int tm_g3d_sa_L{lmax}_S{sct}[{2 * n}] = {{{', '.join(map(str, sa))}}};\n")
                f.write(f"__device__ __constant__ int tm_g3d_sb_L{lmax}_S{sct}[{2 * n}] = {{{', '.join(map(str, sb))}}};\n")
                f.write(f"__device__ __constant__ int tm_g3d_ss_L{lmax}_S{sct}[{2 * n}] = {{{', '.join(map(str, ss))}}};\n")
                # Each block (one sector) produces, for every (l,am,p) of its slots, a contribution to A^own (slot r) and to
                # A^partner (slot n + r).  u~_{l,+-m,p} = (A^+ +- A^-)/2 needs both sectors' contributions, so each sector
                # writes its share of u~ into its own partial buffer (the finishing kernel adds the two):
                #   own kind '+': A^+ part = ar[r], A^- part = ar[n+r]  ->  u~_{+m} += (ar[r] + ar[n+r])/2, u~_{-m} += (ar[r] - ar[n+r])/2
                #   own kind '-': A^- part = ar[r], A^+ part = ar[n+r]  ->  u~_{+m} += (ar[n+r] + ar[r])/2, u~_{-m} += (ar[n+r] - ar[r])/2
                f.write("template <typename R, typename C, int AS>\n__device__ __forceinline__ void "
                        f"tm_g3d_unmix_L{lmax}_S{sct}(const R* ar, const R* ai, C* out) {{\n")
                half_l = len(md) // 2
                for r, (l, am, p, kind) in enumerate(slots):
                    def store(i_flat, re, im):
                        if i_flat >= half_l:
                            f.write(f"  out[{i_flat}].re = {im}; out[{i_flat}].im = -({re});\n")
                        else:
                            f.write(f"  out[{i_flat}].re = {re}; out[{i_flat}].im = {im};\n")
                    if kind == "0":
                        store(idx[(l, 0, p)], f"ar[{r} * AS]", f"ai[{r} * AS]")
                    else:
                        plus_r, plus_i = (f"ar[{r} * AS]", f"ai[{r} * AS]") if kind == "+" else (f"ar[{n + r} * AS]", f"ai[{n + r} * AS]")
                        minus_r, minus_i = (f"ar[{n + r} * AS]", f"ai[{n + r} * AS]") if kind == "+" else (f"ar[{r} * AS]", f"ai[{r} * AS]")
                        store(idx[(l, am, p)], f"R(0.5) * ({plus_r} + {minus_r})", f"R(0.5) * ({plus_i} + {minus_i})")
                        store(idx[(l, -am, p)], f"R(0.5) * ({plus_r} - {minus_r})", f"R(0.5) * ({plus_i} - {minus_i})")
                covered = set()
                for (l, am, p, kind) in slots:
                    covered.add(idx[(l, am, p)]); covered.add(idx[(l, -am, p)])
                for i_flat in range(len(md)):
                    if i_flat not in covered:      # m = 0 modes owned by the other sector: this sector contributes nothing
                        f.write(f"  out[{i_flat}].re = R(0); out[{i_flat}].im = R(0);\n")
                f.write("}\n")
            f.write(f"#define TM_G3D_FPINST_L{lmax} {cost[0]}   // FP instructions per ordered pair (both sectors, generated apply code only)\n")
            f.write(f"#define TM_G3D_FLOP_L{lmax} {cost[1]}     // flop per ordered pair (FMA = 2)\n\n")


# ----------------------------------------------------------------------------- coplanar, four sectors (lmax 4..6)
def coplanar_sectors(lmax):
    """Coplanar operator split by BOTH mirrors into four uncoupled sectors z = 2 h + t:
    h = z-mirror parity (l+m+p) mod 2, t = y'-mirror sector (t = 0: {p=0: '0','+'; p=1: '-'}, t = 1: the rest).
    Returns {z: (slots, rows)} with rows[r][q] = [(c, value)]:  u^new_r = sum_q h_q sum_c value x^new_c."""
    md = modes(lmax)
    idx = {t_: i for i, t_ in enumerate(md)}
    nq = 2 * lmax + 1
    rows0 = coplanar_rows(lmax)
    Kd = {}
    for b in range(len(md)):
        for q in range(nq):
            for (a, v) in rows0[b][q]:
                Kd[(q, b, a)] = Kd.get((q, b, a), mp.mpf(0)) + v
    out = {}
    for h in (0, 1):
        for t in (0, 1):
            slots = []
            for p in (0, 1):
                for l in range(1, lmax + 1):
                    for am in range(0, l + 1):
                        if (l + am + p) % 2 != h:
                            continue
                        for kind in (["0"] if am == 0 else ["+", "-"]):
                            in0 = (p == 0 and kind in "0+") or (p == 1 and kind == "-")
                            if in0 == (t == 0):
                                slots.append((l, am, p, kind))
            rows = [[[] for _ in range(nq)] for _ in slots]
            for r, (lr, mr, pr, kr) in enumerate(slots):
                rws = [(idx[(lr, mr, pr)], 1)] if kr == "0" else [(idx[(lr, mr, pr)], 1), (idx[(lr, -mr, pr)], 1 if kr == "+" else -1)]
                for c, (lc, mc, pc, kc) in enumerate(slots):
                    cls = ([(idx[(lc, mc, pc)], mp.mpf(1))] if kc == "0" else
                           [(idx[(lc, mc, pc)], mp.mpf(1) / 2), (idx[(lc, -mc, pc)], (mp.mpf(1) if kc == "+" else -mp.mpf(1)) / 2)])
                    for q in range(nq):
                        v = mp.mpf(0)
                        for (b, sb) in rws:
                            for (a_, sa) in cls:
                                if (q, b, a_) in Kd:
                                    v += sb * sa * Kd[(q, b, a_)]
                        if abs(v) > mp.mpf(10) ** -30:
                            rows[r][q].append((c, v))
            out[2 * h + t] = (slots, rows)
    return out


COP4_GROUPS = {4: 1, 5: 4, 6: 4, 7: 4}     # row groups per sector: keeps one block's straight-line code near the 32 KB L1.5 I-cache


COP4_AXIAL = True        # False: direct pair-frame operator cut into row groups


def emit_coplanar4(lmaxes, path):
    costs = {}
    with open(path, "w") as f:
        f.write("// GENERATED by gen_tables.py - do not edit.\n")
        f.write("// Coplanar translation apply for lmax 4..6: FOUR uncoupled sectors (z-mirror parity x y'-mirror sector), each split into\n")
        f.write("// G row groups so that one block's straight-line code stays near the instruction-cache size (DESIGN.md, kernel K2c4).\n")
        f.write("// xs: [own slots | partner slots] d-values of the sector; ar/ai: [own rows of the group | their partner share], stride AS.\n#pragma once\n\n")
        f.write("#ifndef TM_PHASE_SYNC\n#define TM_PHASE_SYNC(lmax, k)      // device build: block-wide barrier between code phases (tm_allpairs.cuh)\n#endif\n\n")
        for lmax in lmaxes:
            md = modes(lmax)
            idx = {t_: i for i, t_ in enumerate(md)}
            nq = 2 * lmax + 1
            half_l = len(md) // 2
            G = 1 if COP4_AXIAL else COP4_GROUPS[lmax]
            cost = [0, 0]
            nmax = 0
            rmax = 0
            secs = coplanar_sectors(lmax)
            secs_axial = coplanar_sectors_axial(lmax) if COP4_AXIAL else None
            for z in range(4):
                slots, rows = secs[z]
                n = len(slots)
                nmax = max(nmax, n)
                # staging tables of the sector: own slots then partner slots
                sa, sb, ss = [], [], []
                for (l, am, p, kind) in slots:
                    sa.append(idx[(l, am, p)]); sb.append(idx[(l, -am, p)]); ss.append({"0": 0, "+": 1, "-": -1}[kind])
                for (l, am, p, kind) in slots:
                    sa.append(idx[(l, am, p)]); sb.append(idx[(l, -am, p)]); ss.append({"0": 0, "+": -1, "-": 1}[kind])
                f.write(f"// lmax={lmax} sector z={z}: slots (l,|m|,p,kind) {slots}\n")
                f.write(f"__device__ __constant__ int tm_cop4_sa_L{lmax}_Z{z}[{2 * n}] = {{{', '.join(map(str, sa))}}};\n")
                f.write(f"__device__ __constant__ int tm_cop4_sb_L{lmax}_Z{z}[{2 * n}] = {{{', '.join(map(str, sb))}}};\n")
                f.write(f"__device__ __constant__ int tm_cop4_ss_L{lmax}_Z{z}[{2 * n}] = {{{', '.join(map(str, ss))}}};\n")
                f.write(f"#define TM_COP4_N_L{lmax}_Z{z} {n}\n")
                # row groups: contiguous, balanced by term count
                work = [sum(len(rows[r][q]) for q in range(nq)) + 4 for r in range(n)]
                bounds = [0]
                acc_w, target = 0, sum(work) / G
                for r in range(n):
                    acc_w += work[r]
                    if len(bounds) < G and acc_w >= target * len(bounds) and r + 1 < n:
                        bounds.append(r + 1)
                while len(bounds) < G:
                    bounds.append(n)
                bounds.append(n)
                hpar = z // 2
                covered_sector = set()
                for (l, am, p, kind) in slots:
                    covered_sector.add(idx[(l, am, p)]); covered_sector.add(idx[(l, -am, p)])
                for g in range(G):
                    r0, r1 = bounds[g], bounds[g + 1]
                    nr = r1 - r0
                    rmax = max(rmax, nr)
                    used_cols = list(range(n)) if COP4_AXIAL else sorted({c for r in range(r0, r1) for q in range(nq) for (c, _) in rows[r][q]})
                    f.write(f"// lmax={lmax} z={z} group={g}: rows {r0}..{r1 - 1}\n")
                    f.write(f"#define TM_COP4_NR_L{lmax}_Z{z}_G{g} {nr}\n")
                    f.write("template <typename R, int AS>\n__device__ __forceinline__ void "
                            f"tm_cop4_pair_L{lmax}_Z{z}_G{g}(const R* __restrict__ xs, const R* cm, const R* sm, const R* hr, const R* hi, R* ar, R* ai) {{\n")
                    n_pairs = n_zero = 0
                    for k in used_cols:
                        l, am, p, kind = slots[k]
                        if kind == "0":
                            f.write(f"  const R xr{k} = xs[{2 * k}], xi{k} = xs[{2 * k + 1}];\n")
                            n_zero += 1
                        else:      # x^own = c d^own + i s d^partner
                            f.write(f"  const R xr{k} = xs[{2 * k}] * cm[{am}] - xs[{2 * (n + k) + 1}] * sm[{am}], "
                                    f"xi{k} = xs[{2 * k + 1}] * cm[{am}] + xs[{2 * (n + k)}] * sm[{am}];\n")
                            n_pairs += 1
                    nterm = nrowq = 0
                    core = emit_axial_core(f, secs_axial[z], sync_tag=lmax) if COP4_AXIAL else None
                    for r in range(r0, r1):
                        l, am, p, kind = slots[r]
                        lr = r - r0
                        if COP4_AXIAL:
                            f.write(f"  {{\n    const R ur = ur{r}, ui = ui{r};\n")
                        else:
                            f.write("  {\n    R ur = R(0), ui = R(0), yr, yi;\n")
                        for q in range(nq):
                            terms = rows[r][q]
                            if not terms or COP4_AXIAL:
                                continue
                            nrowq += 1
                            for t_, (c, v) in enumerate(terms):
                                nterm += 1
                                if t_ == 0:
                                    f.write(f"    yr = R({lit(v)}) * xr{c}; yi = R({lit(v)}) * xi{c};\n")
                                else:
                                    f.write(f"    yr = fma(R({lit(v)}), xr{c}, yr); yi = fma(R({lit(v)}), xi{c}, yi);\n")
                            f.write(f"    ur = fma(hr[{q}], yr, ur); ur = fma(-hi[{q}], yi, ur); ui = fma(hr[{q}], yi, ui); ui = fma(hi[{q}], yr, ui);\n")
                        if kind == "0":
                            f.write(f"    ar[{lr} * AS] += ur; ai[{lr} * AS] += ui;\n")
                        else:      # A^own += c u ;  A^partner += -i s u
                            f.write(f"    ar[{lr} * AS] = fma(ur, cm[{am}], ar[{lr} * AS]); ai[{lr} * AS] = fma(ui, cm[{am}], ai[{lr} * AS]);\n")
                            f.write(f"    ar[({nr + lr}) * AS] = fma(ui, sm[{am}], ar[({nr + lr}) * AS]); ai[({nr + lr}) * AS] = fma(-ur, sm[{am}], ai[({nr + lr}) * AS]);\n")
                        f.write("  }\n")
                    f.write("}\n")
                    nrp = sum(1 for r in range(r0, r1) if slots[r][3] != "0")
                    inst = 2 * nterm + 4 * nrowq + 4 * n_pairs + 4 * nrp + 2 * (nr - nrp)
                    flop = (2 * nrowq + 4 * (nterm - nrowq)) + 8 * nrowq + 6 * n_pairs + 8 * nrp + 2 * (nr - nrp)
                    if COP4_AXIAL:
                        inst = core[0] + 4 * n_pairs + 4 * nrp + 2 * (nr - nrp)
                        flop = core[1] + 6 * n_pairs + 8 * nrp + 2 * (nr - nrp)
                        print(f"lmax={lmax} z={z}: n={n} axial: {core[2]} distinct radial sums ({core[3]} terms) -> {inst} FP instructions, {flop} flop", file=sys.stderr)
                    else:
                        print(f"lmax={lmax} z={z} g={g}: rows={nr} cols={len(used_cols)} terms={nterm} (row,q)={nrowq} -> {inst} FP instructions", file=sys.stderr)
                    cost[0] += inst
                    cost[1] += flop
                    # unmix of the group's rows (+ the zero fill of the partner-owned m = 0 modes, done by group 0)
                    f.write("template <typename R, typename C, int AS>\n__device__ __forceinline__ void "
                            f"tm_cop4_unmix_L{lmax}_Z{z}_G{g}(const R* ar, const R* ai, C* out) {{\n")

                    def store(i_flat, re, im):
                        if i_flat >= half_l:
                            f.write(f"  out[{i_flat}].re = {im}; out[{i_flat}].im = -({re});\n")
                        else:
                            f.write(f"  out[{i_flat}].re = {re}; out[{i_flat}].im = {im};\n")
                    for r in range(r0, r1):
                        l, am, p, kind = slots[r]
                        lr = r - r0
                        own_r, own_i = f"ar[{lr} * AS]", f"ai[{lr} * AS]"
                        par_r, par_i = f"ar[({nr + lr}) * AS]", f"ai[({nr + lr}) * AS]"
                        if kind == "0":
                            store(idx[(l, 0, p)], own_r, own_i)
                        else:
                            pr_, pi_ = (own_r, own_i) if kind == "+" else (par_r, par_i)
                            mr_, mi_ = (par_r, par_i) if kind == "+" else (own_r, own_i)
                            store(idx[(l, am, p)], f"R(0.5) * ({pr_} + {mr_})", f"R(0.5) * ({pi_} + {mi_})")
                            store(idx[(l, -am, p)], f"R(0.5) * ({pr_} - {mr_})", f"R(0.5) * ({pi_} - {mi_})")
                    if g == 0:
                        for i_flat, (l, m, p) in enumerate(md):
                            if (l + m + p) % 2 == hpar and i_flat not in covered_sector:
                                f.write(f"  out[{i_flat}].re = R(0); out[{i_flat}].im = R(0);\n")
                    f.write("}\n")
            f.write(f"#define TM_COP4_NMAX_L{lmax} {nmax}\n")
            f.write(f"#define TM_COP4_G_L{lmax} {G}\n")
            for gg in (2, 4, 8):       # TM_COP4_IFn_Lx(code): code if the sector has at least n row groups
                f.write(f"#define TM_COP4_IF{gg}_L{lmax}(...) {'__VA_ARGS__' if G >= gg else ''}\n")
            f.write(f"#define TM_COP4_NRMAX_L{lmax} {rmax}\n")
            f.write(f"#define TM_COP4_FPINST_L{lmax} {cost[0]}   // FP instructions per ordered pair (all sectors and row groups)\n")
            f.write(f"#define TM_COP4_FLOP_L{lmax} {cost[1]}     // flop per ordered pair (FMA = 2)\n\n")
            costs[lmax] = tuple(cost)
    # the cost figures alone (for translation units that do not compile the four-sector code)
    with open(os.path.join(os.path.dirname(path), "tm_coplanar4_cost.h"), "w") as f:
        f.write("// GENERATED by gen_tables.py - do not edit.  Cost figures of tm_coplanar4_gen.cuh.\n#pragma once\n")
        for lmax in lmaxes:
            f.write(f"#ifndef TM_COP4_FPINST_L{lmax}\n#define TM_COP4_FPINST_L{lmax} {costs[lmax][0]}\n#define TM_COP4_FLOP_L{lmax} {costs[lmax][1]}\n#endif\n")


# ----------------------------------------------------------------------------- coplanar, fp32 packed (FFMA2)
def emit_axial_core_f2(f, fac):
    """Packed-fp32 version of emit_axial_core: x' in float2 x{k}, result in float2 u{k}; real x complex = 1 FFMA2,
    complex x complex = 2 FFMA2; h{q} = (Re, Im) h_q must be in scope."""
    slots, slots2, G, entries, Gout = fac
    n = len(slots)
    f2 = lambda a, b: f"make_float2({a}, {b})"

    def lincomb(dst, src, rows):
        for i, row in enumerate(rows):
            expr = None
            for t, (c, v) in enumerate(row):
                kk = lit(v) + "f"
                if t == 0 and v == 1:
                    expr = f"{src}{c}"
                else:
                    expr = f"__fmul2_rn({f2(kk, kk)}, {src}{c})" if t == 0 else f"__ffma2_rn({f2(kk, kk)}, {src}{c}, {expr})"
            f.write(f"  const float2 {dst}{i} = {expr};\n")
    lincomb("w", "x", G)
    known = {}
    by_row = {}
    for (i, j), lst in sorted(entries.items()):
        by_row.setdefault(i, []).append((j, lst))
    for i in range(n):
        first = True
        for (j, lst) in by_row.get(i, []):
            s0 = 1 if lst[0][1] > 0 else -1
            key = tuple((q, mp.nstr(s0 * v, 30)) for (q, v) in lst)
            if key not in known:
                e = len(known)
                known[key] = e
                expr = None
                for t, (q, v) in enumerate(lst):
                    kk = lit(s0 * v) + "f"
                    expr = f"__fmul2_rn({f2(kk, kk)}, h{q})" if t == 0 else f"__ffma2_rn({f2(kk, kk)}, h{q}, {expr})"
                f.write(f"  const float2 e{e} = {expr};\n")
            e = known[key]
            a_re = f2(f"e{e}.x", f"e{e}.x") if s0 > 0 else f2(f"-e{e}.x", f"-e{e}.x")
            a_im = f2(f"-e{e}.y", f"e{e}.y") if s0 > 0 else f2(f"e{e}.y", f"-e{e}.y")
            if first:
                f.write(f"  float2 t{i} = __fmul2_rn({a_re}, w{j}); t{i} = __ffma2_rn({a_im}, tm_swap2(w{j}), t{i});\n")
                first = False
            else:
                f.write(f"  t{i} = __ffma2_rn({a_re}, w{j}, t{i}); t{i} = __ffma2_rn({a_im}, tm_swap2(w{j}), t{i});\n")
    lincomb("u", "t", Gout)


def emit_coplanar_f2(lmaxes, path):
    """fp32 build of the coplanar pair code on Blackwell's packed FP32 instructions (FFMA2 / FMUL2: two FMAs per issue
    slot, immediate and register operands broadcast, LO_HI swap and per-half negation are operand modifiers).  A complex
    number is one float2; real x complex = 1 FFMA2, complex x complex = 2 FFMA2.  Same mathematics as emit_coplanar."""
    f2 = lambda a, b: f"make_float2({a}, {b})"
    with open(path, "w") as f:
        f.write("// GENERATED by gen_tables.py - do not edit.\n")
        f.write("// fp32 coplanar pair code with packed FFMA2 arithmetic (one float2 per complex number); see tm_coplanar_gen.cuh.\n")
        f.write("// xs: d-values of this half; a: accumulators A^0 / A^+- of this half.\n#pragma once\n\n")
        f.write("__device__ __forceinline__ float2 tm_swap2(float2 v) { return make_float2(v.y, v.x); }\n\n")
        for lmax in lmaxes:
            md = modes(lmax)
            idx = {t: i for i, t in enumerate(md)}
            sym = coplanar_sym(lmax)
            axial = coplanar_axial(lmax) if COPLANAR_AXIAL else None
            half_l = len(md) // 2
            for h in (0, 1):
                slots, Knew = sym[h]
                n = len(slots)
                nq = 2 * lmax + 1
                f.write("__device__ __forceinline__ void "
                        f"tm_cop_pair_f2_L{lmax}_H{h}(const float2* __restrict__ xs, const float* cm, const float* sm, const float* hr, const float* hi, float2* a) {{\n")
                k = 0
                while k < n:
                    l, am, p, kind = slots[k]
                    if kind == "0":
                        f.write(f"  const float2 x{k} = xs[{k}];\n")
                        k += 1
                    else:      # x^+ = c d^+ + i s d^- ,  x^- = c d^- + i s d^+   (i s d = s (-d.y, d.x))
                        kp, km = k, k + 1
                        f.write(f"  const float2 x{kp} = __ffma2_rn({f2(f'-sm[{am}]', f'sm[{am}]')}, tm_swap2(xs[{km}]), __fmul2_rn({f2(f'cm[{am}]', f'cm[{am}]')}, xs[{kp}]));\n")
                        f.write(f"  const float2 x{km} = __ffma2_rn({f2(f'-sm[{am}]', f'sm[{am}]')}, tm_swap2(xs[{kp}]), __fmul2_rn({f2(f'cm[{am}]', f'cm[{am}]')}, xs[{km}]));\n")
                        k += 2

                if COPLANAR_AXIAL:
                    for q in range(nq):
                        f.write(f"  const float2 h{q} = make_float2(hr[{q}], hi[{q}]);\n")
                    emit_axial_core_f2(f, axial[h])

                def row_code(r):
                    if COPLANAR_AXIAL:
                        return
                    f.write(f"    float2 u{r} = make_float2(0.f, 0.f);\n")
                    for q in range(nq):
                        terms = Knew[q][r]
                        if not terms:
                            continue
                        for t, (c, v) in enumerate(terms):
                            kk = lit(v) + "f"
                            if t == 0:
                                f.write(f"    y = __fmul2_rn({f2(kk, kk)}, x{c});\n")
                            else:
                                f.write(f"    y = __ffma2_rn({f2(kk, kk)}, x{c}, y);\n")
                        # u += h_q y :  (hr yr - hi yi, hr yi + hi yr)
                        f.write(f"    u{r} = __ffma2_rn({f2(f'hr[{q}]', f'hr[{q}]')}, y, u{r}); u{r} = __ffma2_rn({f2(f'-hi[{q}]', f'hi[{q}]')}, tm_swap2(y), u{r});\n")

                k = 0
                while k < n:
                    l, am, p, kind = slots[k]
                    f.write("  {\n" if COPLANAR_AXIAL else "  {\n    float2 y;\n")
                    if kind == "0":
                        row_code(k)
                        f.write(f"    a[{k}] = __fadd2_rn(a[{k}], u{k});\n")
                        k += 1
                    else:      # A^+ += c u^+ - i s u^- ;  A^- += c u^- - i s u^+    (-i s u = s (u.y, -u.x))
                        kp, km = k, k + 1
                        row_code(kp)
                        row_code(km)
                        f.write(f"    a[{kp}] = __ffma2_rn({f2(f'cm[{am}]', f'cm[{am}]')}, u{kp}, a[{kp}]); a[{kp}] = __ffma2_rn({f2(f'sm[{am}]', f'-sm[{am}]')}, tm_swap2(u{km}), a[{kp}]);\n")
                        f.write(f"    a[{km}] = __ffma2_rn({f2(f'cm[{am}]', f'cm[{am}]')}, u{km}, a[{km}]); a[{km}] = __ffma2_rn({f2(f'sm[{am}]', f'-sm[{am}]')}, tm_swap2(u{kp}), a[{km}]);\n")
                        k += 2
                    f.write("  }\n")
                f.write("}\n")
                f.write("template <typename C>\n__device__ __forceinline__ void "
                        f"tm_cop_unmix_f2_L{lmax}_H{h}(const float2* a, C* out) {{\n")
                k = 0
                while k < n:
                    l, am, p, kind = slots[k]

                    def store(i_flat, re, im):
                        if i_flat >= half_l:      # p = 1: multiply by -i
                            f.write(f"  out[{i_flat}].re = {im}; out[{i_flat}].im = -({re});\n")
                        else:
                            f.write(f"  out[{i_flat}].re = {re}; out[{i_flat}].im = {im};\n")
                    if kind == "0":
                        store(idx[(l, 0, p)], f"a[{k}].x", f"a[{k}].y")
                        k += 1
                    else:
                        kp, km = k, k + 1
                        store(idx[(l, am, p)], f"0.5f * (a[{kp}].x + a[{km}].x)", f"0.5f * (a[{kp}].y + a[{km}].y)")
                        store(idx[(l, -am, p)], f"0.5f * (a[{kp}].x - a[{km}].x)", f"0.5f * (a[{kp}].y - a[{km}].y)")
                        k += 2
                f.write("}\n\n")




# ----------------------------------------------------------------------------- general 3-D, rotation - axial translation - rotation
# Arbitrary pair direction (theta, phi), any lmax: rotate about z by phi (phases), then about y' by theta so that z'' is the
# pair axis, translate along z'' (diagonal in m''), rotate back.  The theta rotation is NOT evaluated through Wigner-d
# recurrences: with A = the fixed frame change F' -> F_y whose z axis is y' (x_y = x', y_y = -z', z_y = y'),
#       D_l(theta) = A_l^-1 diag(e^{i m theta}) A_l ,
# so a rotation by any theta is two applications of a CONSTANT matrix around a phase rotation - the same primitive as the
# phi rotation.  All matrices are obtained numerically (40 digits) from the definition of the frame change (projection
# of Ybar_lm, as frame_rotation), in +- bases in which they come out real and sparse (about 1.3 non-zeros per row), and
# the assembled operator is asserted against the direct one (general_sym) at random angles before any code is emitted.
def frame_rotation_axes(l, ax, _cache={}):
    """D (rows m'' = -l..l, columns m' = -l..l): Ybar_{l,m'}(v) = sum_{m''} D[m'', m'] Ybar_{l,m''}(ax v); ax = rows of the new axes."""
    key = (l, tuple(tuple(mp.nstr(mp.mpf(x), 30) for x in row) for row in ax))
    if key in _cache:
        return _cache[key]
    N = 2 * l + 1
    pts = []
    for i in range(N + 3):
        z = mp.mpf(2 * i + 1) / (N + 3) - 1
        ph = i * mp.pi * (3 - mp.sqrt(5))
        r = mp.sqrt(1 - z * z)
        pts.append((r * mp.cos(ph), r * mp.sin(ph), z))

    def ybar(m, v):
        return pbar_general(l, abs(m), v[2]) * mp.e ** (1j * m * mp.atan2(v[1], v[0]))
    Yp = mp.matrix(len(pts), N)
    Ypp = mp.matrix(len(pts), N)
    for i, v in enumerate(pts):
        vpp = tuple(sum(mp.mpf(ax[a][b]) * v[b] for b in range(3)) for a in range(3))
        for j, m in enumerate(range(-l, l + 1)):
            Yp[i, j] = ybar(m, v)
            Ypp[i, j] = ybar(m, vpp)
    D = mp.inverse(Ypp[:N, :]) * Yp[:N, :]
    assert mp.norm(Ypp * D - Yp) < mp.mpf(10) ** -28, "frame rotation: projection does not reproduce the extra directions"
    _cache[key] = D
    return D


_rot3d_cache = {}


def rot3d_sectors(lmax):
    """Per y'-mirror sector (slots as in general_sym):
      slots   B1 = B3 slots (l, |m|, p, kind) in the pair-azimuth frame F' / the pair-axis frame F''
      slots2  B2 slots (l, |m_y|, p, kind, kappa) in the frame F_y (z_y = y'), kappa in {1, 1j}: the stored value is w / kappa
      M1      rows over slots2: [(col in slots, real value)]     B2 <- B1  (and B2 <- B3)
      M2      rows over slots:  [(col in slots2, real value)]    B3 <- B2  (and B1 <- B2)
      pairs   [(i_plus, i_minus, m_y, form)] theta phase rotation of a (+,-) pair of slots2; form in {'cx', 'r+', 'r-'}:
                 'cx':  a+ -> c a+ + i s a-,  a- -> c a- + i s a+        'r+': a+ -> c a+ + s a-, a- -> c a- - s a+
                 'r-':  a+ -> c a+ - s a-,  a- -> c a- + s a+            (c, s = cos, sin(m_y theta); inverse: s -> -s)
      entries {(row, col): [(q, value)]} axial operator in B3 (same |m''| only)."""
    if lmax in _rot3d_cache:
        return _rot3d_cache[lmax]
    md = modes(lmax)
    L = len(md)
    nq = 2 * lmax + 1
    idx = {t: i for i, t in enumerate(md)}
    eps = mp.mpf(10) ** -28
    ax_y = [[1, 0, 0], [0, 0, -1], [0, 1, 0]]
    By = mp.matrix(L, L)
    for p in (0, 1):
        for l in range(1, lmax + 1):
            A = frame_rotation_axes(l, ax_y)
            for i, m2 in enumerate(range(-l, l + 1)):
                for j, m1 in enumerate(range(-l, l + 1)):
                    By[idx[(l, m2, p)], idx[(l, m1, p)]] = A[i, j]
    Byi = mp.inverse(By)
    Rm, Rinv, Zc, all2, S2, S2inv, pm_matrices = _axial_operators(lmax)
    pos2 = {t: i for i, t in enumerate(all2)}
    out = []
    for sct, (slots, rows) in enumerate(general_sym(lmax)):
        n = len(slots)
        S, Sinv = pm_matrices(slots)
        Mfull = By * Sinv                                      # F_y modes x B1
        nzrows = [r for r in range(L) if any(abs(Mfull[r, c]) > eps for c in range(n))]
        assert len(nzrows) == n, "a y'-sector must map onto one mirror-parity class of F_y modes"
        combos = []
        for p in (0, 1):
            for l in range(1, lmax + 1):
                for am in range(0, l + 1):
                    if idx[(l, am, p)] not in nzrows:
                        continue
                    assert idx[(l, -am, p)] in nzrows
                    combos += [(l, 0, p, "0")] if am == 0 else [(l, am, p, "+"), (l, am, p, "-")]
        assert len(combos) == n
        C, Cinv = pm_matrices(combos)                          # combos x L,  L x combos
        M1c = C * Mfull                                        # B2 <- B1, complex
        kappa = []
        for r in range(n):
            re = max(abs(mp.re(M1c[r, c])) for c in range(n))
            im = max(abs(mp.im(M1c[r, c])) for c in range(n))
            assert min(re, im) < eps and max(re, im) > eps, "rows of the frame change must be purely real or purely imaginary"
            kappa.append(mp.mpc(1) if im < eps else mp.mpc(0, 1))
        Kd = mp.diag(kappa)
        Kdi = mp.diag([1 / k for k in kappa])
        M1m = Kdi * M1c
        M2m = S * Byi * Cinv * Kd                              # B3 <- B2
        assert max(abs(mp.im(M1m[r, c])) for r in range(n) for c in range(n)) < eps
        assert max(abs(mp.im(M2m[r, c])) for r in range(n) for c in range(n)) < eps
        assert mp.norm(M2m * M1m - mp.eye(n)) < eps
        M1 = [[(c, mp.re(M1m[r, c])) for c in range(n) if abs(M1m[r, c]) > eps] for r in range(n)]
        M2 = [[(c, mp.re(M2m[r, c])) for c in range(n) if abs(M2m[r, c]) > eps] for r in range(n)]
        slots2 = [(l, am, p, kind, kappa[r]) for r, (l, am, p, kind) in enumerate(combos)]
        pairs = []
        for r, (l, am, p, kind) in enumerate(combos):
            if kind == "+":
                assert combos[r + 1] == (l, am, p, "-")
                ratio = kappa[r + 1] / kappa[r]                 # a+ -> c a+ + i s ratio a-
                form = "cx" if abs(ratio - 1) < eps else ("r-" if abs(ratio - mp.mpc(0, 1)) < eps else "r+")
                assert form != "r+" or abs(ratio + mp.mpc(0, 1)) < eps
                pairs.append((r, r + 1, am, form))
        entries = {}
        sel = [pos2[t] for t in slots]
        selset = {r: i for i, r in enumerate(sel)}
        for q in range(nq):
            for i, r in enumerate(sel):
                for c in range(len(all2)):
                    if abs(Zc[q][r, c]) > eps:
                        assert c in selset and all2[c][1] == all2[r][1], "axial operator must stay inside the sector and inside |m''|"
                        entries.setdefault((i, selset[c]), []).append((q, Zc[q][r, c]))
        # end-to-end check against the direct operator at two random pair directions (phi = 0: the phi rotation is the kernel's)
        for th in (mp.mpf("0.7317"), mp.mpf("2.4603")):
            ct = mp.cos(th)
            E = mp.matrix(n, n)
            for r in range(n):
                E[r, r] = 1
            for (ip, im_, m, form) in pairs:
                c_, s_ = mp.cos(m * th), mp.sin(m * th)
                E[ip, ip] = c_
                E[im_, im_] = c_
                if form == "cx":
                    E[ip, im_] = mp.mpc(0, 1) * s_
                    E[im_, ip] = mp.mpc(0, 1) * s_
                elif form == "r+":
                    E[ip, im_] = s_
                    E[im_, ip] = -s_
                else:
                    E[ip, im_] = -s_
                    E[im_, ip] = s_
            Ei = mp.inverse(E)
            for q in range(nq):
                Zq = mp.matrix(n, n)
                for (i, j), lst in entries.items():
                    for (qq, v) in lst:
                        if qq == q:
                            Zq[i, j] = v
                Kf = M2m * Ei * M1m * Zq * M2m * E * M1m
                Kq = mp.matrix(n, n)
                for r in range(n):
                    for (c, lst) in rows[r][q]:
                        Kq[r, c] = sum(v * pbar_general(q, mu, ct) for (mu, v) in lst)
                assert mp.norm(Kf - Kq) < mp.mpf(10) ** -25, ("rotation - axial translation - rotation differs from the direct operator", lmax, sct, q)
        out.append((slots, slots2, M1, M2, pairs, entries))
    _rot3d_cache[lmax] = out
    return out


def emit_rot3d(lmaxes, path):
    """Straight-line code of rot3d_sectors(): one y'-mirror sector per call, three phases around a per-thread scratch vector
    (sr/si, stride AS): A) per (l,p) block: phi rotation, frame change, theta rotation, frame change -> w (scratch);
    B) per |m''| block: axial translation w -> t (scratch, in place); C) per (l,p) block: the way back and the accumulation."""
    def lin(f, dst, src, rows, sel, counter):
        """dst{r} = sum_c value * src{c} for r in sel (real constants, complex values)."""
        for r in sel:
            for part in ("r", "i"):
                expr = None
                for t, (c, v) in enumerate(rows[r]):
                    if t == 0:
                        if abs(v) == 1:
                            expr = f"{'-' if v < 0 else ''}{src}{part}{c}"
                        else:
                            expr = f"R({lit(v)}) * {src}{part}{c}"
                            counter[0] += 1
                            counter[1] += 1
                    else:
                        expr = f"fma(R({lit(v)}), {src}{part}{c}, {expr})"
                        counter[0] += 1
                        counter[1] += 2
                f.write(f"    const R {dst}{part}{r} = {expr};\n")

    def theta_rot(f, src, dst, pairs, sel2, inverse, counter):
        """phase rotation of the B2 slots in sel2: pairs get the real 2x2 rotation, m_y = 0 slots pass through."""
        done = set()
        for (ip, im_, m, form) in pairs:
            if ip not in sel2:
                continue
            assert im_ in sel2 and form in ("r+", "r-")
            sg = 1 if form == "r+" else -1          # a+ -> c a+ + sg s a-,  a- -> c a- - sg s a+
            if inverse:
                sg = -sg
            a, b = ("", "-") if sg > 0 else ("-", "")
            for part in ("r", "i"):
                f.write(f"    const R {dst}{part}{ip} = fma({a}stm[{m}], {src}{part}{im_}, ctm[{m}] * {src}{part}{ip});\n")
                f.write(f"    const R {dst}{part}{im_} = fma({b}stm[{m}], {src}{part}{ip}, ctm[{m}] * {src}{part}{im_});\n")
            counter[0] += 8
            counter[1] += 12
            done.update((ip, im_))
        for r in sel2:
            if r not in done:
                f.write(f"    const R {dst}r{r} = {src}r{r}, {dst}i{r} = {src}i{r};\n")

    with open(path, "w") as f:
        f.write("// GENERATED by gen_tables.py - do not edit.\n")
        f.write("// General 3-D translation apply by rotation - axial translation - rotation for ANY pair direction (DESIGN.md, kernel K2r):\n")
        f.write("// phi phases, constant frame change onto the frame whose z axis is y', theta phases, constant frame change back: z'' is the\n")
        f.write("// pair axis; m''-diagonal axial translation; and the same way back.  One y'-mirror SECTOR per call (slots as in\n")
        f.write("// tm_general3d_gen.cuh).  xs: [own | partner] d-values; cph/sph, cth/sth: cos/sin of the pair's azimuth and polar angle; hr/hi: h_q(kr);\n")
        f.write("// sr/si: per-thread scratch (n slots, stride AS); ar/ai: accumulators of the own sector, pr/pi: the partner sector's share (n slots each, stride AS).\n#pragma once\n\n")
        f.write("#ifndef TM_PIN\n#define TM_PIN(v)      // device build: zero-cost scheduling pin (tm_allpairs.cuh)\n#endif\n\n")
        for lmax in lmaxes:
            md = modes(lmax)
            idx = {t: i for i, t in enumerate(md)}
            half_l = len(md) // 2
            cost = [0, 0]
            for sct, (slots, slots2, M1, M2, pairs, entries) in enumerate(rot3d_sectors(lmax)):
                n = len(slots)
                cnt = [0, 0]
                blocks = []                 # (l, p) -> B1/B3 slot indices and B2 slot indices
                for p in (0, 1):
                    for l in range(1, lmax + 1):
                        b1 = [k for k, s_ in enumerate(slots) if s_[0] == l and s_[2] == p]
                        b2 = [k for k, s_ in enumerate(slots2) if s_[0] == l and s_[2] == p]
                        if b1:
                            assert len(b1) == len(b2)
                            for r in b2:
                                assert all(c in b1 for (c, _) in M1[r]), "frame change must be block diagonal in (l, p)"
                            for r in b1:
                                assert all(c in b2 for (c, _) in M2[r])
                            blocks.append((b1, b2))
                f.write(f"// lmax={lmax} sector={sct}: slots (l,|m|,p,kind) {slots}\n")
                f.write("template <typename R, int AS>\n__device__ __forceinline__ void "
                        f"tm_r3d_pair_L{lmax}_S{sct}(const R* __restrict__ xs, R cph, R sph, R cth, R sth, "
                        "R* hr, R* hi, R* sr, R* si, R* ar, R* ai, R* pr, R* pi) {\n")
                phases = ("    R cm[%d], sm[%d], ctm[%d], stm[%d];\n    cm[0] = R(1); sm[0] = R(0); cm[1] = cph; sm[1] = sph; "
                          "ctm[0] = R(1); stm[0] = R(0); ctm[1] = cth; stm[1] = sth;\n" % ((lmax + 1,) * 4))
                for m in range(2, lmax + 1):
                    phases += (f"    cm[{m}] = cm[{m - 1}] * cph - sm[{m - 1}] * sph; sm[{m}] = sm[{m - 1}] * cph + cm[{m - 1}] * sph; "
                               f"ctm[{m}] = ctm[{m - 1}] * cth - stm[{m - 1}] * sth; stm[{m}] = stm[{m - 1}] * cth + ctm[{m - 1}] * sth;\n")
                cnt[0] += 2 * 8 * max(0, lmax - 1)          # cos/sin(m phi), cos/sin(m theta) by recurrence, in phase A and again in phase C
                cnt[1] += 2 * 12 * max(0, lmax - 1)
                # ---- phase A
                f.write("  // A: into the pair-axis frame, block by block in (l, p)\n  {\n" + phases)
                for (b1, b2) in blocks:
                    f.write("  {\n")
                    for k in b1:
                        l, am, p, kind = slots[k]
                        if kind == "0":
                            f.write(f"    const R xr{k} = xs[{2 * k}], xi{k} = xs[{2 * k + 1}];\n")
                        else:
                            f.write(f"    const R xr{k} = xs[{2 * k}] * cm[{am}] - xs[{2 * (n + k) + 1}] * sm[{am}], "
                                    f"xi{k} = xs[{2 * k + 1}] * cm[{am}] + xs[{2 * (n + k)}] * sm[{am}];\n")
                            cnt[0] += 4
                            cnt[1] += 6
                    lin(f, "v", "x", M1, b2, cnt)
                    theta_rot(f, "v", "e", pairs, b2, False, cnt)
                    lin(f, "w", "e", M2, b1, cnt)
                    for k in b1:
                        f.write(f"    sr[{k} * AS] = wr{k}; si[{k} * AS] = wi{k};\n")
                    f.write("  }\n")
                f.write("  }\n")
                # ---- phase B
                f.write("  // B: axial translation along z'', block by block in |m''| (scratch in place)\n")
                for mm in sorted(set(s_[1] for s_ in slots)):
                    grp = [k for k, s_ in enumerate(slots) if s_[1] == mm]
                    f.write("  {\n")
                    for k in grp:
                        f.write(f"    const R wr{k} = sr[{k} * AS], wi{k} = si[{k} * AS];\n")
                    known = {}
                    for i in grp:
                        first = True
                        # opaque pins: the radial sums depend only on h_q, so nothing stops the scheduler from forming all of a block's
                        # sums up front (register spills at lmax >= 5); a zero-cost asm on the h_q a row's NEW sums read keeps
                        # each sum next to its use
                        newq = set()
                        seen = set(known)
                        for j in grp:
                            lst = entries.get((i, j))
                            if lst:
                                s0 = 1 if lst[0][1] > 0 else -1
                                key = tuple((q, mp.nstr(s0 * v, 30)) for (q, v) in lst)
                                if key not in seen:
                                    seen.add(key)
                                    newq.update(q for (q, _) in lst)
                        if newq:
                            f.write("    " + " ".join(f"TM_PIN(hr[{q}]); TM_PIN(hi[{q}]);" for q in sorted(newq)) + "\n")
                        for j in grp:
                            lst = entries.get((i, j))
                            if not lst:
                                continue
                            s0 = 1 if lst[0][1] > 0 else -1
                            key = tuple((q, mp.nstr(s0 * v, 30)) for (q, v) in lst)
                            if key not in known:
                                e = len(known)
                                known[key] = e
                                for part, hh in (("r", "hr"), ("i", "hi")):
                                    expr = None
                                    for t, (q, v) in enumerate(lst):
                                        vv = s0 * v
                                        if t == 0 and abs(vv) == 1:
                                            expr = f"{'-' if vv < 0 else ''}{hh}[{q}]"
                                        elif t == 0:
                                            expr = f"R({lit(vv)}) * {hh}[{q}]"
                                            cnt[0] += 1
                                            cnt[1] += 1
                                        else:
                                            expr = f"fma(R({lit(vv)}), {hh}[{q}], {expr})"
                                            cnt[0] += 1
                                            cnt[1] += 2
                                    f.write(f"    const R e{part}{e} = {expr};\n")
                            e = known[key]
                            sg = "" if s0 > 0 else "-"
                            ng = "-" if s0 > 0 else ""
                            if first:
                                f.write(f"    R tr{i} = {sg}er{e} * wr{j}; tr{i} = fma({ng}ei{e}, wi{j}, tr{i}); "
                                        f"R ti{i} = {sg}er{e} * wi{j}; ti{i} = fma({sg}ei{e}, wr{j}, ti{i});\n")
                                cnt[0] += 4
                                cnt[1] += 6
                                first = False
                            else:
                                f.write(f"    tr{i} = fma({sg}er{e}, wr{j}, tr{i}); tr{i} = fma({ng}ei{e}, wi{j}, tr{i}); "
                                        f"ti{i} = fma({sg}er{e}, wi{j}, ti{i}); ti{i} = fma({sg}ei{e}, wr{j}, ti{i});\n")
                                cnt[0] += 4
                                cnt[1] += 8
                        assert not first
                        f.write(f"    sr[{i} * AS] = tr{i}; si[{i} * AS] = ti{i};\n")     # w_i is already in a register: store t_i at once
                    f.write("  }\n")
                # ---- phase C
                f.write("  // C: back into the pair-azimuth frame and accumulation (own sector: cos, partner sector: sin)\n  {\n" + phases)
                for (b1, b2) in blocks:
                    f.write("  {\n")
                    for k in b1:
                        f.write(f"    const R tr{k} = sr[{k} * AS], ti{k} = si[{k} * AS];\n")
                    lin(f, "v", "t", M1, b2, cnt)
                    theta_rot(f, "v", "e", pairs, b2, True, cnt)
                    lin(f, "u", "e", M2, b1, cnt)
                    for k in b1:
                        l, am, p, kind = slots[k]
                        if kind == "0":
                            f.write(f"    ar[{k} * AS] += ur{k}; ai[{k} * AS] += ui{k};\n")
                            cnt[0] += 2
                            cnt[1] += 2
                        else:
                            f.write(f"    ar[{k} * AS] = fma(ur{k}, cm[{am}], ar[{k} * AS]); ai[{k} * AS] = fma(ui{k}, cm[{am}], ai[{k} * AS]);\n")
                            f.write(f"    pr[{k} * AS] = fma(ui{k}, sm[{am}], pr[{k} * AS]); pi[{k} * AS] = fma(-ur{k}, sm[{am}], pi[{k} * AS]);\n")
                            cnt[0] += 4
                            cnt[1] += 8
                    f.write("  }\n")
                f.write("  }\n}\n")
                cost[0] += cnt[0]
                cost[1] += cnt[1]
                print(f"lmax={lmax} rot3d sector={sct}: n={n} frame-change nnz={sum(len(r) for r in M1)}+{sum(len(r) for r in M2)} "
                      f"axial entries={len(entries)} -> {cnt[0]} FP instructions, {cnt[1]} flop", file=sys.stderr)
                # staging tables and unmix: as in emit_general_sym (same slots)
                sa, sb, ss = [], [], []
                for (l, am, p, kind) in slots:
                    sa.append(idx[(l, am, p)]); sb.append(idx[(l, -am, p)]); ss.append({"0": 0, "+": 1, "-": -1}[kind])
                for (l, am, p, kind) in slots:
                    sa.append(idx[(l, am, p)]); sb.append(idx[(l, -am, p)]); ss.append({"0": 0, "+": -1, "-": 1}[kind])
                f.write(f"__device__ __constant__ int tm_r3d_sa_L{lmax}_S{sct}[{2 * n}] = {{{', '.join(map(str, sa))}}};\n")
                f.write(f"__device__ __constant__ int tm_r3d_sb_L{lmax}_S{sct}[{2 * n}] = {{{', '.join(map(str, sb))}}};\n")
                f.write(f"__device__ __constant__ int tm_r3d_ss_L{lmax}_S{sct}[{2 * n}] = {{{', '.join(map(str, ss))}}};\n")
                f.write("template <typename R, typename C, int AS>\n__device__ __forceinline__ void "
                        f"tm_r3d_unmix_L{lmax}_S{sct}(const R* ar, const R* ai, const R* pr, const R* pi, C* out) {{\n")
                for r, (l, am, p, kind) in enumerate(slots):
                    def store(i_flat, re, im):
                        if i_flat >= half_l:
                            f.write(f"  out[{i_flat}].re = {im}; out[{i_flat}].im = -({re});\n")
                        else:
                            f.write(f"  out[{i_flat}].re = {re}; out[{i_flat}].im = {im};\n")
                    if kind == "0":
                        store(idx[(l, 0, p)], f"ar[{r} * AS]", f"ai[{r} * AS]")
                    else:
                        plus_r, plus_i = (f"ar[{r} * AS]", f"ai[{r} * AS]") if kind == "+" else (f"pr[{r} * AS]", f"pi[{r} * AS]")
                        minus_r, minus_i = (f"pr[{r} * AS]", f"pi[{r} * AS]") if kind == "+" else (f"ar[{r} * AS]", f"ai[{r} * AS]")
                        store(idx[(l, am, p)], f"R(0.5) * ({plus_r} + {minus_r})", f"R(0.5) * ({plus_i} + {minus_i})")
                        store(idx[(l, -am, p)], f"R(0.5) * ({plus_r} - {minus_r})", f"R(0.5) * ({plus_i} - {minus_i})")
                covered = set()
                for (l, am, p, kind) in slots:
                    covered.add(idx[(l, am, p)]); covered.add(idx[(l, -am, p)])
                for i_flat in range(len(md)):
                    if i_flat not in covered:
                        f.write(f"  out[{i_flat}].re = R(0); out[{i_flat}].im = R(0);\n")
                f.write("}\n")
            f.write(f"#define TM_R3D_FPINST_L{lmax} {cost[0]}   // FP instructions per ordered pair (both sectors, generated apply code only)\n")
            f.write(f"#define TM_R3D_FLOP_L{lmax} {cost[1]}     // flop per ordered pair (FMA = 2)\n\n")


# ----------------------------------------------------------------------------- rot3d, warp-split (lmax >= 4)
# Same mathematics as emit_rot3d.  The NP warps of a block share ONE target per lane.  Phases A (into the pair-axis frame) and B
# (axial translation) touch no accumulator, so in a round every warp runs them - the SAME code, hence a shared instruction stream -
# for a DIFFERENT source of the lane's target and leaves t in its own shared-memory scratch vector [slot][lane]; after a block
# barrier, warp g runs phase C (back into the pair-azimuth frame and accumulation) of the (l, p) blocks it OWNS for each of the NP
# sources of the round.  A thread accumulates only its own blocks' rows - n / NP slots, own sector + partner share - which fits
# its registers: nothing is re-read per pair (the one-thread-per-target version rewrote 1.5 KB of accumulators per pair and
# sector at lmax 6 and was memory-bound; splitting ALL phases over the warps made every warp stream its own code and was
# instruction-fetch-bound, profiles/r02_rot3d.md).
def _r3_lin(f, dst, src, rows, sel, counter):
    for r in sel:
        for part in ("r", "i"):
            expr = None
            for t, (c, v) in enumerate(rows[r]):
                if t == 0:
                    if abs(v) == 1:
                        expr = f"{'-' if v < 0 else ''}{src}{part}{c}"
                    else:
                        expr = f"R({lit(v)}) * {src}{part}{c}"
                        counter[0] += 1
                        counter[1] += 1
                else:
                    expr = f"fma(R({lit(v)}), {src}{part}{c}, {expr})"
                    counter[0] += 1
                    counter[1] += 2
            f.write(f"    const R {dst}{part}{r} = {expr};\n")


def _r3_theta(f, src, dst, pairs, sel2, inverse, counter):
    done = set()
    for (ip, im_, m, form) in pairs:
        if ip not in sel2:
            continue
        assert im_ in sel2 and form in ("r+", "r-")
        sg = 1 if form == "r+" else -1
        if inverse:
            sg = -sg
        a, b = ("", "-") if sg > 0 else ("-", "")
        for part in ("r", "i"):
            f.write(f"    const R {dst}{part}{ip} = fma({a}stm[{m}], {src}{part}{im_}, ctm[{m}] * {src}{part}{ip});\n")
            f.write(f"    const R {dst}{part}{im_} = fma({b}stm[{m}], {src}{part}{ip}, ctm[{m}] * {src}{part}{im_});\n")
        counter[0] += 8
        counter[1] += 12
        done.update((ip, im_))
    for r in sel2:
        if r not in done:
            f.write(f"    const R {dst}r{r} = {src}r{r}, {dst}i{r} = {src}i{r};\n")


def rot3d_ws_partition(lmax, sector, NP):
    """-> (blocks, part_blocks, part_rows): (l,p) blocks [(b1, b2)], block indices per part (LPT on the frame-change work),
    B3 rows per part (contiguous in |m''| order, balanced on the axial work)."""
    slots, slots2, M1, M2, pairs, entries = sector
    n = len(slots)
    blocks = []
    for p in (0, 1):
        for l in range(1, lmax + 1):
            b1 = [k for k, s_ in enumerate(slots) if s_[0] == l and s_[2] == p]
            b2 = [k for k, s_ in enumerate(slots2) if s_[0] == l and s_[2] == p]
            if b1:
                blocks.append((b1, b2))
    cost = [sum(len(M1[r]) for r in b2) + sum(len(M2[r]) for r in b1) + 3 * len(b1) for (b1, b2) in blocks]
    part_blocks = [[] for _ in range(NP)]
    load = [0] * NP
    for bi in sorted(range(len(blocks)), key=lambda i: -cost[i]):
        g = min(range(NP), key=lambda q: load[q])
        part_blocks[g].append(bi)
        load[g] += cost[bi]
    for g in range(NP):
        part_blocks[g].sort()
    order = sorted(range(n), key=lambda k: (slots[k][1], k))           # rows by |m''|
    rcost = [sum(4 + 2 * len(entries[(i, j)]) / 3.0 for j in range(n) if (i, j) in entries) for i in range(n)]
    total = sum(rcost)
    part_rows = [[] for _ in range(NP)]
    acc, g = 0.0, 0
    for i in order:
        if g < NP - 1 and acc + 0.5 * rcost[i] > total * (g + 1) / NP:
            g += 1
        part_rows[g].append(i)
        acc += rcost[i]
    return blocks, part_blocks, part_rows


def emit_rot3d_ws(lmaxes, path, NP=4):
    with open(path, "w") as f:
        f.write("// GENERATED by gen_tables.py - do not edit.\n")
        f.write("// Rotation - axial translation - rotation for any pair direction, WARP-SPLIT (DESIGN.md, kernel K2r at lmax >= 4): one y'-mirror\n")
        f.write("// sector per block, one target per lane.  A_*: phi rotation, frame change, theta rotation, frame change of ALL (l, p) blocks -> w\n")
        f.write("// (scratch wr/wi, [slot * AS]);  B_*: axial translation of ALL rows, w -> t (in place when tr = wr: a |m''| group is read before its rows\n")
        f.write(f"// are written);  C_*_P<g>: the way back of the (l, p) blocks OWNED by part g (one of {NP}) and the accumulation into that part's REGISTER\n")
        f.write("// accumulators (ar/ai own sector, pr/pi partner share; local slot order);  unmix_*_P<g>: the part's share of u.\n#pragma once\n\n")
        f.write("#ifndef TM_PIN\n#define TM_PIN(v)\n#endif\n\n")
        for lmax in lmaxes:
            md = modes(lmax)
            idx = {t: i for i, t in enumerate(md)}
            half_l = len(md) // 2
            cost = [0, 0]
            nslmax = 0
            phases = ("    R cm[%d], sm[%d], ctm[%d], stm[%d];\n    cm[0] = R(1); sm[0] = R(0); cm[1] = cph; sm[1] = sph; "
                      "ctm[0] = R(1); stm[0] = R(0); ctm[1] = cth; stm[1] = sth;\n" % ((lmax + 1,) * 4))
            for m in range(2, lmax + 1):
                phases += (f"    cm[{m}] = cm[{m - 1}] * cph - sm[{m - 1}] * sph; sm[{m}] = sm[{m - 1}] * cph + cm[{m - 1}] * sph; "
                           f"ctm[{m}] = ctm[{m - 1}] * cth - stm[{m - 1}] * sth; stm[{m}] = stm[{m - 1}] * cth + ctm[{m - 1}] * sth;\n")
            nph = (8 * max(0, lmax - 1), 12 * max(0, lmax - 1))
            for sct, sector in enumerate(rot3d_sectors(lmax)):
                slots, slots2, M1, M2, pairs, entries = sector
                n = len(slots)
                blocks, part_blocks, _ = rot3d_ws_partition(lmax, sector, NP)
                sa, sb, ss = [], [], []
                for (l, am, p, kind) in slots:
                    sa.append(idx[(l, am, p)]); sb.append(idx[(l, -am, p)]); ss.append({"0": 0, "+": 1, "-": -1}[kind])
                for (l, am, p, kind) in slots:
                    sa.append(idx[(l, am, p)]); sb.append(idx[(l, -am, p)]); ss.append({"0": 0, "+": -1, "-": 1}[kind])
                f.write(f"// lmax={lmax} sector={sct}: slots (l,|m|,p,kind) {slots}\n")
                f.write(f"__device__ __constant__ int tm_r3w_sa_L{lmax}_S{sct}[{2 * n}] = {{{', '.join(map(str, sa))}}};\n")
                f.write(f"__device__ __constant__ int tm_r3w_sb_L{lmax}_S{sct}[{2 * n}] = {{{', '.join(map(str, sb))}}};\n")
                f.write(f"__device__ __constant__ int tm_r3w_ss_L{lmax}_S{sct}[{2 * n}] = {{{', '.join(map(str, ss))}}};\n")
                covered = set()
                for (l, am, p, kind) in slots:
                    covered.add(idx[(l, am, p)]); covered.add(idx[(l, -am, p)])
                cnt = [0, 0]
                tagS = f"L{lmax}_S{sct}"
                # ---- A: all (l, p) blocks
                f.write("template <typename R, int AS>\n__device__ __forceinline__ void "
                        f"tm_r3w_A_{tagS}(const R* __restrict__ xs, R cph, R sph, R cth, R sth, R* wr, R* wi) {{\n" + phases)
                cnt[0] += nph[0]; cnt[1] += nph[1]
                for (b1, b2) in blocks:
                    f.write("  {\n")
                    for k in b1:
                        l, am, p, kind = slots[k]
                        if kind == "0":
                            f.write(f"    const R xr{k} = xs[{2 * k}], xi{k} = xs[{2 * k + 1}];\n")
                        else:
                            f.write(f"    const R xr{k} = xs[{2 * k}] * cm[{am}] - xs[{2 * (n + k) + 1}] * sm[{am}], "
                                    f"xi{k} = xs[{2 * k + 1}] * cm[{am}] + xs[{2 * (n + k)}] * sm[{am}];\n")
                            cnt[0] += 4; cnt[1] += 6
                    _r3_lin(f, "v", "x", M1, b2, cnt)
                    _r3_theta(f, "v", "e", pairs, b2, False, cnt)
                    _r3_lin(f, "w", "e", M2, b1, cnt)
                    for k in b1:
                        f.write(f"    wr[{k} * AS] = wr{k}; wi[{k} * AS] = wi{k};\n")
                    f.write("  }\n")
                f.write("}\n")
                # ---- B: all rows, one |m''| group after the other
                f.write("template <typename R, int AS>\n__device__ __forceinline__ void "
                        f"tm_r3w_B_{tagS}(R* hr, R* hi, const R* wr, const R* wi, R* tr, R* ti) {{\n")
                for mm in sorted(set(s_[1] for s_ in slots)):
                    grp = [k for k, s_ in enumerate(slots) if s_[1] == mm]
                    f.write("  {\n")
                    for j in grp:
                        f.write(f"    const R wr{j} = wr[{j} * AS], wi{j} = wi[{j} * AS];\n")
                    known = {}
                    for i in grp:
                        first = True
                        newq, seen = set(), set(known)
                        for j in grp:
                            lst = entries.get((i, j))
                            if lst:
                                s0 = 1 if lst[0][1] > 0 else -1
                                key = tuple((q, mp.nstr(s0 * v, 30)) for (q, v) in lst)
                                if key not in seen:
                                    seen.add(key)
                                    newq.update(q for (q, _) in lst)
                        if newq:
                            f.write("    " + " ".join(f"TM_PIN(hr[{q}]); TM_PIN(hi[{q}]);" for q in sorted(newq)) + "\n")
                        for j in grp:
                            lst = entries.get((i, j))
                            if not lst:
                                continue
                            s0 = 1 if lst[0][1] > 0 else -1
                            key = tuple((q, mp.nstr(s0 * v, 30)) for (q, v) in lst)
                            if key not in known:
                                e = len(known)
                                known[key] = e
                                for part, hh in (("r", "hr"), ("i", "hi")):
                                    expr = None
                                    for t, (q, v) in enumerate(lst):
                                        vv = s0 * v
                                        if t == 0 and abs(vv) == 1:
                                            expr = f"{'-' if vv < 0 else ''}{hh}[{q}]"
                                        elif t == 0:
                                            expr = f"R({lit(vv)}) * {hh}[{q}]"
                                            cnt[0] += 1; cnt[1] += 1
                                        else:
                                            expr = f"fma(R({lit(vv)}), {hh}[{q}], {expr})"
                                            cnt[0] += 1; cnt[1] += 2
                                    f.write(f"    const R e{part}{e} = {expr};\n")
                            e = known[key]
                            sg = "" if s0 > 0 else "-"
                            ng = "-" if s0 > 0 else ""
                            if first:
                                f.write(f"    R tr{i} = {sg}er{e} * wr{j}; tr{i} = fma({ng}ei{e}, wi{j}, tr{i}); "
                                        f"R ti{i} = {sg}er{e} * wi{j}; ti{i} = fma({sg}ei{e}, wr{j}, ti{i});\n")
                                cnt[0] += 4; cnt[1] += 6
                                first = False
                            else:
                                f.write(f"    tr{i} = fma({sg}er{e}, wr{j}, tr{i}); tr{i} = fma({ng}ei{e}, wi{j}, tr{i}); "
                                        f"ti{i} = fma({sg}er{e}, wi{j}, ti{i}); ti{i} = fma({sg}ei{e}, wr{j}, ti{i});\n")
                                cnt[0] += 4; cnt[1] += 8
                        assert not first
                        f.write(f"    tr[{i} * AS] = tr{i}; ti[{i} * AS] = ti{i};\n")
                    f.write("  }\n")
                f.write("}\n")
                # ---- C and unmix per owning part
                for g in range(NP):
                    myslots = [k for bi in part_blocks[g] for k in blocks[bi][0]]
                    loc = {k: i for i, k in enumerate(myslots)}
                    nslmax = max(nslmax, len(myslots))
                    tag = f"{tagS}_P{g}"
                    f.write(f"// part {g} owns the (l,p) blocks {[(slots[blocks[bi][0][0]][0], slots[blocks[bi][0][0]][2]) for bi in part_blocks[g]]}\n"
                            f"#define TM_R3W_NSL_{tag} {len(myslots)}\n")
                    f.write("template <typename R, int AS>\n__device__ __forceinline__ void "
                            f"tm_r3w_C_{tag}(R cph, R sph, R cth, R sth, const R* tr, const R* ti, R* ar, R* ai, R* pr, R* pi) {{\n" + phases)
                    cnt[0] += nph[0]; cnt[1] += nph[1]
                    for bi in part_blocks[g]:
                        b1, b2 = blocks[bi]
                        f.write("  {\n")
                        for k in b1:
                            f.write(f"    const R tr{k} = tr[{k} * AS], ti{k} = ti[{k} * AS];\n")
                        _r3_lin(f, "v", "t", M1, b2, cnt)
                        _r3_theta(f, "v", "e", pairs, b2, True, cnt)
                        _r3_lin(f, "u", "e", M2, b1, cnt)
                        for k in b1:
                            l, am, p, kind = slots[k]
                            li = loc[k]
                            if kind == "0":
                                f.write(f"    ar[{li}] += ur{k}; ai[{li}] += ui{k};\n")
                                cnt[0] += 2; cnt[1] += 2
                            else:
                                f.write(f"    ar[{li}] = fma(ur{k}, cm[{am}], ar[{li}]); ai[{li}] = fma(ui{k}, cm[{am}], ai[{li}]);\n")
                                f.write(f"    pr[{li}] = fma(ui{k}, sm[{am}], pr[{li}]); pi[{li}] = fma(-ur{k}, sm[{am}], pi[{li}]);\n")
                                cnt[0] += 4; cnt[1] += 8
                        f.write("  }\n")
                    f.write("}\n")
                    f.write("template <typename R, typename C>\n__device__ __forceinline__ void "
                            f"tm_r3w_unmix_{tag}(const R* ar, const R* ai, const R* pr, const R* pi, C* out) {{\n")

                    def store(i_flat, re, im):
                        if i_flat >= half_l:
                            f.write(f"  out[{i_flat}].re = {im}; out[{i_flat}].im = -({re});\n")
                        else:
                            f.write(f"  out[{i_flat}].re = {re}; out[{i_flat}].im = {im};\n")
                    for k in myslots:
                        l, am, p, kind = slots[k]
                        li = loc[k]
                        if kind == "0":
                            store(idx[(l, 0, p)], f"ar[{li}]", f"ai[{li}]")
                        else:
                            plus_r, plus_i = (f"ar[{li}]", f"ai[{li}]") if kind == "+" else (f"pr[{li}]", f"pi[{li}]")
                            minus_r, minus_i = (f"pr[{li}]", f"pi[{li}]") if kind == "+" else (f"ar[{li}]", f"ai[{li}]")
                            store(idx[(l, am, p)], f"R(0.5) * ({plus_r} + {minus_r})", f"R(0.5) * ({plus_i} + {minus_i})")
                            store(idx[(l, -am, p)], f"R(0.5) * ({plus_r} - {minus_r})", f"R(0.5) * ({plus_i} - {minus_i})")
                    if g == 0:
                        for i_flat in range(len(md)):
                            if i_flat not in covered:
                                f.write(f"  out[{i_flat}].re = R(0); out[{i_flat}].im = R(0);\n")
                    f.write("}\n")
                cost[0] += cnt[0]; cost[1] += cnt[1]
                print(f"lmax={lmax} rot3d-ws sector={sct}: n={n} -> {cnt[0]} FP instructions, {cnt[1]} flop", file=sys.stderr)
            f.write(f"#define TM_R3W_NSLMAX_L{lmax} {nslmax}\n")
            f.write(f"#define TM_R3W_FPINST_L{lmax} {cost[0]}   // FP instructions per ordered pair (both sectors, all parts)\n")
            f.write(f"#define TM_R3W_FLOP_L{lmax} {cost[1]}     // flop per ordered pair (FMA = 2)\n\n")


def main():
    os.makedirs(OUT, exist_ok=True)
    emit_tables([1, 2, 3, 4, 5, 6, 7], os.path.join(OUT, "tm_tables_gen.h"))     # 7: internal (gradient at lmax 6)
    emit_coplanar([1, 2, 3], os.path.join(OUT, "tm_coplanar_gen.cuh"))
    emit_general_sym([1, 2, 3], os.path.join(OUT, "tm_general3d_gen.cuh"))
    emit_coplanar4([4, 5, 6, 7], os.path.join(OUT, "tm_coplanar4_gen.cuh"))     # 7: internal (gradient at lmax 6)
    emit_coplanar_f2([1, 2, 3], os.path.join(OUT, "tm_coplanar_f2_gen.cuh"))
    emit_rot3d([1, 2, 3, 4, 5, 6, 7], os.path.join(OUT, "tm_rot3d_gen.cuh"))      # 7: internal (gradient at lmax 6)
    emit_rot3d_ws([4, 5, 6], os.path.join(OUT, "tm_rot3d_ws_gen.cuh"))


if __name__ == "__main__":
    main()
