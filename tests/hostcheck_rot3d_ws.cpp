// CPU harness for tests/test_generated_code.py: compiles the GENERATED warp-split 3-D pair code (csrc/generated/
// tm_rot3d_ws_gen.cuh, lmax 4..6) as plain host C++ and evaluates u = A_ji x for one pair exactly as k_allpairs_rot3d_ws does:
// per sector, phase A (into the scratch vector w), phase B (w -> t, in place), then every part's phase C (into that part's own
// accumulators) and unmix (its share of u).
// Build: g++ -DLMAX=4 [-DGEN=\"path\"] ...   stdin: dx dy dz, then L complex numbers x;  stdout: L complex numbers u.
#include <cmath>
#include <cstdio>
#define __device__
#define __forceinline__ inline
#define __constant__ static const
#define __restrict__
#ifndef GEN
#define GEN "../paper_2107_09879_b200/csrc/generated/tm_rot3d_ws_gen.cuh"
#endif
#include GEN
#define CAT6_(a, b, c, d, e, f) a##b##c##d##e##f
#define CAT6(a, b, c, d, e, f) CAT6_(a, b, c, d, e, f)
#define CAT4_(a, b, c, d) a##b##c##d
#define CAT4(a, b, c, d) CAT4_(a, b, c, d)
#define CAT2_(a, b) a##b
#define CAT2(a, b) CAT2_(a, b)
struct C { double re, im; };
#define NSLMAX CAT2(TM_R3W_NSLMAX_L, LMAX)
#define SEC_AB(S) CAT4(tm_r3w_A_L, LMAX, _S, S)<double, 1>(xs, cph, sph, cth, sth, wr, wi); \
                  CAT4(tm_r3w_B_L, LMAX, _S, S)<double, 1>(hr, hi, wr, wi, wr, wi);
#define PART_C(S, P) CAT6(tm_r3w_C_L, LMAX, _S, S, _P, P)<double, 1>(cph, sph, cth, sth, wr, wi, ar[P], ai[P], pr[P], pi[P]);
#define PART_U(S, P) CAT6(tm_r3w_unmix_L, LMAX, _S, S, _P, P)<double, C>(ar[P], ai[P], pr[P], pi[P], part);
#define ALL(M, S) M(S, 0) M(S, 1) M(S, 2) M(S, 3)
int main() {
  const int L = 2 * LMAX * (LMAX + 2), NS = L / 2, NQ = 2 * LMAX + 1;
  double dx, dy, dz;
  if (scanf("%lf %lf %lf", &dx, &dy, &dz) != 3) return 1;
  C x[L], u[L];
  for (int i = 0; i < L; ++i) { if (scanf("%lf %lf", &x[i].re, &x[i].im) != 2) return 1; u[i].re = u[i].im = 0.0; }
  const double k = 2 * M_PI, rho = std::sqrt(dx * dx + dy * dy), r = std::sqrt(rho * rho + dz * dz), t = 1 / (k * r);
  const double cph = rho > 0 ? dx / rho : 1.0, sph = rho > 0 ? dy / rho : 0.0, cth = dz / r, sth = rho / r;
  const double c = std::cos(k * r), s = std::sin(k * r);
  double hr[NQ], hi[NQ], p_r = c * t, p_i = s * t;
  hr[0] = s * t; hi[0] = -c * t;
  for (int q = 0; q + 1 < NQ; ++q) {
    const double f = (2 * q + 1) * t, nr = f * hr[q] - p_r, ni = f * hi[q] - p_i;
    p_r = hr[q]; p_i = hi[q]; hr[q + 1] = nr; hi[q + 1] = ni;
  }
  for (int sct = 0; sct < 2; ++sct) {
    const int* sa = sct ? CAT4(tm_r3w_sa_L, LMAX, _S, 1) : CAT4(tm_r3w_sa_L, LMAX, _S, 0);
    const int* sb = sct ? CAT4(tm_r3w_sb_L, LMAX, _S, 1) : CAT4(tm_r3w_sb_L, LMAX, _S, 0);
    const int* ss = sct ? CAT4(tm_r3w_ss_L, LMAX, _S, 1) : CAT4(tm_r3w_ss_L, LMAX, _S, 0);
    double xs[4 * NS], wr[NS], wi[NS];
    double ar[4][NSLMAX], ai[4][NSLMAX], pr[4][NSLMAX], pi[4][NSLMAX];
    for (int g = 0; g < 4; ++g) for (int q = 0; q < NSLMAX; ++q) ar[g][q] = ai[g][q] = pr[g][q] = pi[g][q] = 0.0;
    for (int kk = 0; kk < 2 * NS; ++kk) {
      C v = x[sa[kk]];
      if (ss[kk]) { const C o = x[sb[kk]]; v.re += ss[kk] * o.re; v.im += ss[kk] * o.im; }
      if (sa[kk] >= NS) { const double q = v.re; v.re = -v.im; v.im = q; }
      xs[2 * kk] = v.re; xs[2 * kk + 1] = v.im;
    }
    C part[L];
    for (int i = 0; i < L; ++i) part[i].re = part[i].im = 0.0;
    if (sct == 0) { SEC_AB(0) ALL(PART_C, 0) ALL(PART_U, 0) }
    else          { SEC_AB(1) ALL(PART_C, 1) ALL(PART_U, 1) }
    for (int i = 0; i < L; ++i) { u[i].re += part[i].re; u[i].im += part[i].im; }
  }
  for (int i = 0; i < L; ++i) printf("%.17g %.17g\n", u[i].re, u[i].im);
  return 0;
}
