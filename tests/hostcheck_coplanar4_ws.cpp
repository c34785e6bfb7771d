// CPU harness for tests/test_generated_code.py: compiles the GENERATED warp-split planar pair code (csrc/generated/
// tm_coplanar4_ws_gen.cuh, lmax 4..6) as plain host C++ and evaluates u = A_ji x for one in-plane pair exactly as
// k_allpairs_coplanar4_ws does: per mirror sector, phase A (phi rotation + frame change -> w), phase B (axial translation, in
// place), then every owner part's phase C (frame change back + accumulation into that part's accumulators) and unmix.
// Build: g++ -DLMAX=6 [-DGEN=\"path\"] ...   stdin: dx dy, then L complex numbers x;  stdout: L complex numbers u.
#include <cmath>
#include <cstdio>
#include <vector>
#define __device__
#define __forceinline__ inline
#define __constant__ static const
#define __restrict__
#ifndef GEN
#define GEN "../paper_2107_09879_b200/csrc/generated/tm_coplanar4_ws_gen.cuh"
#endif
#include GEN
#define CAT6_(a, b, c, d, e, f) a##b##c##d##e##f
#define CAT6(a, b, c, d, e, f) CAT6_(a, b, c, d, e, f)
#define CAT4_(a, b, c, d) a##b##c##d
#define CAT4(a, b, c, d) CAT4_(a, b, c, d)
#define CAT2_(a, b) a##b
#define CAT2(a, b) CAT2_(a, b)
struct C { double re, im; };
#define NSLMAX CAT2(TM_C4W_NSLMAX_L, LMAX)
#define PART_C(Z, P) CAT6(tm_c4w_C_L, LMAX, _Z, Z, _P, P)<double, 1>(cph, sph, wr.data(), wi.data(), ar[P], ai[P], pr[P], pi[P]);
#define PART_U(Z, P) CAT6(tm_c4w_unmix_L, LMAX, _Z, Z, _P, P)<double, C>(ar[P], ai[P], pr[P], pi[P], part.data());
#define SECTOR(Z)                                                                                                  \
  {                                                                                                                \
    const int n = CAT4(TM_C4W_N_L, LMAX, _Z, Z);                                                                   \
    const int *sa = CAT4(tm_c4w_sa_L, LMAX, _Z, Z), *sb = CAT4(tm_c4w_sb_L, LMAX, _Z, Z), *ss = CAT4(tm_c4w_ss_L, LMAX, _Z, Z); \
    std::vector<double> xs(4 * n), wr(n), wi(n);                                                                   \
    double ar[4][NSLMAX], ai[4][NSLMAX], pr[4][NSLMAX], pi[4][NSLMAX];                                             \
    for (int g = 0; g < 4; ++g) for (int q = 0; q < NSLMAX; ++q) ar[g][q] = ai[g][q] = pr[g][q] = pi[g][q] = 0.0;  \
    for (int kk = 0; kk < 2 * n; ++kk) {                                                                           \
      C v = x[sa[kk]];                                                                                             \
      if (ss[kk]) { const C o = x[sb[kk]]; v.re += ss[kk] * o.re; v.im += ss[kk] * o.im; }                         \
      if (sa[kk] >= L / 2) { const double q = v.re; v.re = -v.im; v.im = q; }                                      \
      xs[2 * kk] = v.re; xs[2 * kk + 1] = v.im;                                                                    \
    }                                                                                                              \
    std::vector<C> part(L, C{0.0, 0.0});                                                                           \
    CAT4(tm_c4w_A_L, LMAX, _Z, Z)<double, 1>(xs.data(), cph, sph, wr.data(), wi.data());                           \
    CAT4(tm_c4w_B_L, LMAX, _Z, Z)<double, 1>(hr, hi, wr.data(), wi.data(), wr.data(), wi.data());                  \
    PART_C(Z, 0) PART_C(Z, 1) PART_C(Z, 2) PART_C(Z, 3) PART_U(Z, 0) PART_U(Z, 1) PART_U(Z, 2) PART_U(Z, 3)        \
    for (int i = 0; i < L; ++i) { u[i].re += part[i].re; u[i].im += part[i].im; }                                  \
  }
int main() {
  const int L = 2 * LMAX * (LMAX + 2), NQ = 2 * LMAX + 1;
  double dx, dy;
  if (scanf("%lf %lf", &dx, &dy) != 2) return 1;
  std::vector<C> x(L), u(L, C{0.0, 0.0});
  for (int i = 0; i < L; ++i) if (scanf("%lf %lf", &x[i].re, &x[i].im) != 2) return 1;
  const double k = 2 * M_PI, r = std::sqrt(dx * dx + dy * dy), t = 1 / (k * r);
  const double cph = dx / r, sph = dy / r;
  const double c = std::cos(k * r), s = std::sin(k * r);
  double hr[NQ], hi[NQ], p_r = c * t, p_i = s * t;
  hr[0] = s * t; hi[0] = -c * t;
  for (int q = 0; q + 1 < NQ; ++q) {
    const double f = (2 * q + 1) * t, nr = f * hr[q] - p_r, ni = f * hi[q] - p_i;
    p_r = hr[q]; p_i = hi[q]; hr[q + 1] = nr; hi[q + 1] = ni;
  }
  SECTOR(0) SECTOR(1) SECTOR(2) SECTOR(3)
  for (int i = 0; i < L; ++i) printf("%.17g %.17g\n", u[i].re, u[i].im);
  return 0;
}
