// CPU harness for tests/test_generated_code.py: compiles the GENERATED rotation-based 3-D pair code (csrc/generated/
// tm_rot3d_gen.cuh, any lmax 1..7) as plain host C++ and evaluates u = A_ji x for one pair exactly as k_allpairs_rot3d
// does (staging of own + partner slots, pair angles, Hankel recurrence, both sectors, unmix, sum).
// Build: g++ -DLMAX=3 [-DGEN=\"path\"] ...   stdin: dx dy dz, then L complex numbers x;  stdout: L complex numbers u.
#include <cmath>
#include <cstdio>
#define __device__
#define __forceinline__ inline
#define __constant__ static const
#define __restrict__
#ifndef GEN
#define GEN "../paper_2107_09879_b200/csrc/generated/tm_rot3d_gen.cuh"
#endif
#include GEN
#define CAT2(a, b, c, d) a##b##c##d
#define CAT(a, b, c, d) CAT2(a, b, c, d)
struct C { double re, im; };
int main() {
  const int L = 2 * LMAX * (LMAX + 2), NS = L / 2, NQ = 2 * LMAX + 1;
  double dx, dy, dz;
  if (scanf("%lf %lf %lf", &dx, &dy, &dz) != 3) return 1;
  C x[L], u[L];
  for (int i = 0; i < L; ++i) { if (scanf("%lf %lf", &x[i].re, &x[i].im) != 2) return 1; u[i].re = u[i].im = 0.0; }
  const double k = 2 * M_PI, rho = std::sqrt(dx * dx + dy * dy), r = std::sqrt(rho * rho + dz * dz), t = 1 / (k * r);
  const double cph = rho > 0 ? dx / rho : 1.0, sph = rho > 0 ? dy / rho : 0.0, cth = dz / r, sth = rho / r;
  const double c = std::cos(k * r), s = std::sin(k * r);
  double hr[NQ], hi[NQ], pr = c * t, pi = s * t;
  hr[0] = s * t; hi[0] = -c * t;
  for (int q = 0; q + 1 < NQ; ++q) {
    const double f = (2 * q + 1) * t, nr = f * hr[q] - pr, ni = f * hi[q] - pi;
    pr = hr[q]; pi = hi[q]; hr[q + 1] = nr; hi[q + 1] = ni;
  }
  for (int sct = 0; sct < 2; ++sct) {
    const int* sa = sct ? CAT(tm_r3d_sa_L, LMAX, _S, 1) : CAT(tm_r3d_sa_L, LMAX, _S, 0);
    const int* sb = sct ? CAT(tm_r3d_sb_L, LMAX, _S, 1) : CAT(tm_r3d_sb_L, LMAX, _S, 0);
    const int* ss = sct ? CAT(tm_r3d_ss_L, LMAX, _S, 1) : CAT(tm_r3d_ss_L, LMAX, _S, 0);
    double xs[4 * NS], ar[2 * NS], ai[2 * NS], sr[NS], si[NS];
    for (int kk = 0; kk < 2 * NS; ++kk) {
      ar[kk] = ai[kk] = 0.0;
      C v = x[sa[kk]];
      if (ss[kk]) { const C o = x[sb[kk]]; v.re += ss[kk] * o.re; v.im += ss[kk] * o.im; }
      if (sa[kk] >= NS) { const double tr = v.re; v.re = -v.im; v.im = tr; }
      xs[2 * kk] = v.re; xs[2 * kk + 1] = v.im;
    }
    C part[L];
    for (int i = 0; i < L; ++i) part[i].re = part[i].im = 0.0;
    if (sct == 0) { CAT(tm_r3d_pair_L, LMAX, _S, 0)<double, 1>(xs, cph, sph, cth, sth, hr, hi, sr, si, ar, ai, ar + NS, ai + NS); CAT(tm_r3d_unmix_L, LMAX, _S, 0)<double, C, 1>(ar, ai, ar + NS, ai + NS, part); }
    else { CAT(tm_r3d_pair_L, LMAX, _S, 1)<double, 1>(xs, cph, sph, cth, sth, hr, hi, sr, si, ar, ai, ar + NS, ai + NS); CAT(tm_r3d_unmix_L, LMAX, _S, 1)<double, C, 1>(ar, ai, ar + NS, ai + NS, part); }
    for (int i = 0; i < L; ++i) { u[i].re += part[i].re; u[i].im += part[i].im; }
  }
  for (int i = 0; i < L; ++i) printf("%.17g %.17g\n", u[i].re, u[i].im);
  return 0;
}
