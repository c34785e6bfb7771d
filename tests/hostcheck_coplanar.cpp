// CPU harness for tests/test_generated_code.py: compiles the GENERATED coplanar pair code (csrc/generated/
// tm_coplanar_gen.cuh) as plain host C++ and evaluates u = A_ji x for one pair exactly as k_allpairs_coplanar does
// (staging in the +- basis, phase/Hankel recurrences, both parity halves, unmix).  Build: g++ -DLMAX=3 ...
// stdin: dx dy, then L complex numbers x;  stdout: L complex numbers u.
#include <cmath>
#include <cstdio>
#define __device__
#define __forceinline__ inline
#define __constant__ static const
#define __restrict__
#include "../paper_2107_09879_b200/csrc/generated/tm_coplanar_gen.cuh"
#define CAT2(a, b, c, d) a##b##c##d
#define CAT(a, b, c, d) CAT2(a, b, c, d)
struct C { double re, im; };
int main() {
  const int L = 2 * LMAX * (LMAX + 2), NH = L / 2, NQ = 2 * LMAX + 1;
  double dx, dy;
  if (scanf("%lf %lf", &dx, &dy) != 2) return 1;
  C x[L], out[L];
  for (int i = 0; i < L; ++i) if (scanf("%lf %lf", &x[i].re, &x[i].im) != 2) return 1;
  const double k = 2 * M_PI, r = std::sqrt(dx * dx + dy * dy), t = 1 / (k * r);
  double cm[LMAX + 1], sm[LMAX + 1];
  cm[0] = 1; sm[0] = 0; cm[1] = dx / r; sm[1] = dy / r;
  for (int m = 2; m <= LMAX; ++m) { cm[m] = cm[m - 1] * cm[1] - sm[m - 1] * sm[1]; sm[m] = sm[m - 1] * cm[1] + cm[m - 1] * sm[1]; }
  const double c = std::cos(k * r), s = std::sin(k * r);
  double hr[NQ], hi[NQ], pr = c * t, pi = s * t;
  hr[0] = s * t; hi[0] = -c * t;
  for (int q = 0; q + 1 < NQ; ++q) {
    const double f = (2 * q + 1) * t, nr = f * hr[q] - pr, ni = f * hi[q] - pi;
    pr = hr[q]; pi = hi[q]; hr[q + 1] = nr; hi[q + 1] = ni;
  }
  for (int h = 0; h < 2; ++h) {
    const int* sa = h ? CAT(tm_cop_sa_L, LMAX, _H, 1) : CAT(tm_cop_sa_L, LMAX, _H, 0);
    const int* sb = h ? CAT(tm_cop_sb_L, LMAX, _H, 1) : CAT(tm_cop_sb_L, LMAX, _H, 0);
    const int* ss = h ? CAT(tm_cop_ss_L, LMAX, _H, 1) : CAT(tm_cop_ss_L, LMAX, _H, 0);
    double xs[2 * NH], ar[NH], ai[NH];
    for (int kk = 0; kk < NH; ++kk) {
      ar[kk] = ai[kk] = 0.0;
      C v = x[sa[kk]];
      if (ss[kk]) { const C o = x[sb[kk]]; v.re += ss[kk] * o.re; v.im += ss[kk] * o.im; }
      if (sa[kk] >= NH) { const double tr = v.re; v.re = -v.im; v.im = tr; }
      xs[2 * kk] = v.re; xs[2 * kk + 1] = v.im;
    }
    if (h == 0) { CAT(tm_cop_pair_L, LMAX, _H, 0)<double>(xs, cm, sm, hr, hi, ar, ai); CAT(tm_cop_unmix_L, LMAX, _H, 0)<double, C>(ar, ai, out); }
    else { CAT(tm_cop_pair_L, LMAX, _H, 1)<double>(xs, cm, sm, hr, hi, ar, ai); CAT(tm_cop_unmix_L, LMAX, _H, 1)<double, C>(ar, ai, out); }
  }
  for (int i = 0; i < L; ++i) printf("%.17g %.17g\n", out[i].re, out[i].im);
  return 0;
}
