// CPU harness for tests/test_generated_code.py: compiles the GENERATED four-sector coplanar pair code (csrc/generated/
// tm_coplanar4_gen.cuh, lmax 4..6) as plain host C++ and evaluates u = A_ji x for one in-plane pair exactly as
// k_allpairs_coplanar4 does (staging of own + partner slots, rotation, Hankel recurrence, four sectors, unmix, sum).
// Build: g++ -DLMAX=6 ...   stdin: dx dy, then L complex numbers x;  stdout: L complex numbers u.
#include <cmath>
#include <cstdio>
#include <vector>
#define __device__
#define __forceinline__ inline
#define __constant__ static const
#define __restrict__
#include "../paper_2107_09879_b200/csrc/generated/tm_coplanar4_gen.cuh"
#define CAT2(a, b, c, d) a##b##c##d
#define CAT(a, b, c, d) CAT2(a, b, c, d)
struct C { double re, im; };
template <int Z> struct Sec;
#define SEC(Z_)                                                                                                   \
  template <> struct Sec<Z_> {                                                                                    \
    static constexpr int n = CAT(TM_COP4_N_L, LMAX, _Z, Z_);                                                      \
    static const int* sa() { return CAT(tm_cop4_sa_L, LMAX, _Z, Z_); }                                            \
    static const int* sb() { return CAT(tm_cop4_sb_L, LMAX, _Z, Z_); }                                            \
    static const int* ss() { return CAT(tm_cop4_ss_L, LMAX, _Z, Z_); }                                            \
    static void pair(const double* xs, const double* cm, const double* sm, const double* hr, const double* hi,    \
                     double* ar, double* ai) { CAT(tm_cop4_pair_L, LMAX, _Z, Z_)<double, 1>(xs, cm, sm, hr, hi, ar, ai); } \
    static void unmix(const double* ar, const double* ai, C* out) { CAT(tm_cop4_unmix_L, LMAX, _Z, Z_)<double, C, 1>(ar, ai, out); } \
  };
SEC(0) SEC(1) SEC(2) SEC(3)
template <int Z>
void run(const C* x, const double* cm, const double* sm, const double* hr, const double* hi, C* u, int L) {
  constexpr int n = Sec<Z>::n;
  std::vector<double> xs(4 * n), ar(2 * n, 0.0), ai(2 * n, 0.0);
  for (int kk = 0; kk < 2 * n; ++kk) {
    C v = x[Sec<Z>::sa()[kk]];
    const int sg = Sec<Z>::ss()[kk];
    if (sg) { const C o = x[Sec<Z>::sb()[kk]]; v.re += sg * o.re; v.im += sg * o.im; }
    if (Sec<Z>::sa()[kk] >= L / 2) { const double tr = v.re; v.re = -v.im; v.im = tr; }
    xs[2 * kk] = v.re; xs[2 * kk + 1] = v.im;
  }
  std::vector<C> part(L, C{0.0, 0.0});
  Sec<Z>::pair(xs.data(), cm, sm, hr, hi, ar.data(), ai.data());
  Sec<Z>::unmix(ar.data(), ai.data(), part.data());
  for (int i = 0; i < L; ++i) { u[i].re += part[i].re; u[i].im += part[i].im; }
}
int main() {
  const int L = 2 * LMAX * (LMAX + 2), NQ = 2 * LMAX + 1;
  double dx, dy;
  if (scanf("%lf %lf", &dx, &dy) != 2) return 1;
  std::vector<C> x(L), u(L, C{0.0, 0.0});
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
  run<0>(x.data(), cm, sm, hr, hi, u.data(), L); run<1>(x.data(), cm, sm, hr, hi, u.data(), L);
  run<2>(x.data(), cm, sm, hr, hi, u.data(), L); run<3>(x.data(), cm, sm, hr, hi, u.data(), L);
  for (int i = 0; i < L; ++i) printf("%.17g %.17g\n", u[i].re, u[i].im);
  return 0;
}
