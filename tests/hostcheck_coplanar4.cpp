// CPU harness for tests/test_generated_code.py: compiles the GENERATED four-sector coplanar pair code (csrc/generated/
// tm_coplanar4_gen.cuh, lmax 4..6) as plain host C++ and evaluates u = A_ji x for one in-plane pair exactly as
// k_allpairs_coplanar4 does (staging of own + partner slots, rotation, Hankel recurrence, four sectors x row groups, unmix, sum).
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
#define CAT6_(a, b, c, d, e, f) a##b##c##d##e##f
#define CAT6(a, b, c, d, e, f) CAT6_(a, b, c, d, e, f)
#define NGROUPS CAT(TM_COP4_G_L, LMAX, , )
struct C { double re, im; };
template <int Z, int G> struct Sec;
#define SEC(Z_, G_)                                                                                               \
  template <> struct Sec<Z_, G_> {                                                                                \
    static constexpr int n = CAT(TM_COP4_N_L, LMAX, _Z, Z_);                                                      \
    static constexpr int nr = CAT6(TM_COP4_NR_L, LMAX, _Z, Z_, _G, G_);                                           \
    static const int* sa() { return CAT(tm_cop4_sa_L, LMAX, _Z, Z_); }                                            \
    static const int* sb() { return CAT(tm_cop4_sb_L, LMAX, _Z, Z_); }                                            \
    static const int* ss() { return CAT(tm_cop4_ss_L, LMAX, _Z, Z_); }                                            \
    static void pair(const double* xs, const double* cm, const double* sm, const double* hr, const double* hi,    \
                     double* ar, double* ai) { CAT6(tm_cop4_pair_L, LMAX, _Z, Z_, _G, G_)<double, 1>(xs, cm, sm, hr, hi, ar, ai); } \
    static void unmix(const double* ar, const double* ai, C* out) { CAT6(tm_cop4_unmix_L, LMAX, _Z, Z_, _G, G_)<double, C, 1>(ar, ai, out); } \
  };
#define SECZ(G_) SEC(0, G_) SEC(1, G_) SEC(2, G_) SEC(3, G_)
SECZ(0)
#if NGROUPS > 1
SECZ(1)
#endif
#if NGROUPS > 2
SECZ(2) SECZ(3)
#endif
#if NGROUPS > 4
SECZ(4) SECZ(5) SECZ(6) SECZ(7)
#endif
// one (sector, row group) block of the kernel: stage, accumulate the group's rows, unmix into the group's output modes
template <int Z, int G>
void run(const C* x, const double* cm, const double* sm, const double* hr, const double* hi, C* u, int L) {
  using S = Sec<Z, G>;
  constexpr int n = S::n, nr = S::nr;
  std::vector<double> xs(4 * n), ar(2 * nr, 0.0), ai(2 * nr, 0.0);
  for (int kk = 0; kk < 2 * n; ++kk) {
    C v = x[S::sa()[kk]];
    const int sg = S::ss()[kk];
    if (sg) { const C o = x[S::sb()[kk]]; v.re += sg * o.re; v.im += sg * o.im; }
    if (S::sa()[kk] >= L / 2) { const double tr = v.re; v.re = -v.im; v.im = tr; }
    xs[2 * kk] = v.re; xs[2 * kk + 1] = v.im;
  }
  std::vector<C> part(L, C{0.0, 0.0});
  S::pair(xs.data(), cm, sm, hr, hi, ar.data(), ai.data());
  S::unmix(ar.data(), ai.data(), part.data());
  for (int i = 0; i < L; ++i) { u[i].re += part[i].re; u[i].im += part[i].im; }
}
template <int G>
void run_group(const C* x, const double* cm, const double* sm, const double* hr, const double* hi, C* u, int L) {
  run<0, G>(x, cm, sm, hr, hi, u, L); run<1, G>(x, cm, sm, hr, hi, u, L);
  run<2, G>(x, cm, sm, hr, hi, u, L); run<3, G>(x, cm, sm, hr, hi, u, L);
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
  run_group<0>(x.data(), cm, sm, hr, hi, u.data(), L);
#if NGROUPS > 1
  run_group<1>(x.data(), cm, sm, hr, hi, u.data(), L);
#endif
#if NGROUPS > 2
  run_group<2>(x.data(), cm, sm, hr, hi, u.data(), L); run_group<3>(x.data(), cm, sm, hr, hi, u.data(), L);
#endif
#if NGROUPS > 4
  run_group<4>(x.data(), cm, sm, hr, hi, u.data(), L); run_group<5>(x.data(), cm, sm, hr, hi, u.data(), L);
  run_group<6>(x.data(), cm, sm, hr, hi, u.data(), L); run_group<7>(x.data(), cm, sm, hr, hi, u.data(), L);
#endif
  for (int i = 0; i < L; ++i) printf("%.17g %.17g\n", u[i].re, u[i].im);
  return 0;
}
