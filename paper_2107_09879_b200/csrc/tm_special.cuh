// Special functions used outside the all-pairs kernel (incident expansion, field evaluation, host tables).
// Own recurrences; shares nothing with oracle/.
#pragma once
#include "tm_common.cuh"
#include <cmath>

// Normalised angular functions for l = 1..LMAX, 0 <= m <= l at polar angle theta (ct = cos, st = sin >= 0)
//   P[l][m]   = Pbar_l^m(cos theta)                       (reading R2: no Condon-Shortley phase)
//   PI[l][m]  = Pbar_l^m(cos theta) / sin theta           (0 for m = 0: always multiplied by m)
//   TAU[l][m] = d Pbar_l^m(cos theta) / d theta
// (PAPER.md:221, 430-434).  Built from U_l^m = d^m P_l/dx^m, a polynomial recurrence that stays regular at the poles:
//   Pbar = N s^m U_l^m,  pibar = N s^{m-1} U_l^m,  taubar = N (m s^{m-1} x U_l^m - s^{m+1} U_l^{m+1}).
template <int LMAX>
__host__ __device__ inline void ang_functions(double ct, double st, double (*P)[LMAX + 1], double (*PI)[LMAX + 1],
                                              double (*TAU)[LMAX + 1]) {
  double U[LMAX + 2][LMAX + 2];                      // U[l][m], m <= l ; U[l][l+1] = 0
  for (int l = 0; l <= LMAX + 1; ++l)
    for (int m = 0; m <= LMAX + 1; ++m) U[l][m] = 0.0;
  double dfact = 1.0;                                // (2m-1)!!
  for (int m = 0; m <= LMAX; ++m) {
    if (m > 0) dfact *= (2 * m - 1);
    U[m][m] = dfact;
    if (m + 1 <= LMAX) U[m + 1][m] = (2 * m + 1) * ct * dfact;
    for (int l = m + 2; l <= LMAX; ++l) U[l][m] = ((2 * l - 1) * ct * U[l - 1][m] - (l + m - 1) * U[l - 2][m]) / (l - m);
  }
  double spow[LMAX + 2];                             // st^k
  spow[0] = 1.0;
  for (int k = 1; k <= LMAX + 1; ++k) spow[k] = spow[k - 1] * st;
  for (int l = 1; l <= LMAX; ++l) {
    double ratio = 1.0;                              // (l-m)!/(l+m)!
    for (int m = 0; m <= l; ++m) {
      if (m > 0) ratio /= (double)((l + m) * (l - m + 1));
      const double N = sqrt(0.5 * (2 * l + 1) * ratio);
      P[l][m] = N * spow[m] * U[l][m];
      PI[l][m] = (m == 0) ? 0.0 : N * spow[m - 1] * U[l][m];
      const double up = (m + 1 <= l) ? U[l][m + 1] : 0.0;
      TAU[l][m] = N * ((m == 0 ? 0.0 : m * spow[m - 1] * ct * U[l][m]) - spow[m + 1] * up);
    }
  }
}

// Cylindrical Bessel J_0..J_nmax(x), x >= 0, by Miller's backward recurrence normalised with
// 1 = J_0 + 2 sum_{k>=1} J_2k  (absolute accuracy ~1e-15, uniform in x; used for Eq. II11).
// The recurrence J_{n-1} = (2n/x) J_n - J_{n+1} starts at an even N = x + 18 x^{1/3} + 30 with J_{N+1} = 0, J_N = 1e-250.  Two steps per
// loop iteration down to the orders that are needed (no stores, no parity test; the coefficient 2n/x is formed from an exact
// double counter), then a fully unrolled tail that stores J_0..J_NMAX.  No rescaling: from 1e-250 the unnormalised values grow by
// at most ~1e100 for the arguments that occur (k rho sin(beta) <= a few hundred), far from overflow.
template <int NMAX>
__host__ __device__ inline void bessel_j_all(double x, double* J) {
  if (x < 1e-8) {
    J[0] = 1.0 - 0.25 * x * x;
    double t = 1.0;
    for (int n = 1; n <= NMAX; ++n) { t *= 0.5 * x / n; J[n] = t; }
    return;
  }
  constexpr int NSTOP = (NMAX + 3) & ~1;             // smallest even number >= NMAX + 2
  int N = (int)(x + 18.0 * cbrt(x > 1.0 ? x : 1.0)) + 30;
  N += (N & 1);                                      // even start
  if (N < NSTOP) N = NSTOP;
  const double tx = 2.0 / x;
  double jp1 = 0.0, jn = 1e-250, sum = 0.0;          // J_{n+1}, J_n (unnormalised), n = N
  double dn = (double)N;
  for (int n = N; n > NSTOP; n -= 2) {
    const double jm1 = fma(dn * tx, jn, -jp1);       // J_{n-1}
    dn -= 1.0;
    const double jm2 = fma(dn * tx, jm1, -jn);       // J_{n-2}, n - 2 even and > 0
    dn -= 1.0;
    sum = fma(2.0, jm2, sum);
    jp1 = jm1; jn = jm2;
  }
#pragma unroll
  for (int m = NSTOP; m >= 1; --m) {                 // jn = J_m -> J_{m-1}
    const double jm1 = fma(dn * tx, jn, -jp1);
    dn -= 1.0;
    jp1 = jn; jn = jm1;
    if (m - 1 <= NMAX) J[m - 1] = jn;
    if (((m - 1) & 1) == 0 && m - 1 > 0) sum = fma(2.0, jn, sum);
  }
  sum += jn;                                         // J_0 term
  const double inv = 1.0 / sum;
#pragma unroll
  for (int n = 0; n <= NMAX; ++n) J[n] *= inv;
}
