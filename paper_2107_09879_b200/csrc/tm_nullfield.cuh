// Null-field (extended boundary condition) transition matrix of homogeneous bodies of revolution - SURVEY.md 8(f) NEXT-4.
// PAPER.md:258-267, Eqs. I10-I11, with the readings R18 (the two terms of the integrand add) and R19 (the matrix with the
// OUTGOING background function is the one that is inverted: T = -B_rg B_out^{-1}); DESIGN.md section 9.
//
//   B_{nu,mu} = int_S [ RPhi_{l'm'p'}(k_s x) x Psi_{l,-m,1-p}(k_b x) + (k_s/k_b) RPhi_{l'm'1-p'}(k_s x) x Psi_{l,-m,p}(k_b x) ] . n dS
//   nu = (l,m,p) background test function, mu = (l',m',p') internal expansion function, Psi = RPhi (B_rg) or Phi (B_out).
//
// For a surface of revolution r = r(theta) the phi integral is 2 pi delta_{mm'} (dropped: it cancels in T), so T is block
// diagonal in m and each block needs one line integral over the generatrix with
//   n dS = r^2 sin(theta) ( r_hat - (r'/r) theta_hat ) dtheta dphi ,
//   (A x B).r_hat = A_th B_ph - A_ph B_th ,  (A x B).theta_hat = A_ph B_r - A_r B_ph ,
// and the wavefunctions in spherical components at phi = 0 (Eq. I6):
//   Psi_{l,m,0} = g_l z_l [ i m pibar theta_hat - taubar phi_hat ] ,
//   Psi_{l,m,1} = g_l { l(l+1) z_l/(kr) Pbar r_hat + [kr z_l]'/(kr) ( taubar theta_hat + i m pibar phi_hat ) } ,  g_l = [2l(l+1)]^{-1/2}.
// One block per (shape, m): the node quantities are staged through shared memory 16 nodes at a time (thread = node), then
// thread = matrix entry accumulates B_rg and the Neumann part B_y (B_out = B_rg + i B_y) in registers in node order
// (deterministic), and the block solves its (<= 24 x 24) system by Gauss-Jordan elimination with row equilibration and
// partial pivoting.  Own code: shares nothing with oracle/nullfield.py, which integrates over the whole surface in 2-D.
#pragma once
#include "tm_common.cuh"
#include "tm_special.cuh"

namespace nullfield {

constexpr int NF_MAX_L = 12;           // largest INTERNAL truncation (the retained lmax is <= TM_MAX_LMAX)
constexpr int NC = 16;                 // nodes per shared-memory stage
constexpr int NLM = NF_MAX_L;          // l values per block (l0..l_int)
constexpr int NBM = 2 * NLM;           // block dimension (l, p)
constexpr int NT = NBM * NBM;          // threads per block = matrix entries of the largest block (576)

// j_l(x), y_l(x), l = 0..lmax+1 (x > 0): j by Miller's downward recurrence normalised with the larger of j_0 / j_1
// (upward recurrence loses j_l for x < l), y upward (stable).
__device__ inline void sph_jy(int lmax, double x, double* j, double* y) {
  const int top = lmax + 1;
  const double s = sin(x), c = cos(x), ix = 1.0 / x;
  const double j0 = s * ix, j1 = (s * ix - c) * ix;
  int N = top + 24 + (int)x;
  double fp1 = 0.0, f = 1e-280;
  for (int n = N; n >= 1; --n) {                     // f = f_n ; f_{n-1} = (2n+1)/x f_n - f_{n+1}
    const double fm1 = (2 * n + 1) * ix * f - fp1;
    fp1 = f; f = fm1;
    if (n - 1 <= top) j[n - 1] = f;
    if (fabs(f) > 1e250) {
      f *= 1e-250; fp1 *= 1e-250;
      for (int q = n - 1; q <= top; ++q) j[q] *= 1e-250;
    }
  }
  const double scale = (fabs(j0) >= fabs(j1)) ? j0 / j[0] : j1 / j[1];
  for (int q = 0; q <= top; ++q) j[q] *= scale;
  y[0] = -c * ix;
  y[1] = (-c * ix - s) * ix;
  for (int q = 1; q < top; ++q) y[q + 1] = (2 * q + 1) * ix * y[q] - y[q - 1];
}

// j_l(z), l = 0..lmax+1, for complex z = k_s r (lossy scatterer medium): the same downward recurrence in complex arithmetic.
__device__ __forceinline__ Cx<double> cdivd(Cx<double> a, Cx<double> b) {
  if (fabs(b.re) >= fabs(b.im)) {                      // Smith's algorithm: no overflow / underflow of |b|^2
    const double t = b.im / b.re, inv = 1.0 / (b.re + b.im * t);
    return cx<double>((a.re + a.im * t) * inv, (a.im - a.re * t) * inv);
  }
  const double t = b.re / b.im, inv = 1.0 / (b.re * t + b.im);
  return cx<double>((a.re * t + a.im) * inv, (a.im * t - a.re) * inv);
}
__device__ inline void sph_j_complex(int lmax, Cx<double> z, Cx<double>* j) {
  const int top = lmax + 1;
  const Cx<double> iz = cdivd(cx<double>(1.0, 0.0), z);
  const double sa = sin(z.re), ca = cos(z.re), ch = cosh(z.im), sh = sinh(z.im);
  const Cx<double> s = cx<double>(sa * ch, ca * sh), c = cx<double>(ca * ch, -sa * sh);
  const Cx<double> j0 = cmul(s, iz), j1 = cmul(csub(cmul(s, iz), c), iz);
  const int N = top + 24 + (int)sqrt(z.re * z.re + z.im * z.im);
  Cx<double> fp1 = cx<double>(0.0, 0.0), f = cx<double>(1e-100, 0.0);
  for (int n = N; n >= 1; --n) {
    const Cx<double> t = cmul(iz, f);
    const Cx<double> fm1 = cx<double>((2 * n + 1) * t.re - fp1.re, (2 * n + 1) * t.im - fp1.im);
    fp1 = f; f = fm1;
    if (n - 1 <= top) j[n - 1] = f;
    if (fabs(f.re) + fabs(f.im) > 1e100) {
      f.re *= 1e-100; f.im *= 1e-100; fp1.re *= 1e-100; fp1.im *= 1e-100;
      for (int q = n - 1; q <= top; ++q) { j[q].re *= 1e-100; j[q].im *= 1e-100; }
    }
  }
  const bool use0 = j0.re * j0.re + j0.im * j0.im >= j1.re * j1.re + j1.im * j1.im;
  const Cx<double> scale = use0 ? cdivd(j0, j[0]) : cdivd(j1, j[1]);
  for (int q = 0; q <= top; ++q) j[q] = cmul(j[q], scale);
}

struct Node {                          // per (node, l): radial triples (z, [x z]'/x, z/x) and angular functions at |m|
  Cx<double> jS[NLM], dS[NLM], qS[NLM];   // regular, scatterer medium (z = k_s r, complex for a lossy medium)
  double jB[NLM], dB[NLM], qB[NLM];    // regular, background         (x = k_b r)
  double yB[NLM], eB[NLM], pB[NLM];    // Neumann part of the outgoing function, background
  double P[NLM], PI[NLM], TAU[NLM];
  double n_r, n_th;                    // r^2 sin(theta) w  and  -r r' sin(theta) w
};

// (A x B) . n dS for vectors given by spherical components
__device__ __forceinline__ Cx<double> cross_dot_n(const Cx<double>* A, const Cx<double>* B, double n_r, double n_th) {
  const Cx<double> er = csub(cmul(A[1], B[2]), cmul(A[2], B[1]));
  const Cx<double> et = csub(cmul(A[2], B[0]), cmul(A[0], B[2]));
  return cx<double>(n_r * er.re + n_th * et.re, n_r * er.im + n_th * et.im);
}

// components (r, theta, phi) at phi = 0 of Psi_{l,m,p} with the radial triple (z, d, q)
__device__ __forceinline__ void comps(int l, int m, int p, double z, double d, double q, double P, double PI, double TAU,
                                      Cx<double>* out) {
  const double g = rsqrt(2.0 * l * (l + 1));
  if (p == 0) {
    out[0] = cx<double>(0.0, 0.0);
    out[1] = cx<double>(0.0, g * z * m * PI);
    out[2] = cx<double>(-g * z * TAU, 0.0);
  } else {
    out[0] = cx<double>(g * l * (l + 1) * q * P, 0.0);
    out[1] = cx<double>(g * d * TAU, 0.0);
    out[2] = cx<double>(0.0, g * d * m * PI);
  }
}

// the same with a complex radial triple (internal field of a lossy medium)
__device__ __forceinline__ void comps_c(int l, int m, int p, Cx<double> z, Cx<double> d, Cx<double> q, double P, double PI, double TAU,
                                        Cx<double>* out) {
  const double g = rsqrt(2.0 * l * (l + 1));
  if (p == 0) {
    const double a = g * m * PI, b = -g * TAU;
    out[0] = cx<double>(0.0, 0.0);
    out[1] = cx<double>(-a * z.im, a * z.re);
    out[2] = cx<double>(b * z.re, b * z.im);
  } else {
    const double a = g * l * (l + 1) * P, b = g * TAU, c = g * m * PI;
    out[0] = cx<double>(a * q.re, a * q.im);
    out[1] = cx<double>(b * d.re, b * d.im);
    out[2] = cx<double>(-c * d.im, c * d.re);
  }
}

// The surface integrals are truncated at l_int >= lmax (the INTERNAL truncation: field expansions inside the method); the
// block system is solved at that size and the rows / columns with l <= lmax are written.  l_int = lmax is the paper's setting.
__global__ void __launch_bounds__(NT)
k_nullfield(int lmax, int l_int, double k_b, Cx<double> k_s, int n_nodes, const double* __restrict__ theta, const double* __restrict__ rad,
            const double* __restrict__ drad, const double* __restrict__ wgt, double2* __restrict__ T_out) {
  __shared__ Node node[NC];
  __shared__ Cx<double> aug[NBM][2 * NBM];
  __shared__ Cx<double> fac[NBM];
  __shared__ int piv;
  const int shape = blockIdx.x, m = (int)blockIdx.y - lmax, am = m < 0 ? -m : m;
  const int l0 = am > 1 ? am : 1, nl = l_int - l0 + 1, nb = 2 * nl;
  const int L = 2 * lmax * (lmax + 2), LH = L / 2;
  const int e = threadIdx.x;
  const bool is_entry = e < nb * nb;
  const int ra = is_entry ? e / nb : 0, cb = is_entry ? e % nb : 0;
  const int l_row = l0 + ra % nl, p_row = ra / nl, l_col = l0 + cb % nl, p_col = cb / nl;
  const Cx<double> ratio = cx<double>(k_s.re / k_b, k_s.im / k_b);
  Cx<double> b_rg = cx<double>(0.0, 0.0), b_y = cx<double>(0.0, 0.0);
  const size_t base = (size_t)shape * n_nodes;

  for (int c0 = 0; c0 < n_nodes; c0 += NC) {
    const int cnt = min(NC, n_nodes - c0);
    __syncthreads();
    if (e < cnt) {                                                        // thread = node
      const double th = theta[base + c0 + e], r = rad[base + c0 + e], dr = drad[base + c0 + e], w = wgt[base + c0 + e];
      double st, ct;
      sincos(th, &st, &ct);
      double P[NF_MAX_L + 1][NF_MAX_L + 1], PI[NF_MAX_L + 1][NF_MAX_L + 1], TAU[NF_MAX_L + 1][NF_MAX_L + 1];
      ang_functions<NF_MAX_L>(ct, st, P, PI, TAU);
      Cx<double> js[NF_MAX_L + 2];
      double jb[NF_MAX_L + 2], yb[NF_MAX_L + 2];
      const Cx<double> xs = cx<double>(k_s.re * r, k_s.im * r);
      const double xb = k_b * r;
      sph_j_complex(l_int, xs, js);
      sph_jy(l_int, xb, jb, yb);
      Node& nd = node[e];
      for (int a = 0; a < nl; ++a) {
        const int l = l0 + a;
        const Cx<double> qs = cdivd(js[l], xs);
        nd.jS[a] = js[l]; nd.dS[a] = cx<double>(js[l - 1].re - l * qs.re, js[l - 1].im - l * qs.im); nd.qS[a] = qs;   // [x z_l]'/x = z_{l-1} - l z_l / x
        nd.jB[a] = jb[l]; nd.dB[a] = jb[l - 1] - l * jb[l] / xb; nd.qB[a] = jb[l] / xb;
        nd.yB[a] = yb[l]; nd.eB[a] = yb[l - 1] - l * yb[l] / xb; nd.pB[a] = yb[l] / xb;
        nd.P[a] = P[l][am]; nd.PI[a] = PI[l][am]; nd.TAU[a] = TAU[l][am];
      }
      nd.n_r = r * r * st * w;
      nd.n_th = -r * dr * st * w;
    }
    __syncthreads();
    if (is_entry) {                                                       // thread = matrix entry
      const int a = l_row - l0, b = l_col - l0;
      for (int i = 0; i < cnt; ++i) {
        const Node& nd = node[i];
        Cx<double> U[3], Us[3], W[3], Ws[3];
        comps_c(l_col, m, p_col, nd.jS[b], nd.dS[b], nd.qS[b], nd.P[b], nd.PI[b], nd.TAU[b], U);         // RPhi_{l'm p'}(k_s)
        comps_c(l_col, m, 1 - p_col, nd.jS[b], nd.dS[b], nd.qS[b], nd.P[b], nd.PI[b], nd.TAU[b], Us);    // RPhi_{l'm 1-p'}(k_s)
        comps(l_row, -m, p_row, nd.jB[a], nd.dB[a], nd.qB[a], nd.P[a], nd.PI[a], nd.TAU[a], W);        // RPhi_{l,-m,p}(k_b)
        comps(l_row, -m, 1 - p_row, nd.jB[a], nd.dB[a], nd.qB[a], nd.P[a], nd.PI[a], nd.TAU[a], Ws);
        Cx<double> t1 = cross_dot_n(U, Ws, nd.n_r, nd.n_th), t2 = cross_dot_n(Us, W, nd.n_r, nd.n_th);
        t2 = cmul(ratio, t2);
        b_rg.re += t1.re + t2.re; b_rg.im += t1.im + t2.im;
        comps(l_row, -m, p_row, nd.yB[a], nd.eB[a], nd.pB[a], nd.P[a], nd.PI[a], nd.TAU[a], W);        // Neumann part
        comps(l_row, -m, 1 - p_row, nd.yB[a], nd.eB[a], nd.pB[a], nd.P[a], nd.PI[a], nd.TAU[a], Ws);
        t1 = cross_dot_n(U, Ws, nd.n_r, nd.n_th); t2 = cmul(ratio, cross_dot_n(Us, W, nd.n_r, nd.n_th));
        b_y.re += t1.re + t2.re; b_y.im += t1.im + t2.im;
      }
    }
  }

  // T_block = -B_rg B_out^{-1}  <=>  B_out^T X^T = -B_rg^T : augmented [ B_out^T | -B_rg^T ], rows = internal index mu
  __syncthreads();
  if (is_entry) {
    aug[cb][ra] = cx<double>(b_rg.re - b_y.im, b_rg.im + b_y.re);          // B_out = B_rg + i B_y
    aug[cb][nb + ra] = cx<double>(-b_rg.re, -b_rg.im);
  }
  __syncthreads();
  if (e < nb) {                                                            // row equilibration
    double big = 0.0;
    for (int j = 0; j < nb; ++j) big = fmax(big, fmax(fabs(aug[e][j].re), fabs(aug[e][j].im)));
    const double s = big > 0.0 ? 1.0 / big : 1.0;
    for (int j = 0; j < 2 * nb; ++j) { aug[e][j].re *= s; aug[e][j].im *= s; }
  }
  __syncthreads();
  for (int k = 0; k < nb; ++k) {
    if (e == 0) {
      int best = k; double bm = -1.0;
      for (int i = k; i < nb; ++i) {
        const double v = aug[i][k].re * aug[i][k].re + aug[i][k].im * aug[i][k].im;
        if (v > bm) { bm = v; best = i; }
      }
      piv = best;
    }
    __syncthreads();
    if (e < 2 * nb && piv != k) { const Cx<double> t = aug[k][e]; aug[k][e] = aug[piv][e]; aug[piv][e] = t; }
    __syncthreads();
    if (e < nb) {
      const Cx<double> d = aug[k][k];
      const double inv = 1.0 / (d.re * d.re + d.im * d.im);
      const Cx<double> x = aug[e][k];
      fac[e] = (e == k) ? cx<double>(0.0, 0.0) : cx<double>((x.re * d.re + x.im * d.im) * inv, (x.im * d.re - x.re * d.im) * inv);
    }
    __syncthreads();
    for (int q = e; q < nb * 2 * nb; q += blockDim.x) {
      const int i = q / (2 * nb), j = q % (2 * nb);
      if (i == k) continue;
      const Cx<double> f = fac[i], v = aug[k][j];
      aug[i][j].re -= f.re * v.re - f.im * v.im;
      aug[i][j].im -= f.re * v.im + f.im * v.re;
    }
    __syncthreads();
  }
  if (is_entry && l_row <= lmax && l_col <= lmax) {                        // T[ra][cb] = X^T[cb][ra] / pivot
    const Cx<double> d = aug[cb][cb], x = aug[cb][nb + ra];
    const double inv = 1.0 / (d.re * d.re + d.im * d.im);
    const int row = p_row * LH + l_row * (l_row + 1) - 1 + m, col = p_col * LH + l_col * (l_col + 1) - 1 + m;
    T_out[((size_t)shape * L + row) * L + col] = make_double2((x.re * d.re + x.im * d.im) * inv, (x.im * d.re - x.re * d.im) * inv);
  }
}

}  // namespace nullfield
