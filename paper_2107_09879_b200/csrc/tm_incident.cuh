// Incident-field expansion  p_j = a^(0)_j  (Eq. I12) on the device.
//   plane wave:    Eqs. II6-II7: one L-vector (host, closed form) times exp(i k . x_j)
//   Gaussian beam: reading R9 - Eqs. II9-II17 with the alpha integral in closed form
//                  (Gamma_m, Eq. II11) and a Gauss-Legendre sum in beta, Gaussian spectral weight.
//   jinc sources:  the paper's own case (flat spectrum inside the light cone, Eqs. II3-II17), superposed per window
//                  with the Nyquist amplitudes of reading R17 (Eq. II1).
#pragma once
#include "tm_common.cuh"
#include "tm_special.cuh"

// p[j][a] = coef[a] * exp(i kvec . x_j)
__global__ void k_incident_plane(const double* __restrict__ pos, int n_scat, int L, const double2* __restrict__ coef,
                                 double kx, double ky, double kz, double2* __restrict__ p) {
  const size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (e >= (size_t)n_scat * L) return;
  const int j = (int)(e / L), a = (int)(e - (size_t)j * L);
  double s, c;
  sincos(kx * pos[3 * j] + ky * pos[3 * j + 1] + kz * pos[3 * j + 2], &s, &c);
  const double2 q = coef[a];
  p[e] = make_double2(q.x * c - q.y * s, q.x * s + q.y * c);
}

// Per-node table of the beta quadrature (built once per tm_set_incident on the device):
//   wgt = w_q * G(beta) * sin(beta),  cb = cos(beta), sb = sin(beta), pibar/taubar_l^m(beta)
template <int LMAX> struct GaussNode {
  double wgt, cb, sb;
  double pi_[LMAX + 1][LMAX + 1];
  double tau[LMAX + 1][LMAX + 1];
};

// kw0 > 0: Gaussian spectral weight G(beta) = (k w0)^2/2 exp(-(k w0 sin beta)^2/4) (reading R9);
// kw0 <= 0: flat spectrum inside the light cone = jinc source (Eq. II3 with the k_0^2 of d^2k dropped as in Eq. II9).
template <int LMAX>
__global__ void k_gauss_nodes(const double* __restrict__ beta, const double* __restrict__ wq, int n_beta, double kw0,
                              GaussNode<LMAX>* __restrict__ nodes) {
  const int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= n_beta) return;
  double sb, cb;
  sincos(beta[q], &sb, &cb);
  double P[LMAX + 1][LMAX + 1], PI[LMAX + 1][LMAX + 1], TAU[LMAX + 1][LMAX + 1];
  ang_functions<LMAX>(cb, sb, P, PI, TAU);
  GaussNode<LMAX>& nd = nodes[q];
  nd.wgt = wq[q] * (kw0 > 0.0 ? 0.5 * kw0 * kw0 * exp(-0.25 * kw0 * kw0 * sb * sb) : 1.0) * sb;
  nd.cb = cb; nd.sb = sb;
  for (int l = 1; l <= LMAX; ++l)
    for (int m = 0; m <= l; ++m) { nd.pi_[l][m] = PI[l][m]; nd.tau[l][m] = TAU[l][m]; }
}

// One block (128 threads) per scatterer; threads stride over (source, beta node), each accumulating all L modes.
//   rel = x_j - source centre = (rho_T, phi0, z);  rho = k rho_T sin(beta);  ez = exp(i k z cos(beta))
//   Gamma_m(xi, eta, rho) = i^{m-1} e^{-i m xi}/2 [ e^{i(xi-eta)} J_{m-1}(rho) - e^{-i(xi-eta)} J_{m+1}(rho) ]   (II11)
//   p = 0: -4 i^l     c_l ez [ (i m pi Ax + tau cb Ay) G(0) + (i m pi Ay - tau cb Ax) G(pi/2) ]                    (II15)
//   p = 1: -4 i^{l+1} c_l ez [ (tau Ax - i m pi cb Ay) G(0) + (tau Ay + i m pi cb Ax) G(pi/2) ]                    (II17)
template <int LMAX>
__global__ void __launch_bounds__(128)
k_incident_gauss(const double* __restrict__ pos, const int* __restrict__ win_of, const double* __restrict__ src,
                 const double2* __restrict__ amp, const int* __restrict__ src_ptr,
                 const GaussNode<LMAX>* __restrict__ nodes, int n_beta, double k, double2* __restrict__ p) {
  // Sources (beam foci or jinc-source centres) of the scatterer's window: src_ptr[w] <= s < src_ptr[w+1], centre src[s],
  // transverse amplitude (amp[2s], amp[2s+1]).  The block's threads stride over the flattened (source, node) pairs.
  constexpr int L = 2 * LMAX * (LMAX + 2);
  constexpr int LH = L / 2;
  const int j = blockIdx.x;
  const int w = win_of[j];
  const int s_lo = src_ptr[w], n_src = src_ptr[w + 1] - s_lo;
  double ar[L], ai[L];
#pragma unroll
  for (int a = 0; a < L; ++a) { ar[a] = 0.0; ai[a] = 0.0; }

  for (long long it = threadIdx.x; it < (long long)n_src * n_beta; it += blockDim.x) {
    const int sidx = s_lo + (int)(it / n_beta), q = (int)(it % n_beta);
    const double rx = pos[3 * j] - src[3 * sidx], ry = pos[3 * j + 1] - src[3 * sidx + 1], rz = pos[3 * j + 2] - src[3 * sidx + 2];
    const double2 Ax = amp[2 * sidx], Ay = amp[2 * sidx + 1];
    const double rhoT = sqrt(rx * rx + ry * ry);
    const double cph = rhoT > 0.0 ? rx / rhoT : 1.0, sph = rhoT > 0.0 ? ry / rhoT : 0.0;    // e^{i phi0}
    {
    const GaussNode<LMAX>& nd = nodes[q];
    double J[LMAX + 2];
    bessel_j_all<LMAX + 1>(k * rhoT * nd.sb, J);
    double sz, cz;
    sincos(k * rz * nd.cb, &sz, &cz);
    const double fr = nd.wgt * cz, fi = nd.wgt * sz;                 // weight * ez
    // e^{-i m phi0}, m = -LMAX..LMAX, by recurrence
    double er[2 * LMAX + 1], ei[2 * LMAX + 1];
    er[LMAX] = 1.0; ei[LMAX] = 0.0;
    for (int m = 1; m <= LMAX; ++m) {
      er[LMAX + m] = er[LMAX + m - 1] * cph + ei[LMAX + m - 1] * sph;      // e^{-i m phi0}
      ei[LMAX + m] = ei[LMAX + m - 1] * cph - er[LMAX + m - 1] * sph;
      er[LMAX - m] = er[LMAX + m]; ei[LMAX - m] = -ei[LMAX + m];
    }
#pragma unroll
    for (int l = 1; l <= LMAX; ++l) {
      const double cl = 1.0 / sqrt(2.0 * l * (l + 1));
#pragma unroll
      for (int m = -l; m <= l; ++m) {
        const int am = m < 0 ? -m : m;
        // J_{m-1}, J_{m+1} with J_{-n} = (-1)^n J_n
        const int n1 = m - 1, n2 = m + 1;
        const double j1 = (n1 >= 0) ? J[n1] : (((-n1) & 1) ? -J[-n1] : J[-n1]);
        const double j2 = (n2 >= 0) ? J[n2] : (((-n2) & 1) ? -J[-n2] : J[-n2]);
        // G(eta) = i^{m-1} e^{-i m phi0}/2 [ e^{i(phi0-eta)} j1 - e^{-i(phi0-eta)} j2 ]
        // eta = 0:    bracket = (cph + i sph) j1 - (cph - i sph) j2
        // eta = pi/2: e^{i(phi0 - pi/2)} = -i e^{i phi0} = (sph - i cph);  e^{-i(phi0-pi/2)} = (sph + i cph)
        double b0r = cph * (j1 - j2), b0i = sph * (j1 + j2);
        double b1r = sph * (j1 - j2), b1i = -cph * (j1 + j2);
        // multiply by e^{-i m phi0} / 2
        const double emr = 0.5 * er[LMAX + m], emi = 0.5 * ei[LMAX + m];
        double g0r = b0r * emr - b0i * emi, g0i = b0r * emi + b0i * emr;
        double g1r = b1r * emr - b1i * emi, g1i = b1r * emi + b1i * emr;
        // multiply by i^{m-1}
        const int ip = ((m - 1) % 4 + 4) % 4;
        double t;
        if (ip == 1) { t = g0r; g0r = -g0i; g0i = t; t = g1r; g1r = -g1i; g1i = t; }
        else if (ip == 2) { g0r = -g0r; g0i = -g0i; g1r = -g1r; g1i = -g1i; }
        else if (ip == 3) { t = g0r; g0r = g0i; g0i = -t; t = g1r; g1r = g1i; g1i = -t; }
        const double mpi = m * nd.pi_[l][am], tau = nd.tau[l][am], cb = nd.cb;
        // p = 0 bracket: (i mpi Ax + tau cb Ay) g0 + (i mpi Ay - tau cb Ax) g1
        const double c0r = -mpi * Ax.y + tau * cb * Ay.x, c0i = mpi * Ax.x + tau * cb * Ay.y;
        const double c1r = -mpi * Ay.y - tau * cb * Ax.x, c1i = mpi * Ay.x - tau * cb * Ax.y;
        double v0r = c0r * g0r - c0i * g0i + c1r * g1r - c1i * g1i;
        double v0i = c0r * g0i + c0i * g0r + c1r * g1i + c1i * g1r;
        // p = 1 bracket: (tau Ax - i mpi cb Ay) g0 + (tau Ay + i mpi cb Ax) g1
        const double d0r = tau * Ax.x + mpi * cb * Ay.y, d0i = tau * Ax.y - mpi * cb * Ay.x;
        const double d1r = tau * Ay.x - mpi * cb * Ax.y, d1i = tau * Ay.y + mpi * cb * Ax.x;
        double v1r = d0r * g0r - d0i * g0i + d1r * g1r - d1i * g1i;
        double v1i = d0r * g0i + d0i * g0r + d1r * g1i + d1i * g1r;
        // times -4 i^l c_l (p=0), -4 i^{l+1} c_l (p=1), times weight*ez
        const int il = l & 3;
        if (il == 1) { t = v0r; v0r = -v0i; v0i = t; }
        else if (il == 2) { v0r = -v0r; v0i = -v0i; }
        else if (il == 3) { t = v0r; v0r = v0i; v0i = -t; }
        const int il1 = (l + 1) & 3;
        if (il1 == 1) { t = v1r; v1r = -v1i; v1i = t; }
        else if (il1 == 2) { v1r = -v1r; v1i = -v1i; }
        else if (il1 == 3) { t = v1r; v1r = v1i; v1i = -t; }
        const double sc = -4.0 * cl;
        const int a0 = l * (l + 1) - 1 + m, a1 = LH + a0;
        ar[a0] += sc * (v0r * fr - v0i * fi); ai[a0] += sc * (v0r * fi + v0i * fr);
        ar[a1] += sc * (v1r * fr - v1i * fi); ai[a1] += sc * (v1r * fi + v1i * fr);
      }
    }
  }
  }
  // block reduction
  __shared__ double s_r[4][2 * L];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
  for (int a = 0; a < L; ++a) {
    const double vr = warp_sum(ar[a]), vi = warp_sum(ai[a]);
    if (lane == 0) { s_r[warp][2 * a] = vr; s_r[warp][2 * a + 1] = vi; }
  }
  __syncthreads();
  for (int a = threadIdx.x; a < L; a += blockDim.x)
    p[(size_t)j * L + a] = make_double2(s_r[0][2 * a] + s_r[1][2 * a] + s_r[2][2 * a] + s_r[3][2 * a],
                                        s_r[0][2 * a + 1] + s_r[1][2 * a + 1] + s_r[2][2 * a + 1] + s_r[3][2 * a + 1]);
}
