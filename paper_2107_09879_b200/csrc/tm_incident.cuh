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

// ------------------------------------------------------------------------------------------------ lmax >= 4
// Same sums as k_incident_gauss, organised for L = 48..96 modes (round 2): ONE WARP per scatterer, LANE = one (l, m >= 0)
// group.  For a (scatterer, source) pair everything that depends on the node beta_q is
//     f_q = w_q G(beta_q) sin(beta_q) e^{i k z cos(beta_q)},  J_n(k rho_T sin(beta_q)),  m pibar_l^m, taubar_l^m, cos(beta_q),
// so the beta sums of Eqs. II15 / II17 factorise into 8 complex node sums per group,
//     X1 = sum_q f_q a_X J_{m-1},  X2 = sum_q f_q a_X J_{m+1},   a_P = m pibar,  a_T = taubar cos(beta),  a_Q = taubar,  a_R = m pibar cos(beta),
// and the source-only algebra (e^{-i m phi0}, i^{m-1}, the amplitudes, Eq. II11's e^{+-i(phi0 - eta)}) is applied ONCE per
// (scatterer, source) and group - for +m and, through J_{-n} = (-1)^n J_n, for -m from the same sums.  Node quantities of the pair
// (J_0..J_{LMAX+1}, f) are staged per warp in shared memory, 64 nodes at a time (lane = node); two sources are processed
// together so that the angular table of a node is loaded once per two sources.  k_incident_gauss keeps all L complex
// accumulators per thread and redoes the source-only algebra at every node (lmax 6: 1.9-5 KB of spills per thread).
template <int LMAX> struct IncGroups {
  static constexpr int NG = LMAX * (LMAX + 3) / 2;        // sum_{l=1..LMAX} (l + 1)
};

template <int LMAX>
__global__ void __launch_bounds__(128)
k_incident_modes(const double* __restrict__ pos, const int* __restrict__ win_of, const double* __restrict__ src,
                 const double2* __restrict__ amp, const int* __restrict__ src_ptr,
                 const GaussNode<LMAX>* __restrict__ nodes, int n_beta, double k, int n_scat, double2* __restrict__ p) {
  constexpr int L = 2 * LMAX * (LMAX + 2), LH = L / 2, NG = IncGroups<LMAX>::NG, NJ = LMAX + 2, NCH = 64, SB = 2;
  static_assert(NG <= 32, "one lane per (l, m >= 0) group");
  __shared__ double s_J[4][SB][NCH][NJ];
  __shared__ double s_F[4][SB][NCH][2];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int j = blockIdx.x * 4 + warp;
  if (j >= n_scat) return;                                // whole warp
  // lane -> (l, m)
  int gl = 1, gm = 0;
  {
    int g = lane < NG ? lane : 0;
    while (g > gl) { g -= gl + 1; ++gl; }
    gm = g;
  }
  const bool active = lane < NG;
  const int w = win_of[j];
  const int s_lo = src_ptr[w], n_src = src_ptr[w + 1] - s_lo;
  const double xj = pos[3 * j], yj = pos[3 * j + 1], zj = pos[3 * j + 2];
  double o_r[4] = {0, 0, 0, 0}, o_i[4] = {0, 0, 0, 0};    // (l,+m,p0), (l,+m,p1), (l,-m,p0), (l,-m,p1)
  const double cl = 1.0 / sqrt(2.0 * gl * (gl + 1));
  const double sgn_m = (gm & 1) ? -1.0 : 1.0;             // (-1)^m

  for (int sb0 = 0; sb0 < n_src; sb0 += SB) {
    const int nsb = min(SB, n_src - sb0);
    double rhoT[SB], rz[SB], cph[SB], sph[SB];
#pragma unroll
    for (int b = 0; b < SB; ++b) {
      const int sidx = s_lo + sb0 + (b < nsb ? b : 0);
      const double rx = xj - src[3 * sidx], ry = yj - src[3 * sidx + 1];
      rz[b] = zj - src[3 * sidx + 2];
      rhoT[b] = sqrt(rx * rx + ry * ry);
      cph[b] = rhoT[b] > 0.0 ? rx / rhoT[b] : 1.0; sph[b] = rhoT[b] > 0.0 ? ry / rhoT[b] : 0.0;    // e^{i phi0}
    }
    // node sums: [b][X][1|2] complex
    double S_r[SB][8], S_i[SB][8];
#pragma unroll
    for (int b = 0; b < SB; ++b)
#pragma unroll
      for (int t = 0; t < 8; ++t) { S_r[b][t] = 0.0; S_i[b][t] = 0.0; }

    for (int q0 = 0; q0 < n_beta; q0 += NCH) {
      const int nq = min(NCH, n_beta - q0);
      __syncwarp();
      // table phase: lane = node
      for (int n = lane; n < nq; n += 32) {
        const double cb = nodes[q0 + n].cb, sbq = nodes[q0 + n].sb, wgt = nodes[q0 + n].wgt;
#pragma unroll
        for (int b = 0; b < SB; ++b) {
          double J[NJ];
          bessel_j_all<LMAX + 1>(k * rhoT[b] * sbq, J);
#pragma unroll
          for (int t = 0; t < NJ; ++t) s_J[warp][b][n][t] = J[t];
          double sz, cz;
          sincos(k * rz[b] * cb, &sz, &cz);
          s_F[warp][b][n][0] = wgt * cz; s_F[warp][b][n][1] = wgt * sz;
        }
      }
      __syncwarp();
      // sum phase: lane = (l, m) group
      if (active) {
        for (int n = 0; n < nq; ++n) {
          const GaussNode<LMAX>& nd = nodes[q0 + n];
          const double mpi = gm * nd.pi_[gl][gm], tau = nd.tau[gl][gm], cb = nd.cb;
          const double aP = mpi, aT = tau * cb, aQ = tau, aR = mpi * cb;
#pragma unroll
          for (int b = 0; b < SB; ++b) {
            const double fr = s_F[warp][b][n][0], fi = s_F[warp][b][n][1];
            const double j2 = s_J[warp][b][n][gm + 1];
            const double j1 = gm > 0 ? s_J[warp][b][n][gm - 1] : -s_J[warp][b][n][1];      // J_{-1} = -J_1
            const double f1r = fr * j1, f1i = fi * j1, f2r = fr * j2, f2i = fi * j2;
            S_r[b][0] = fma(aP, f1r, S_r[b][0]); S_i[b][0] = fma(aP, f1i, S_i[b][0]);      // P1
            S_r[b][1] = fma(aP, f2r, S_r[b][1]); S_i[b][1] = fma(aP, f2i, S_i[b][1]);      // P2
            S_r[b][2] = fma(aT, f1r, S_r[b][2]); S_i[b][2] = fma(aT, f1i, S_i[b][2]);      // T1
            S_r[b][3] = fma(aT, f2r, S_r[b][3]); S_i[b][3] = fma(aT, f2i, S_i[b][3]);      // T2
            S_r[b][4] = fma(aQ, f1r, S_r[b][4]); S_i[b][4] = fma(aQ, f1i, S_i[b][4]);      // Q1
            S_r[b][5] = fma(aQ, f2r, S_r[b][5]); S_i[b][5] = fma(aQ, f2i, S_i[b][5]);      // Q2
            S_r[b][6] = fma(aR, f1r, S_r[b][6]); S_i[b][6] = fma(aR, f1i, S_i[b][6]);      // R1
            S_r[b][7] = fma(aR, f2r, S_r[b][7]); S_i[b][7] = fma(aR, f2i, S_i[b][7]);      // R2
          }
        }
      }
    }
    // source-only algebra, once per (scatterer, source) and group
    if (active) {
#pragma unroll
      for (int b = 0; b < SB; ++b) {
        if (b >= nsb) continue;
        const int sidx = s_lo + sb0 + b;
        const Cx<double> Ax = cx<double>(amp[2 * sidx].x, amp[2 * sidx].y), Ay = cx<double>(amp[2 * sidx + 1].x, amp[2 * sidx + 1].y);
        const Cx<double> iAx = cx<double>(-Ax.im, Ax.re), iAy = cx<double>(-Ay.im, Ay.re);
        const Cx<double> Ep = cx<double>(cph[b], sph[b]), Em = cx<double>(cph[b], -sph[b]);
        Cx<double> em = cx<double>(1.0, 0.0);                                            // e^{-i m phi0}
        for (int t = 0; t < gm; ++t) em = cmul(em, Em);
#pragma unroll
        for (int sg = 0; sg < 2; ++sg) {                                                  // sg = 0: +m, 1: -m
          if (sg == 1 && gm == 0) continue;
          const int m = sg == 0 ? gm : -gm;
          // sums of the signed m (J_{-n} = (-1)^n J_n; pibar, taubar depend on |m|; a_P, a_R carry the sign of m)
          Cx<double> X1[4], X2[4];
#pragma unroll
          for (int t = 0; t < 4; ++t) {
            const Cx<double> a1 = cx<double>(S_r[b][2 * t], S_i[b][2 * t]), a2 = cx<double>(S_r[b][2 * t + 1], S_i[b][2 * t + 1]);
            if (sg == 0) { X1[t] = a1; X2[t] = a2; }
            else {
              const double s = (t == 0 || t == 3) ? sgn_m : -sgn_m;                      // P, R: (-1)^m;  T, Q: (-1)^{m+1}
              X1[t] = cx<double>(s * a2.re, s * a2.im); X2[t] = cx<double>(s * a1.re, s * a1.im);
            }
          }
          // kappa = i^{m-1} e^{-i m phi0} / 2
          const Cx<double> e_m = sg == 0 ? em : cconj(em);
          const Cx<double> kap = cmul_ipow(cx<double>(0.5 * e_m.re, 0.5 * e_m.im), ((m - 1) % 4 + 4) % 4);
          Cx<double> G0[4], G1[4];
#pragma unroll
          for (int t = 0; t < 4; ++t) {
            const Cx<double> a = cmul(Ep, X1[t]), c2 = cmul(Em, X2[t]);
            G0[t] = cmul(kap, csub(a, c2));
            const Cx<double> sum = cmul(kap, cadd(a, c2));
            G1[t] = cx<double>(sum.im, -sum.re);                                          // times -i
          }
          // X order: 0 P, 1 T, 2 Q, 3 R
          Cx<double> v0 = cadd(cadd(cmul(iAx, G0[0]), cmul(Ay, G0[1])), csub(cmul(iAy, G1[0]), cmul(Ax, G1[1])));
          Cx<double> v1 = cadd(csub(cmul(Ax, G0[2]), cmul(iAy, G0[3])), cadd(cmul(Ay, G1[2]), cmul(iAx, G1[3])));
          v0 = cmul_ipow(v0, gl & 3); v1 = cmul_ipow(v1, (gl + 1) & 3);
          const double sc = -4.0 * cl;
          o_r[2 * sg] += sc * v0.re; o_i[2 * sg] += sc * v0.im;
          o_r[2 * sg + 1] += sc * v1.re; o_i[2 * sg + 1] += sc * v1.im;
        }
      }
    }
  }
  if (active) {
    const int a0 = gl * (gl + 1) - 1;
    double2* pj = p + (size_t)j * L;
    pj[a0 + gm] = make_double2(o_r[0], o_i[0]);
    pj[LH + a0 + gm] = make_double2(o_r[1], o_i[1]);
    if (gm > 0) {
      pj[a0 - gm] = make_double2(o_r[2], o_i[2]);
      pj[LH + a0 - gm] = make_double2(o_r[3], o_i[3]);
    }
  }
}
