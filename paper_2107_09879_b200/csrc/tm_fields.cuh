// Scattered-field evaluation (Eqs. I13 / I24):
//   E_sca(x) = sum_i sum_{lmp} s_{lmp;i} Phi_{lmp}(k (x - x_i)),   Z_b H_sca = -i sum_i sum s_{lmp;i} Phi_{l,m,1-p}  (R10)
// with the outgoing VSWFs of Eq. I6 written in spherical components (c_l = [2l(l+1)]^{-1/2}):
//   Phi_{l,m,0} = c_l h_l(kr) [ i m pibar theta_hat - taubar phi_hat ] e^{i m phi}
//   Phi_{l,m,1} = c_l { l(l+1) h_l(kr)/(kr) Pbar r_hat + ([kr h_l]'/(kr)) (taubar theta_hat + i m pibar phi_hat) } e^{i m phi}
//   [x h_l(x)]'/x = h_{l-1}(x) - l h_l(x)/x.
// grid = (ceil(n_pts/128), n_chunk): thread = detector point, blockIdx.y = chunk of sources; partial sums are
// reduced in a fixed order by k_fields_reduce (deterministic).
#pragma once
#include "tm_common.cuh"
#include "tm_special.cuh"

template <int LMAX>
__global__ void __launch_bounds__(128)
k_fields(const double* __restrict__ pos, int n_scat, const double2* __restrict__ s, const double* __restrict__ pts,
         int n_pts, double k, int swap_p, double2* __restrict__ part) {
  constexpr int L = 2 * LMAX * (LMAX + 2);
  constexpr int LH = L / 2;
  const int ip = blockIdx.x * blockDim.x + threadIdx.x;
  const int per = (n_scat + gridDim.y - 1) / gridDim.y;
  const int i0 = blockIdx.y * per, i1 = min(n_scat, i0 + per);
  if (ip >= n_pts) return;
  const double px = pts[3 * ip], py = pts[3 * ip + 1], pz = pts[3 * ip + 2];
  double ex_r = 0, ex_i = 0, ey_r = 0, ey_i = 0, ez_r = 0, ez_i = 0;
  for (int i = i0; i < i1; ++i) {
    const double dx = px - pos[3 * i], dy = py - pos[3 * i + 1], dz = pz - pos[3 * i + 2];
    const double rho2 = dx * dx + dy * dy, r2 = rho2 + dz * dz;
    if (r2 == 0.0) continue;                         // point on this scatterer's centre: its own outgoing waves are singular there
    const double r = sqrt(r2), rho = sqrt(rho2);
    const double ct = dz / r, st = rho / r;
    const double cph = rho > 0.0 ? dx / rho : 1.0, sph = rho > 0.0 ? dy / rho : 0.0;
    const double x = k * r, t = 1.0 / x;
    double sx, cx_;
    sincos(x, &sx, &cx_);
    // h_{-1}..h_LMAX
    double hr[LMAX + 2], hi[LMAX + 2];               // index q+1
    hr[0] = cx_ * t; hi[0] = sx * t; hr[1] = sx * t; hi[1] = -cx_ * t;
    for (int q = 0; q < LMAX; ++q) {
      hr[q + 2] = (2 * q + 1) * t * hr[q + 1] - hr[q];
      hi[q + 2] = (2 * q + 1) * t * hi[q + 1] - hi[q];
    }
    double P[LMAX + 1][LMAX + 1], PI[LMAX + 1][LMAX + 1], TAU[LMAX + 1][LMAX + 1];
    ang_functions<LMAX>(ct, st, P, PI, TAU);
    double er[LMAX + 1], ei[LMAX + 1];               // e^{i m phi}, m >= 0
    er[0] = 1.0; ei[0] = 0.0;
    for (int m = 1; m <= LMAX; ++m) { er[m] = er[m - 1] * cph - ei[m - 1] * sph; ei[m] = ei[m - 1] * cph + er[m - 1] * sph; }
    double fr_r = 0, fr_i = 0, ft_r = 0, ft_i = 0, fp_r = 0, fp_i = 0;   // spherical components
    const double2* si = s + (size_t)i * L;
    for (int l = 1; l <= LMAX; ++l) {
      const double cl = 1.0 / sqrt(2.0 * l * (l + 1));
      const double zr = hr[l + 1], zi = hi[l + 1];                       // h_l
      const double dr = hr[l] - l * t * zr, di = hi[l] - l * t * zi;     // [x h_l]'/x
      const double rr = l * (l + 1) * t * zr, ri = l * (l + 1) * t * zi; // l(l+1) h_l / x
      for (int m = -l; m <= l; ++m) {
        const int am = m < 0 ? -m : m;
        const double pr = er[am], pi = m < 0 ? -ei[am] : ei[am];         // e^{i m phi}
        const int a0 = l * (l + 1) - 1 + m;
        const double2 c0 = swap_p ? si[LH + a0] : si[a0];                // coefficient multiplying Phi_{l,m,0}
        const double2 c1 = swap_p ? si[a0] : si[LH + a0];                // coefficient multiplying Phi_{l,m,1}
        const double mpi = m * PI[l][am], tau = TAU[l][am], pb = P[l][am];
        // A0 = cl * c0 * h_l * e^{i m phi}
        double ur = zr * pr - zi * pi, ui = zr * pi + zi * pr;
        const double A0r = cl * (c0.x * ur - c0.y * ui), A0i = cl * (c0.x * ui + c0.y * ur);
        // theta += i mpi A0 ; phi += -tau A0
        ft_r += -mpi * A0i; ft_i += mpi * A0r;
        fp_r += -tau * A0r; fp_i += -tau * A0i;
        // A1 = cl * c1 * e^{i m phi}
        const double A1r = cl * (c1.x * pr - c1.y * pi), A1i = cl * (c1.x * pi + c1.y * pr);
        // radial: A1 * rr * pb ; theta: A1 * d * tau ; phi: A1 * d * i mpi
        const double Rr = A1r * rr - A1i * ri, Ri = A1r * ri + A1i * rr;
        fr_r += pb * Rr; fr_i += pb * Ri;
        const double Dr = A1r * dr - A1i * di, Di = A1r * di + A1i * dr;
        ft_r += tau * Dr; ft_i += tau * Di;
        fp_r += -mpi * Di; fp_i += mpi * Dr;
      }
    }
    // spherical -> Cartesian: r_hat = (st cph, st sph, ct), theta_hat = (ct cph, ct sph, -st), phi_hat = (-sph, cph, 0)
    ex_r += fr_r * st * cph + ft_r * ct * cph - fp_r * sph;  ex_i += fr_i * st * cph + ft_i * ct * cph - fp_i * sph;
    ey_r += fr_r * st * sph + ft_r * ct * sph + fp_r * cph;  ey_i += fr_i * st * sph + ft_i * ct * sph + fp_i * cph;
    ez_r += fr_r * ct - ft_r * st;                           ez_i += fr_i * ct - ft_i * st;
  }
  double2* o = part + ((size_t)blockIdx.y * n_pts + ip) * 3;
  if (swap_p) {                                      // multiply by -i
    o[0] = make_double2(ex_i, -ex_r); o[1] = make_double2(ey_i, -ey_r); o[2] = make_double2(ez_i, -ez_r);
  } else {
    o[0] = make_double2(ex_r, ex_i); o[1] = make_double2(ey_r, ey_i); o[2] = make_double2(ez_r, ez_i);
  }
}

__global__ void k_fields_reduce(const double2* __restrict__ part, int n_chunk, size_t n, double2* __restrict__ out) {
  const size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (e >= n) return;
  double2 a = part[e];
  for (int c = 1; c < n_chunk; ++c) { a.x += part[(size_t)c * n + e].x; a.y += part[(size_t)c * n + e].y; }
  out[e] = a;
}

// ------------------------------------------------------------------------------------------------ incident field
// Plane wave (Eq. II6): E_inc(x) = E0 exp(i k . x),  E0 = A_beta beta_hat + A_alpha alpha_hat (Cartesian, complex).
__global__ void k_inc_field_plane(const double* __restrict__ pts, int n_pts, double kx, double ky, double kz,
                                  double2 e0x, double2 e0y, double2 e0z, double2* __restrict__ out) {
  const int ip = blockIdx.x * blockDim.x + threadIdx.x;
  if (ip >= n_pts) return;
  double s, c;
  sincos(kx * pts[3 * ip] + ky * pts[3 * ip + 1] + kz * pts[3 * ip + 2], &s, &c);
  out[3 * ip] = make_double2(e0x.x * c - e0x.y * s, e0x.x * s + e0x.y * c);
  out[3 * ip + 1] = make_double2(e0y.x * c - e0y.y * s, e0y.x * s + e0y.y * c);
  out[3 * ip + 2] = make_double2(e0z.x * c - e0z.y * s, e0z.x * s + e0z.y * c);
}

// Angular-spectrum sources (Gaussian beams: reading R9; jinc sources: Eqs. II3-II5), all sources of all windows summed:
//   E(x) = (1/2pi) int A(beta,alpha) exp(i k.(x - x0)) G(beta) sin(beta) cos(beta) dalpha dbeta,
//   A = A^T - z_hat tan(beta) (Ax cos(alpha) + Ay sin(alpha))                                           (Eq. II5)
// with the alpha integral in closed form (Jacobi-Anger): transverse part J_0(rho), z part i J_1(rho) (Ax cos xi + Ay sin xi),
// rho = k rho_T sin(beta), (rho_T, xi) = polar coordinates of x^T - x0^T, and the same Gauss-Legendre nodes in beta as the
// coefficient kernel (wq[q] already holds w_q G(beta_q) sin(beta_q)).  One thread per detector point.
__global__ void __launch_bounds__(128)
k_inc_field_beams(const double* __restrict__ pts, int n_pts, const double* __restrict__ src, const double2* __restrict__ amp,
                  int n_src, const double* __restrict__ wq, const double* __restrict__ cb, const double* __restrict__ sb,
                  int n_beta, double k, double2* __restrict__ out) {
  const int ip = blockIdx.x * blockDim.x + threadIdx.x;
  if (ip >= n_pts) return;
  const double px = pts[3 * ip], py = pts[3 * ip + 1], pz = pts[3 * ip + 2];
  double exr = 0, exi = 0, eyr = 0, eyi = 0, ezr = 0, ezi = 0;
  for (int s = 0; s < n_src; ++s) {
    const double rx = px - src[3 * s], ry = py - src[3 * s + 1], rz = pz - src[3 * s + 2];
    const double rhoT = sqrt(rx * rx + ry * ry);
    const double cxi = rhoT > 0.0 ? rx / rhoT : 1.0, sxi = rhoT > 0.0 ? ry / rhoT : 0.0;
    const double2 Ax = amp[2 * s], Ay = amp[2 * s + 1];
    double tr = 0, ti = 0, zr = 0, zi = 0;           // int w cos(b) J0 e^{ikz cos b},  int w sin(b) J1 e^{ikz cos b}
    for (int q = 0; q < n_beta; ++q) {
      double J[2];
      bessel_j_all<1>(k * rhoT * sb[q], J);
      double sz, cz;
      sincos(k * rz * cb[q], &sz, &cz);
      const double wt = wq[q] * cb[q] * J[0], wz = wq[q] * sb[q] * J[1];
      tr += wt * cz; ti += wt * sz;
      zr += wz * cz; zi += wz * sz;
    }
    exr += Ax.x * tr - Ax.y * ti; exi += Ax.x * ti + Ax.y * tr;
    eyr += Ay.x * tr - Ay.y * ti; eyi += Ay.x * ti + Ay.y * tr;
    // E_z = -i (Ax cos xi + Ay sin xi) (zr + i zi)
    const double gr = Ax.x * cxi + Ay.x * sxi, gi = Ax.y * cxi + Ay.y * sxi;
    const double mr = gr * zr - gi * zi, mi = gr * zi + gi * zr;
    ezr += mi; ezi += -mr;
  }
  out[3 * ip] = make_double2(exr, exi); out[3 * ip + 1] = make_double2(eyr, eyi); out[3 * ip + 2] = make_double2(ezr, ezi);
}
