// Scattered-field evaluation (Eqs. I13 / I24):
//   E_sca(x) = sum_i sum_{lmp} s_{lmp;i} Phi_{lmp}(k (x - x_i)),   Z_b H_sca = -i sum_i sum s_{lmp;i} Phi_{l,m,1-p}  (R10)
// with the outgoing VSWFs of Eq. I6 written in spherical components (c_l = [2l(l+1)]^{-1/2}):
//   Phi_{l,m,0} = c_l h_l(kr) [ i m pibar theta_hat - taubar phi_hat ] e^{i m phi}
//   Phi_{l,m,1} = c_l { l(l+1) h_l(kr)/(kr) Pbar r_hat + ([kr h_l]'/(kr)) (taubar theta_hat + i m pibar phi_hat) } e^{i m phi}
//   [x h_l(x)]'/x = h_{l-1}(x) - l h_l(x)/x.
// grid = (ceil(n_pts/128), n_chunk): thread = detector point, blockIdx.y = chunk of sources; partial sums are
// reduced in a fixed order by k_fields_reduce (deterministic).
#pragma once
#include <type_traits>

#include "tm_common.cuh"
#include "tm_special.cuh"

// k_fields_sym, organised for the FP64 pipe:
//  * +m and -m are taken together.  Phi_{l,-m,p} uses the same Pbar, pibar, taubar as Phi_{l,m,p} with m -> -m in the factor of
//    pibar and in the phase, so with  c^+- = c_{l,m} +- c_{l,-m}  (formed once per source and block while the source is staged
//    in shared memory, scaled by c_l):
//        c_m e^{im phi} + c_{-m} e^{-im phi} = c^+ cos(m phi) + i c^- sin(m phi)        (factor of Pbar, taubar)
//        c_m e^{im phi} - c_{-m} e^{-im phi} = c^- cos(m phi) + i c^+ sin(m phi)        (factor of m pibar)
//    i.e. real trigonometric factors, half the complex products of the m loop;
//  * the radial functions do not depend on m: the five m-sums of an l (radial, theta / phi of p = 1, theta / phi of p = 0) are
//    formed first and multiplied by h_l, [x h_l]'/x, l(l+1) h_l / x once per l;
//  * every loop over modes has a compile-time trip count and is unrolled (static_for below): the normalised N_lm U_l^m (recurrence
//    with the constants folded), the trigonometric and radial tables live in registers, the constants are immediates; divisions by loop constants are multiplications by
//    constexpr reciprocals, 1/r and 1/rho come from rsqrt;
//  * 16 sources per round are staged in shared memory (positions + combined coefficients) and read back as broadcasts.
// Staged coefficients of a source, L complex numbers: for l = 1..LMAX at offset 2 (l^2 - 1):
//    [0] c_l c0_{l,0}   [1] c_l c1_{l,0}   then for m = 1..l:  [2 + 4 (m - 1) + {0,1,2,3}] = c_l {c0^+, c0^-, c1^+, c1^-}
// (c0 / c1 = coefficient multiplying Phi_{l,m,0} / Phi_{l,m,1}: s_{l,m,0} / s_{l,m,1} for E, interchanged for Z H, reading R10).
// Measured (profiles/r02_fields.md): 1.43e10 (point, source) pairs/s at lmax 6, 3.6e10 at lmax 3 = 0.80 of the FP64 issue slots; the
// first version of this kernel (loops over m with local-memory tables, +-m separately, global loads) ran at 3.2e9 / 1.0e10.
namespace fsym {

template <int I, int N, typename F>
__device__ __forceinline__ void static_for(F&& f) {
  if constexpr (I < N) {
    f(std::integral_constant<int, I>{});
    static_for<I + 1, N>(f);
  }
}

__host__ __device__ constexpr double csqrt(double x) {                     // Newton from above; compile-time only
  double g = x > 1.0 ? x : 1.0;
  for (int it = 0; it < 80; ++it) g = 0.5 * (g + x / g);
  return g;
}
__host__ __device__ constexpr double norm_lm(int l, int m) {               // sqrt((2l+1)/2 (l-m)!/(l+m)!)
  double r = 1.0;
  for (int k = l - m + 1; k <= l + m; ++k) r /= (double)k;
  return csqrt(0.5 * (2 * l + 1) * r);
}
__host__ __device__ constexpr double dfact(int m) {                        // (2m-1)!!
  double d = 1.0;
  for (int k = 1; k <= m; ++k) d *= (2 * k - 1);
  return d;
}
__host__ __device__ constexpr double c_l(int l) { return 1.0 / csqrt(2.0 * l * (l + 1)); }

}  // namespace fsym

template <int LMAX>
__global__ void __launch_bounds__(128, 3)
k_fields_sym(const double* __restrict__ pos, int n_scat, const double2* __restrict__ s, const double* __restrict__ pts,
             int n_pts, double k, double inv_k, int swap_p, double2* __restrict__ part) {
  using fsym::static_for;
  constexpr int L = 2 * LMAX * (LMAX + 2), LH = L / 2;
  constexpr int SS = 16;                             // sources staged per round: positions + coefficients, read back as broadcasts
  __shared__ double2 s_c[SS * L];
  __shared__ double s_pos[SS * 3];
  const int ip_raw = blockIdx.x * blockDim.x + threadIdx.x;
  const int ip = min(ip_raw, n_pts - 1);             // threads past the end compute a duplicate and do not store (they take part in the barriers)
  const int per = (n_scat + gridDim.y - 1) / gridDim.y;
  const int i0 = blockIdx.y * per, i1 = min(n_scat, i0 + per);
  const double px = pts[3 * ip], py = pts[3 * ip + 1], pz = pts[3 * ip + 2];
  double ex_r = 0, ex_i = 0, ey_r = 0, ey_i = 0, ez_r = 0, ez_i = 0;
  for (int c0 = i0; c0 < i1; c0 += SS) {
   const int ns = min(SS, i1 - c0);
   __syncthreads();
   for (int e = threadIdx.x; e < ns * LH; e += 128) {   // one (source, l, m) per thread; the thread of m >= 0 writes the +-m pair
     const int ii = e / LH, a = e - ii * LH;            // a = l (l + 1) - 1 + m: flat index inside a p half
     int l = 1;
     while ((l + 1) * (l + 1) - 1 <= a) ++l;
     const int m = a - (l * (l + 1) - 1);
     if (m < 0) continue;
     const double2* raw = s + (size_t)(c0 + ii) * L;
     double2* o = s_c + ii * L + 2 * (l * l - 1);
     const double cl = rsqrt(2.0 * l * (l + 1));
     const int h0 = swap_p ? LH : 0, h1 = swap_p ? 0 : LH;
     if (m == 0) {
       const double2 c0v = raw[h0 + a], c1v = raw[h1 + a];
       o[0] = make_double2(cl * c0v.x, cl * c0v.y);
       o[1] = make_double2(cl * c1v.x, cl * c1v.y);
     } else {
       const double2 c0p = raw[h0 + a], c0m = raw[h0 + a - 2 * m], c1p = raw[h1 + a], c1m = raw[h1 + a - 2 * m];
       double2* q = o + 2 + 4 * (m - 1);
       q[0] = make_double2(cl * (c0p.x + c0m.x), cl * (c0p.y + c0m.y));
       q[1] = make_double2(cl * (c0p.x - c0m.x), cl * (c0p.y - c0m.y));
       q[2] = make_double2(cl * (c1p.x + c1m.x), cl * (c1p.y + c1m.y));
       q[3] = make_double2(cl * (c1p.x - c1m.x), cl * (c1p.y - c1m.y));
     }
   }
   for (int e = threadIdx.x; e < ns * 3; e += 128) s_pos[e] = pos[3 * (size_t)c0 + e];
   __syncthreads();
   for (int ii = 0; ii < ns; ++ii) {
    const double dx = px - s_pos[3 * ii], dy = py - s_pos[3 * ii + 1], dz = pz - s_pos[3 * ii + 2];
    const double rho2 = dx * dx + dy * dy, r2 = rho2 + dz * dz;
    if (r2 == 0.0) continue;                         // point on this scatterer's centre: its own outgoing waves are singular there
    const double inv_r = rsqrt(r2);
    const double inv_rho = rho2 > 0.0 ? rsqrt(rho2) : 0.0;
    const double r = r2 * inv_r, rho = rho2 * inv_rho;
    const double ct = dz * inv_r, st = rho * inv_r;
    const double cph = rho2 > 0.0 ? dx * inv_rho : 1.0, sph = dy * inv_rho;
    const double x = k * r, t = inv_r * inv_k;
    double sx, cx_;
    sincos(x, &sx, &cx_);
    double hr[LMAX + 2], hi[LMAX + 2];               // h_{-1}..h_LMAX at index q + 1
    hr[0] = cx_ * t; hi[0] = sx * t; hr[1] = sx * t; hi[1] = -cx_ * t;
    static_for<0, LMAX>([&](auto Q) {
      constexpr int q = decltype(Q)::value;
      hr[q + 2] = fma((2 * q + 1) * t, hr[q + 1], -hr[q]);
      hi[q + 2] = fma((2 * q + 1) * t, hi[q + 1], -hi[q]);
    });
    double V[LMAX + 1][LMAX + 1];                    // normalised N_lm U_l^m, m <= l, by the recurrence of U_l^m with the constants folded
    static_for<0, LMAX + 1>([&](auto M) {
      constexpr int m = decltype(M)::value;
      constexpr double df = fsym::dfact(m);
      V[m][m] = fsym::norm_lm(m, m) * df;
      if constexpr (m + 1 <= LMAX) V[m + 1][m] = (fsym::norm_lm(m + 1, m) * (2 * m + 1) * df) * ct;
      static_for<m + 2, LMAX + 1>([&](auto Lq) {
        constexpr int l = decltype(Lq)::value;
        constexpr double a = (2 * l - 1) * fsym::norm_lm(l, m) / ((l - m) * fsym::norm_lm(l - 1, m));
        constexpr double b = (l + m - 1) * fsym::norm_lm(l, m) / ((l - m) * fsym::norm_lm(l - 2, m));
        V[l][m] = fma(a * ct, V[l - 1][m], -b * V[l - 2][m]);
      });
    });
    double sp_[LMAX + 2];                            // st^k
    sp_[0] = 1.0;
    static_for<1, LMAX + 2>([&](auto K) { constexpr int kk = decltype(K)::value; sp_[kk] = sp_[kk - 1] * st; });
    double cm[LMAX + 1], sm[LMAX + 1];               // cos / sin(m phi)
    cm[0] = 1.0; sm[0] = 0.0;
    static_for<1, LMAX + 1>([&](auto M) {
      constexpr int m = decltype(M)::value;
      cm[m] = cm[m - 1] * cph - sm[m - 1] * sph;
      sm[m] = sm[m - 1] * cph + cm[m - 1] * sph;
    });
    double fr_r = 0, fr_i = 0, ft_r = 0, ft_i = 0, fp_r = 0, fp_i = 0;   // spherical components
    const double2* si = s_c + ii * L;
    static_for<1, LMAX + 1>([&](auto Lq) {
      constexpr int l = decltype(Lq)::value;
      const double2* sl = si + 2 * (l * l - 1);
      // Pbar_{l,m} = s^m V_l^m;  m pibar = m s^{m-1} V_l^m;  taubar_{l,m} = x (m pibar) - kappa_{l,m} Pbar_{l,m+1},
      // kappa_{l,m} = N_{l,m} / N_{l,m+1} = sqrt((l - m)(l + m + 1))  (Pbar_{l,l+1} = 0)
      double Pb[l + 2];
      static_for<0, l + 1>([&](auto M) { constexpr int m = decltype(M)::value; Pb[m] = m == 0 ? V[l][0] : sp_[m] * V[l][m]; });
      Pb[l + 1] = 0.0;
      // m = 0: pibar term absent
      constexpr double K0 = fsym::norm_lm(l, 0) / fsym::norm_lm(l, 1);
      const double P0 = Pb[0], T0 = -K0 * Pb[1];
      const double2 a0 = sl[0], a1 = sl[1];
      double Fr_r = P0 * a1.x, Fr_i = P0 * a1.y;     // sum_m Pbar S1
      double Ft1_r = T0 * a1.x, Ft1_i = T0 * a1.y;   // sum_m taubar S1
      double Fp0_r = T0 * a0.x, Fp0_i = T0 * a0.y;   // sum_m taubar U0
      double Fp1_r = 0, Fp1_i = 0, Ft0_r = 0, Ft0_i = 0;   // sum_m m pibar D1, sum_m m pibar V0
      static_for<1, l + 1>([&](auto M) {
        constexpr int m = decltype(M)::value;
        const double P = Pb[m];
        const double MPI = (m * sp_[m - 1]) * V[l][m];
        double TAU = ct * MPI;
        if constexpr (m < l) {
          constexpr double K = fsym::norm_lm(l, m) / fsym::norm_lm(l, m + 1);
          TAU = fma(-K, Pb[m + 1], TAU);
        }
        const double2 c0p = sl[2 + 4 * (m - 1)], c0m = sl[3 + 4 * (m - 1)];
        const double2 c1p = sl[4 + 4 * (m - 1)], c1m = sl[5 + 4 * (m - 1)];
        const double c = cm[m], s_ = sm[m];
        // S1 = c1+ cos + i c1- sin feeds two sums; U0 = c0+ cos + i c0- sin, V0 = c0- cos + i c0+ sin, D1 = c1- cos + i c1+ sin feed one
        // each: their real factors are applied to cos / sin first
        const double S1r = fma(c1p.x, c, -c1m.y * s_), S1i = fma(c1p.y, c, c1m.x * s_);
        Fr_r = fma(P, S1r, Fr_r);       Fr_i = fma(P, S1i, Fr_i);
        Ft1_r = fma(TAU, S1r, Ft1_r);   Ft1_i = fma(TAU, S1i, Ft1_i);
        const double Tc = TAU * c, Ts = TAU * s_, Mc = MPI * c, Ms = MPI * s_;
        Fp0_r = fma(Tc, c0p.x, fma(-Ts, c0m.y, Fp0_r));   Fp0_i = fma(Tc, c0p.y, fma(Ts, c0m.x, Fp0_i));
        Ft0_r = fma(Mc, c0m.x, fma(-Ms, c0p.y, Ft0_r));   Ft0_i = fma(Mc, c0m.y, fma(Ms, c0p.x, Ft0_i));
        Fp1_r = fma(Mc, c1m.x, fma(-Ms, c1p.y, Fp1_r));   Fp1_i = fma(Mc, c1m.y, fma(Ms, c1p.x, Fp1_i));
      });
      const double zr = hr[l + 1], zi = hi[l + 1];                               // h_l
      const double dr = fma(-(l * t), zr, hr[l]), di = fma(-(l * t), zi, hi[l]); // [x h_l]'/x
      const double rr = (l * (l + 1) * t) * zr, ri = (l * (l + 1) * t) * zi;     // l(l+1) h_l / x
      // radial += rr Fr ; theta += d Ft1 + i h Ft0 ; phi += i d Fp1 - h Fp0
      fr_r = fma(rr, Fr_r, fma(-ri, Fr_i, fr_r));
      fr_i = fma(rr, Fr_i, fma(ri, Fr_r, fr_i));
      ft_r = fma(dr, Ft1_r, fma(-di, Ft1_i, ft_r));
      ft_i = fma(dr, Ft1_i, fma(di, Ft1_r, ft_i));
      ft_r = fma(-zr, Ft0_i, fma(-zi, Ft0_r, ft_r));
      ft_i = fma(zr, Ft0_r, fma(-zi, Ft0_i, ft_i));
      fp_r = fma(-dr, Fp1_i, fma(-di, Fp1_r, fp_r));
      fp_i = fma(dr, Fp1_r, fma(-di, Fp1_i, fp_i));
      fp_r = fma(-zr, Fp0_r, fma(zi, Fp0_i, fp_r));
      fp_i = fma(-zr, Fp0_i, fma(-zi, Fp0_r, fp_i));
    });
    // spherical -> Cartesian: r_hat = (st cph, st sph, ct), theta_hat = (ct cph, ct sph, -st), phi_hat = (-sph, cph, 0)
    const double hr_ = fma(fr_r, st, ft_r * ct), hi_ = fma(fr_i, st, ft_i * ct);     // component along (cph, sph, 0)
    ex_r += fma(hr_, cph, -fp_r * sph);  ex_i += fma(hi_, cph, -fp_i * sph);
    ey_r += fma(hr_, sph, fp_r * cph);   ey_i += fma(hi_, sph, fp_i * cph);
    ez_r += fma(fr_r, ct, -ft_r * st);   ez_i += fma(fr_i, ct, -ft_i * st);
   }
  }
  if (ip_raw >= n_pts) return;
  double2* o = part + ((size_t)blockIdx.y * n_pts + ip) * 3;
  if (swap_p) {                                      // Z H = -i (...)
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
