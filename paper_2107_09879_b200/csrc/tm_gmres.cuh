// Per-window scalar part of the device-resident restarted GMRES ("operations in GMRES other
// than the matrix-vector product"; reading R13): Givens-rotated Hessenberg, residual estimate, convergence
// mask, back-substitution.  All in double precision regardless of the vector precision.  One thread per
// window: these are O(m) / O(m^2) scalar recurrences, their cost is the launch.
#pragma once
#include "tm_common.cuh"

struct TmGmresDev {
  double2* h1;        // [n_win][ldh]   first CGS pass  V^H w
  double2* h2;        // [n_win][ldh]   second CGS pass
  double2* Rm;        // [n_win][m][ldh] rotated Hessenberg columns (upper triangular after rotation)
  double*  cs;        // [n_win][m]
  double2* sn;        // [n_win][m]
  double2* g;         // [n_win][ldh]
  double2* y;         // [n_win][ldh]   solution of the small least-squares problem (zero-padded)
  double*  normw;     // [n_win]        sqrt(sum |w|^2) of the current vector
  double*  bnorm;     // [n_win]
  double*  inv_norm;  // [n_win]
  double*  beta0;     // [n_win]        ||r|| at the start of the cycle
  double*  resid;     // [n_win]        current estimate / true relative residual
  int*     kcols;     // [n_win]        Krylov columns accepted in this cycle
  int*     done;      // [n_win]
  int*     n_active;  // [1]            windows still iterating in this cycle
  int ldh;            // restart + 1
  int m;              // restart
  double inner_floor; // mixed precision: a cycle also ends once the estimate has dropped by this factor (0: off)
};

__device__ __forceinline__ double2 d2mul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 d2conj(double2 a) { return make_double2(a.x, -a.y); }

// Start of a restart cycle: beta = ||r||; first cycle also fixes ||b||.
__global__ void k_gmres_init_cycle(TmGmresDev S, int n_win, int first, double tol) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= n_win) return;
  const double beta = S.normw[w];
  S.beta0[w] = beta;
  if (first) S.bnorm[w] = beta;
  const double bn = S.bnorm[w];
  S.kcols[w] = 0;
  for (int i = 0; i < S.ldh; ++i) { S.g[(size_t)w * S.ldh + i] = make_double2(0.0, 0.0); S.y[(size_t)w * S.ldh + i] = make_double2(0.0, 0.0); }
  S.g[(size_t)w * S.ldh] = make_double2(beta, 0.0);
  const bool fin = !(beta > tol * bn) || beta == 0.0;       // also catches NaN-free zero RHS
  S.done[w] = fin ? 1 : 0;
  S.inv_norm[w] = fin ? 0.0 : 1.0 / beta;
  S.resid[w] = bn > 0.0 ? beta / bn : 0.0;
  if (!fin) atomicAdd(S.n_active, 1);
}

// After Arnoldi step j (0-based): column j of the Hessenberg is h1 + h2 (rows 0..j) and ||w|| (row j+1).
// One WARP per window (blockDim = 32, grid = n_win): the lanes first reduce the window's chunk norms (fixed order) and
// stage the column and the previous rotations in shared memory with parallel loads; lane 0 then runs the sequential
// rotation recurrence out of shared memory.
// (called by one full warp; s_col: shared scratch of (2j+2) double2 + (j+1) doubles)
__device__ __forceinline__ void givens_body(const TmGmresDev& S, int w, int j, double tol, const double* __restrict__ normpart,
                                            const int* __restrict__ win_chunk_ptr, int lane, double2* s_col) {
  if (S.done[w]) return;
  double2* s_sn = s_col + (j + 1);
  double* s_cs = reinterpret_cast<double*>(s_sn + j);
  const int ldh = S.ldh;
  double nn = 0.0;
  for (int c = win_chunk_ptr[w] + lane; c < win_chunk_ptr[w + 1]; c += 32) nn += normpart[c];
  nn = warp_sum(nn);
  const double hn = sqrt(nn);
  const double2* a1 = S.h1 + (size_t)w * ldh;
  const double2* a2 = S.h2 + (size_t)w * ldh;
  double* cs = S.cs + (size_t)w * S.m;
  double2* sn = S.sn + (size_t)w * S.m;
  for (int i = lane; i <= j; i += 32) s_col[i] = make_double2(a1[i].x + a2[i].x, a1[i].y + a2[i].y);
  for (int i = lane; i < j; i += 32) { s_sn[i] = sn[i]; s_cs[i] = cs[i]; }
  __syncwarp();
  if (lane != 0) return;
  double2* col = S.Rm + ((size_t)w * S.m + j) * ldh;
  double2* g = S.g + (size_t)w * ldh;
  S.normw[w] = hn;
  for (int i = 0; i < j; ++i) {            // previous rotations
    const double2 a = s_col[i], b = s_col[i + 1];
    const double2 sb = d2mul(s_sn[i], b);
    const double2 sa = d2mul(d2conj(s_sn[i]), a);
    s_col[i] = make_double2(s_cs[i] * a.x + sb.x, s_cs[i] * a.y + sb.y);
    s_col[i + 1] = make_double2(s_cs[i] * b.x - sa.x, s_cs[i] * b.y - sa.y);
  }
  const double2 a = s_col[j];
  const double aa = sqrt(a.x * a.x + a.y * a.y);
  const double den = sqrt(aa * aa + hn * hn);
  double c; double2 s, r;
  if (den == 0.0) { c = 1.0; s = make_double2(0.0, 0.0); r = make_double2(0.0, 0.0); }
  else if (aa == 0.0) { c = 0.0; s = make_double2(1.0, 0.0); r = make_double2(hn, 0.0); }
  else {
    c = aa / den;
    const double f = hn / (aa * den);                        // s = (a/|a|) * conj(b)/den, b = hn real
    s = make_double2(a.x * f, a.y * f);
    r = make_double2(a.x / aa * den, a.y / aa * den);
  }
  cs[j] = c; sn[j] = s; s_col[j] = r;
  for (int i = 0; i <= j; ++i) col[i] = s_col[i];
  const double2 gj = g[j];
  const double2 gn = d2mul(d2conj(s), gj);
  g[j + 1] = make_double2(-gn.x, -gn.y);
  g[j] = make_double2(c * gj.x, c * gj.y);
  const double est = sqrt(gn.x * gn.x + gn.y * gn.y);
  S.kcols[w] = j + 1;
  const double bn = S.bnorm[w];
  S.resid[w] = est / bn;
  const bool fin = !(est > fmax(tol * bn, S.inner_floor * S.beta0[w])) || !(hn > 0.0);
  if (fin) { S.done[w] = 1; S.inv_norm[w] = 0.0; atomicSub(S.n_active, 1); }
  else S.inv_norm[w] = 1.0 / hn;
}

__global__ void __launch_bounds__(32)
k_gmres_givens(TmGmresDev S, int n_win, int j, double tol, const double* __restrict__ normpart,
               const int* __restrict__ win_chunk_ptr) {
  const int w = blockIdx.x;
  if (w >= n_win || *S.n_active == 0) return;
  extern __shared__ double2 s_givens[];               // [j+1] column, then [j] sn, then cs as doubles
  givens_body(S, w, j, tol, normpart, win_chunk_ptr, threadIdx.x, s_givens);
}

// y = R^{-1} g over the accepted columns.  One warp per window (grid = n_win, block = 32): each row's dot product is
// split over the lanes (parallel loads of the rotated Hessenberg row, fixed summation order), y is kept in shared memory.
#define TM_MAX_LDH 304
__global__ void __launch_bounds__(32) k_gmres_solve_y(TmGmresDev S, int n_win) {
  const int w = blockIdx.x, lane = threadIdx.x;
  if (w >= n_win) return;
  __shared__ double2 s_y[TM_MAX_LDH];
  const int ldh = S.ldh, k = S.kcols[w];
  double2* y = S.y + (size_t)w * ldh;
  for (int i = lane; i < ldh; i += 32) { s_y[i] = i < k ? S.g[(size_t)w * ldh + i] : make_double2(0.0, 0.0); y[i] = make_double2(0.0, 0.0); }
  __syncwarp();
  for (int i = k - 1; i >= 0; --i) {
    double ar = 0.0, ai = 0.0;
    for (int c = i + 1 + lane; c < k; c += 32) {
      const double2 t = d2mul(S.Rm[((size_t)w * S.m + c) * ldh + i], s_y[c]);       // s_y[c] holds y[c] for c > i
      ar += t.x; ai += t.y;
    }
    ar = warp_sum(ar); ai = warp_sum(ai);
    if (lane == 0) {
      const double2 d = S.Rm[((size_t)w * S.m + i) * ldh + i];
      const double dd = d.x * d.x + d.y * d.y;
      const double nr = s_y[i].x - ar, ni = s_y[i].y - ai;
      const double2 yi = dd > 0.0 ? make_double2((nr * d.x + ni * d.y) / dd, (ni * d.x - nr * d.y) / dd) : make_double2(0.0, 0.0);
      s_y[i] = yi;
      y[i] = yi;
    }
    __syncwarp();
  }
}

// resid[w] = normw[w] / bnorm[w]  (true residual after the cycle's update)
__global__ void k_gmres_true_resid(TmGmresDev S, int n_win) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= n_win) return;
  S.resid[w] = S.bnorm[w] > 0.0 ? S.normw[w] / S.bnorm[w] : 0.0;
}
