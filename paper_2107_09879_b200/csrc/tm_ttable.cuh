// T-matrix look-up table: interpolation in a geometry parameter and the derivative from the same table (reading R20
// of DESIGN.md: cubic Lagrange through the four nodes around the interval that holds p, derivative of the same piece).
//
// Two kernels.  k_ttable_weights: thread per output site - interval by bisection, the four weights and their derivatives (12
// divisions: done once per site, not once per entry) into a structure-of-arrays scratch; a site outside the table raises a
// flag the host turns into TM_E_INVALID.  k_ttable_apply_{wide,narrow}: per output entry 4 table loads (the table is L2-resident:
// n_tab x n_entry x 16 B), 8 or 16 real FMAs, 1 or 2 coalesced 16-byte stores; bound by the HBM write of T (and dT).
#pragma once
#include <cuda_runtime.h>

namespace ttable {

constexpr int TT_NW = 8;      // w[0..3], dw[0..3] per site, scratch layout [TT_NW][n_out]

__global__ void k_ttable_weights(const double* __restrict__ p_tab, int n_tab, const double* __restrict__ p, int n_out,
                                 int* __restrict__ i0_out, double* __restrict__ w_out, int* __restrict__ bad) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n_out) return;
  const double pj = p[j];
  if (!(pj >= p_tab[0] && pj <= p_tab[n_tab - 1])) {      // also catches NaN
    atomicOr(bad, 1);
    i0_out[j] = 0;
    for (int a = 0; a < TT_NW; ++a) w_out[(size_t)a * n_out + j] = 0.0;
    return;
  }
  // largest i in [0, n_tab - 2] with p_tab[i] <= pj (the last interval is closed on the right)
  int lo = 0, hi = n_tab - 2;
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (p_tab[mid] <= pj) lo = mid; else hi = mid - 1;
  }
  const int i0 = min(max(lo - 1, 0), n_tab - 4);
  double x[4], d[4];
#pragma unroll
  for (int a = 0; a < 4; ++a) { x[a] = p_tab[i0 + a]; d[a] = pj - x[a]; }
#pragma unroll
  for (int a = 0; a < 4; ++a) {
    // the three other nodes of a
    const int b0 = (a + 1) & 3, b1 = (a + 2) & 3, b2 = (a + 3) & 3;
    const double inv = 1.0 / ((x[a] - x[b0]) * (x[a] - x[b1]) * (x[a] - x[b2]));
    w_out[(size_t)a * n_out + j] = d[b0] * d[b1] * d[b2] * inv;
    w_out[(size_t)(4 + a) * n_out + j] = (d[b0] * d[b1] + d[b0] * d[b2] + d[b1] * d[b2]) * inv;
  }
  i0_out[j] = i0;
}

// T_out[j][e] = sum_a w_a(j) T_tab[i0(j) + a][e],  dT_out likewise with dw (dT_out = nullptr when !DERIV).
// Wide tables (n_entry > 256, a full T): one block walks whole sites - the site's weights sit in registers, a thread streams
// entries e = tid, tid + 256, ... two at a time (8 independent 16-byte loads in flight), no index division anywhere (a flat
// "thread per entry" version with idx / n_entry in 64 bits was bound by that division: 3.6 TB/s written against 5.6 TB/s here,
// 0.85 of the measured HBM peak - profiles/r02_ttable.md).
template <bool DERIV>
__global__ void __launch_bounds__(256) k_ttable_apply_wide(const double2* __restrict__ T_tab, unsigned n_entry, const int* __restrict__ i0_in,
                                                           const double* __restrict__ w_in, int n_out, double2* __restrict__ T_out,
                                                           double2* __restrict__ dT_out) {
  constexpr int U = 2;
  for (unsigned j = blockIdx.x; j < (unsigned)n_out; j += gridDim.x) {
    double w[4], dw[4];
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      w[a] = w_in[(size_t)a * n_out + j];
      dw[a] = DERIV ? w_in[(size_t)(4 + a) * n_out + j] : 0.0;
    }
    const double2* row = T_tab + (size_t)i0_in[j] * n_entry;
    double2* o = T_out + (size_t)j * n_entry;
    double2* d = DERIV ? dT_out + (size_t)j * n_entry : nullptr;
    for (unsigned e0 = 0; e0 < n_entry; e0 += 256 * U) {
      double2 t[U][4];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const unsigned e = e0 + u * 256 + threadIdx.x;
#pragma unroll
        for (int a = 0; a < 4; ++a) t[u][a] = e < n_entry ? __ldg(row + (size_t)a * n_entry + e) : make_double2(0.0, 0.0);
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const unsigned e = e0 + u * 256 + threadIdx.x;
        double tr = 0.0, ti = 0.0, dr = 0.0, di = 0.0;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
          tr = fma(w[a], t[u][a].x, tr);
          ti = fma(w[a], t[u][a].y, ti);
          if (DERIV) { dr = fma(dw[a], t[u][a].x, dr); di = fma(dw[a], t[u][a].y, di); }
        }
        if (e < n_entry) {
          __stcs(o + e, make_double2(tr, ti));              // streamed once: keep the table, not the output, in L2
          if (DERIV) __stcs(d + e, make_double2(dr, di));
        }
      }
    }
  }
}

// Narrow tables (n_entry <= 256, a diagonal T): a block holds S = 256 / n_entry sites at a time, thread = (site in block, entry),
// the one division done once per thread.
template <bool DERIV>
__global__ void __launch_bounds__(256) k_ttable_apply_narrow(const double2* __restrict__ T_tab, unsigned n_entry, const int* __restrict__ i0_in,
                                                             const double* __restrict__ w_in, int n_out, double2* __restrict__ T_out,
                                                             double2* __restrict__ dT_out) {
  const unsigned S = 256u / n_entry;
  const unsigned sl = threadIdx.x / n_entry, e = threadIdx.x - sl * n_entry;
  if (sl >= S) return;
  for (size_t j = (size_t)blockIdx.x * S + sl; j < (size_t)n_out; j += (size_t)gridDim.x * S) {
    const double2* row = T_tab + (size_t)i0_in[j] * n_entry + e;
    double tr = 0.0, ti = 0.0, dr = 0.0, di = 0.0;
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      const double2 t = __ldg(row + (size_t)a * n_entry);
      const double w = w_in[(size_t)a * n_out + j];
      tr = fma(w, t.x, tr);
      ti = fma(w, t.y, ti);
      if (DERIV) {
        const double dw = w_in[(size_t)(4 + a) * n_out + j];
        dr = fma(dw, t.x, dr);
        di = fma(dw, t.y, di);
      }
    }
    T_out[j * n_entry + e] = make_double2(tr, ti);
    if (DERIV) dT_out[j * n_entry + e] = make_double2(dr, di);
  }
}

}  // namespace ttable
