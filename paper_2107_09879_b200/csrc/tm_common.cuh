// Shared device/host helpers of libtm (B200, sm_100a).  Product code: never includes anything from oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>

#define TM_MAX_LMAX 6                                      // largest truncation of the public API (the paper's)
#define TM_INT_LMAX 7                                      // internal: the position gradient at lmax runs one all-pairs product at lmax + 1
#define TM_MAX_NQ (2 * TM_INT_LMAX + 1)
#define TM_MAX_MODES (2 * TM_INT_LMAX * (TM_INT_LMAX + 2))  // 126

template <typename R> struct Cx;                       // interleaved complex of the compute precision
template <> struct __align__(16) Cx<double> { double re, im; };
template <> struct __align__(8) Cx<float> { float re, im; };

template <typename R> __host__ __device__ __forceinline__ Cx<R> cx(R a, R b) { Cx<R> z; z.re = a; z.im = b; return z; }
template <typename R> __device__ __forceinline__ Cx<R> cmul(Cx<R> a, Cx<R> b) {
  return cx<R>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
template <typename R> __device__ __forceinline__ Cx<R> cfma(Cx<R> a, Cx<R> b, Cx<R> c) {   // a*b + c
  c.re = fma(a.re, b.re, c.re); c.re = fma(-a.im, b.im, c.re);
  c.im = fma(a.re, b.im, c.im); c.im = fma(a.im, b.re, c.im);
  return c;
}
template <typename R> __device__ __forceinline__ Cx<R> cadd(Cx<R> a, Cx<R> b) { return cx<R>(a.re + b.re, a.im + b.im); }
template <typename R> __device__ __forceinline__ Cx<R> csub(Cx<R> a, Cx<R> b) { return cx<R>(a.re - b.re, a.im - b.im); }
template <typename R> __device__ __forceinline__ Cx<R> cconj(Cx<R> a) { return cx<R>(a.re, -a.im); }
// multiply by i^k, k = 0..3
template <typename R> __device__ __forceinline__ Cx<R> cmul_ipow(Cx<R> a, int k) {
  switch (k & 3) {
    case 0: return a;
    case 1: return cx<R>(-a.im, a.re);
    case 2: return cx<R>(-a.re, -a.im);
    default: return cx<R>(a.im, -a.re);
  }
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Work item of the all-pairs kernels: a tile of consecutive targets inside one window.
struct TmTile { int tgt_start, tgt_count, src_start, src_count; };

// Optional rigid displacement of all TARGETS against the sources (A/B experiments on the displacement argument of the
// translation operator).  With a non-zero shift the self pair no longer has r = 0 and is excluded by index instead.
struct TmShift { double x, y, z; int on; };

// Term table of the table-driven kernel on the device: for destination row b, terms row_ptr[b] <= t < row_ptr[b+1] with
// source column col[t], scalar-wave index widx[t] = q^2 + q + mu and coefficient coef[t] (real part if !imag[t]).
struct TmTermsDev { const int* row_ptr; const uint8_t* col; const uint8_t* widx; const uint8_t* imag; const double* coef; };

// Small per-lmax tables, one device copy per context (tm_ctx::d_const).
struct TmConst {
  int perm_neg_m[TM_MAX_MODES];          // flat index of (l,-m,p)               (structural identity S3)
  int mode_l[TM_MAX_MODES], mode_m[TM_MAX_MODES], mode_p[TM_MAX_MODES];
  double leg_a[TM_MAX_NQ + 1][TM_MAX_NQ + 1];   // normalised Legendre recurrence Pbar_q^mu = a (ct Pbar_{q-1}^mu - b Pbar_{q-2}^mu)
  double leg_b[TM_MAX_NQ + 1][TM_MAX_NQ + 1];
  double leg_d[TM_MAX_NQ + 1];                  // Pbar_mu^mu = d[mu] * sin(theta) * Pbar_{mu-1}^{mu-1}
};
