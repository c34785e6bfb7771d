// Vector-phase kernels: conversions, per-scatterer T application (Eq. I25), and the
// device-resident GMRES building blocks (reading R13).  All are HBM/L2-streaming kernels.
// Windows (independent problems batched on one GPU) are handled through a chunk table: every
// chunk of <= EPT * TM_VT consecutive vector elements lies inside exactly one window.
#pragma once
#include "tm_common.cuh"

#define TM_VT 256                // threads per block of the vector kernels
// A chunk holds EPT * TM_VT complex elements (EPT = elements per thread: 4 for large problems, 1 for small ones so
// that a 30 720-element vector still spreads over 120 blocks; chosen once per context).

struct TmChunk { int win; int start; int count; };
#ifdef TM_ARN_STAMPS                // debug build: fine time stamps (clock64) of thread 0 of block 0 inside the vector phases
__device__ unsigned long long g_fine[64];
__device__ int g_fine_base;
#define TM_FSTAMP(k) do { if (blockIdx.x == 0 && threadIdx.x == 0) g_fine[g_fine_base + (k)] = clock64(); } while (0)
#else
#define TM_FSTAMP(k) do { } while (0)
#endif   // element range [start, start+count) of window win

// ------------------------------------------------------------------------------------------------ conversions
template <typename R>
__global__ void k_from_c64(const double* __restrict__ in, Cx<R>* __restrict__ out, size_t n) {
  for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x)
    out[e] = cx<R>((R)in[2 * e], (R)in[2 * e + 1]);
}
template <typename R>
__global__ void k_to_c64(const Cx<R>* __restrict__ in, double* __restrict__ out, size_t n) {
  for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
    out[2 * e] = (double)in[e].re; out[2 * e + 1] = (double)in[e].im;
  }
}

// ------------------------------------------------------------------------------------------------ T application
// One block per JB scatterers.  mode:
//   0  y = x - T (sum_c u_c)          forward operator  (I - T A) x
//   1  y = x - P (sum_c u_c)          transposed operator, u = A (P T^T x)   (identity S3: A^T = P A P)
//   2  y = sum_c u_c                  bare A x
//   3  y = T x                        right-hand side b = T p  (u unused)
//   4  y = P T^T x                    pre-step of the transposed operator (u unused)
template <typename R, int JB>
__global__ void __launch_bounds__(256)
k_tapply(int mode, int L, int n_scat, int n_chunk, const Cx<R>* __restrict__ x, const Cx<R>* __restrict__ u_part,
         Cx<R>* __restrict__ y, const Cx<R>* __restrict__ T, int diag, const int* __restrict__ type_of,
         const TmConst* __restrict__ cst, const int* __restrict__ n_active) {
  if (n_active != nullptr && *n_active == 0) return;
  __shared__ Cx<R> s_v[JB * TM_MAX_MODES];
  const int j0 = blockIdx.x * JB;
  const int nj = min(JB, n_scat - j0);
  const int ne = nj * L;
  // stage the vector T (or P) acts on
  for (int e = threadIdx.x; e < ne; e += blockDim.x) {
    const size_t g = (size_t)j0 * L + e;
    Cx<R> v;
    if (mode <= 2) {
      v = u_part[g];
      for (int c = 1; c < n_chunk; ++c) v = cadd(v, u_part[(size_t)c * n_scat * L + g]);   // fixed order
    } else {
      v = x[g];
    }
    s_v[e] = v;
  }
  __syncthreads();
  for (int e = threadIdx.x; e < ne; e += blockDim.x) {
    const int jj = e / L, a = e - jj * L;
    const size_t g = (size_t)j0 * L + e;
    const Cx<R>* v = s_v + jj * L;
    Cx<R> out;
    if (mode == 2) out = v[a];
    else if (mode == 1) out = csub(x[g], v[cst->perm_neg_m[a]]);
    else {
      const int ty = type_of[j0 + jj];
      Cx<R> tv;
      if (mode == 4) {                      // (P T^T x)[a] = (T^T x)[perm a] = sum_b T[b][perm a] x[b]
        const int ap = cst->perm_neg_m[a];
        if (diag) tv = cmul(T[(size_t)ty * L + ap], v[ap]);
        else {
          tv = cx<R>(R(0), R(0));
          const Cx<R>* Tt = T + (size_t)ty * L * L;
          for (int b = 0; b < L; ++b) tv = cfma(Tt[(size_t)b * L + ap], v[b], tv);
        }
        out = tv;
      } else {
        if (diag) tv = cmul(T[(size_t)ty * L + a], v[a]);
        else {
          tv = cx<R>(R(0), R(0));
          const Cx<R>* Tr = T + ((size_t)ty * L + a) * L;
          for (int b = 0; b < L; ++b) tv = cfma(Tr[b], v[b], tv);
        }
        out = (mode == 0) ? csub(x[g], tv) : tv;
      }
    }
    y[g] = out;
  }
}

// ------------------------------------------------------------------------------------------------ GMRES pieces
// part[i * n_chunks + c] = sum_{e in chunk c} conj(V_i[e]) w[e],  i < nvec  (double accumulation).
// grid = (n_chunks, G): block (c, g) handles the basis vectors i = g, g + G, ...; inside the block the chunk of w is
// staged in shared memory and every WARP takes whole vectors (lanes stride over the chunk, one shuffle reduction per
// vector instead of one per vector and warp).
// VC (k_arnoldi_fused only): 0 = basis vectors from global memory; 1 = from global memory, and the chunk of every vector
// i < vcap is left in the block's shared-memory cache s_V[i][EPT * TM_VT]; 2 = vectors i < vcap from that cache.
// With a short chunk (EPT = 1) a warp has TWO vectors in flight (16 independent loads per lane): the pass is bound
// by the L2 latency, not by bandwidth.  Every sum keeps its order, so the results do not depend on VC or the pairing.
template <typename R, int EPT, int VC = 0>
__device__ __forceinline__ void dots_body(const Cx<R>* __restrict__ V, size_t stride, int nvec, const Cx<R>* __restrict__ w,
                                          const TmChunk ch, int cidx, int n_chunks, double2* __restrict__ part, int gy, int ngy,
                                          Cx<R>* s_w, Cx<R>* s_V = nullptr, int vcap = 0) {
  constexpr int CH = EPT * TM_VT, NK = CH / 32;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  TM_FSTAMP(0);
#pragma unroll
  for (int k = 0; k < EPT; ++k) {
    const int e = threadIdx.x + k * TM_VT;
    s_w[e] = e < ch.count ? w[(size_t)ch.start + e] : cx<R>(R(0), R(0));
  }
  __syncthreads();
  TM_FSTAMP(1);
  auto fetch = [&](int iv, int e) -> Cx<R> {
    if (VC == 2 && iv < vcap) return s_V[(size_t)iv * CH + e];
    const Cx<R> a = V[(size_t)iv * stride + ch.start + e];
    if (VC == 1 && iv < vcap) s_V[(size_t)iv * CH + e] = a;
    return a;
  };
  const int step = ngy * (TM_VT / 32);
  int i = gy + warp * ngy;
  if constexpr (NK <= 8) {
    for (; i + step < nvec; i += 2 * step) {
      Cx<R> a0[NK], a1[NK];
#pragma unroll
      for (int k = 0; k < NK; ++k) {
        const int e = lane + 32 * k;
        if (e < ch.count) { a0[k] = fetch(i, e); a1[k] = fetch(i + step, e); }
      }
      double sr = 0.0, si = 0.0, tr = 0.0, ti = 0.0;
#pragma unroll
      for (int k = 0; k < NK; ++k) {
        const int e = lane + 32 * k;
        if (e < ch.count) {
          const Cx<R> b = s_w[e];
          { const Cx<R> a = a0[k];
            sr += (double)a.re * (double)b.re + (double)a.im * (double)b.im;
            si += (double)a.re * (double)b.im - (double)a.im * (double)b.re; }
          { const Cx<R> a = a1[k];
            tr += (double)a.re * (double)b.re + (double)a.im * (double)b.im;
            ti += (double)a.re * (double)b.im - (double)a.im * (double)b.re; }
        }
      }
      sr = warp_sum(sr); si = warp_sum(si); tr = warp_sum(tr); ti = warp_sum(ti);
      if (lane == 0) {
        part[(size_t)i * n_chunks + cidx] = make_double2(sr, si);
        part[(size_t)(i + step) * n_chunks + cidx] = make_double2(tr, ti);
      }
    }
  }
  TM_FSTAMP(2);
  for (; i < nvec; i += step) {
    double sr = 0.0, si = 0.0;
#pragma unroll
    for (int k = 0; k < NK; ++k) {
      const int e = lane + 32 * k;
      if (e < ch.count) {
        const Cx<R> a = fetch(i, e), b = s_w[e];
        sr += (double)a.re * (double)b.re + (double)a.im * (double)b.im;
        si += (double)a.re * (double)b.im - (double)a.im * (double)b.re;
      }
    }
    sr = warp_sum(sr); si = warp_sum(si);
    if (lane == 0) part[(size_t)i * n_chunks + cidx] = make_double2(sr, si);
  }
  TM_FSTAMP(3);
}

template <typename R, int EPT>
__global__ void __launch_bounds__(TM_VT)
k_dots(const Cx<R>* __restrict__ V, size_t stride, int nvec, const Cx<R>* __restrict__ w,
       const TmChunk* __restrict__ chunks, int n_chunks, double2* __restrict__ part, const int* __restrict__ n_active) {
  if (n_active != nullptr && *n_active == 0) return;
  __shared__ Cx<R> s_w[EPT * TM_VT];
  dots_body<R, EPT>(V, stride, nvec, w, chunks[blockIdx.x], blockIdx.x, n_chunks, part, blockIdx.y, gridDim.y, s_w);
}

// h[win * ldh + i] (+)= sum over the window's chunks of part[i][c].  grid = (nvec, n_win), block = 64.
__global__ void k_reduce_h(const double2* __restrict__ part, int n_chunks, const int* __restrict__ win_chunk_ptr,
                           double2* __restrict__ h, int ldh, int accumulate, const int* __restrict__ n_active) {
  if (n_active != nullptr && *n_active == 0) return;
  const int i = blockIdx.x, w = blockIdx.y;
  double sr = 0.0, si = 0.0;
  for (int c = win_chunk_ptr[w] + threadIdx.x; c < win_chunk_ptr[w + 1]; c += blockDim.x) {
    const double2 p = part[(size_t)i * n_chunks + c];
    sr += p.x; si += p.y;
  }
  __shared__ double2 s[2];
  sr = warp_sum(sr); si = warp_sum(si);
  if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = make_double2(sr, si);
  __syncthreads();
  if (threadIdx.x == 0) {
    double2 r = make_double2(s[0].x + s[1].x, s[0].y + s[1].y);
    if (accumulate) { r.x += h[(size_t)w * ldh + i].x; r.y += h[(size_t)w * ldh + i].y; }
    h[(size_t)w * ldh + i] = r;
  }
}

// w += sign * sum_i coef_i V_i ;  optionally normpart[c] = sum |w|^2 over the chunk (after the update).
// The coefficients of window `win` are either given (coef[win * ldc + i]) or, when `part` != nullptr, reduced here from
// the per-chunk partial dot products of k_dots (coef_i = sum over the window's chunks of part[i][c], fixed order ->
// deterministic); the block owning the window's first chunk then also stores them to coef for the Givens kernel.
// Basis vectors must hold finite numbers (the workspace is zeroed at the start of a solve): a zero coefficient
// multiplies whatever is there.
// (R: precision of the basis vectors, RW: precision of the updated vector - they differ in mixed-precision solves)
// (VC = 2: the chunks of the basis vectors i < vcap come from the shared-memory cache s_V, see dots_body)
template <typename R, int EPT, typename RW = R, int VC = 0>
__device__ __forceinline__ void axpy_body(const Cx<R>* __restrict__ V, size_t stride, int nvec, double2* __restrict__ coef, int ldc,
                                          double sign, Cx<RW>* __restrict__ w, const TmChunk ch, int cidx,
                                          double* __restrict__ normpart, const double2* __restrict__ part, int n_chunks,
                                          const int* __restrict__ win_chunk_ptr, double2* s_c, double* s_n,
                                          const Cx<R>* s_V = nullptr, int vcap = 0) {
  TM_FSTAMP(0);
  if (part != nullptr) {
    const int c0 = win_chunk_ptr[ch.win], c1 = win_chunk_ptr[ch.win + 1];
    // 4 lanes per vector, each sums a contiguous quarter of the chunk list; lanes combined in fixed order
    for (int base = 0; base < nvec; base += TM_VT / 4) {
      const int i = base + (threadIdx.x >> 2), q = threadIdx.x & 3;
      double sr = 0.0, si = 0.0;
      if (i < nvec) {
        const int len = (c1 - c0 + 3) / 4;
        const int lo = c0 + q * len, hi = min(c1, lo + len);
        const double2* p = part + (size_t)i * n_chunks;
        // 16 loads in flight, then the additions in list order (the pass is latency-bound: L2 round trips, not bytes)
        for (int c = lo; c < hi; c += 16) {
          double2 t[16];
#pragma unroll
          for (int u = 0; u < 16; ++u) if (c + u < hi) t[u] = p[c + u];
#pragma unroll
          for (int u = 0; u < 16; ++u) if (c + u < hi) { sr += t[u].x; si += t[u].y; }
        }
      }
      sr += __shfl_xor_sync(0xffffffffu, sr, 1); si += __shfl_xor_sync(0xffffffffu, si, 1);
      sr += __shfl_xor_sync(0xffffffffu, sr, 2); si += __shfl_xor_sync(0xffffffffu, si, 2);
      if (i < nvec && q == 0) {
        s_c[i] = make_double2(sign * sr, sign * si);
        if (cidx == c0) coef[(size_t)ch.win * ldc + i] = make_double2(sr, si);
      }
    }
  } else {
    for (int i = threadIdx.x; i < nvec; i += TM_VT) {
      const double2 c = coef[(size_t)ch.win * ldc + i];
      s_c[i] = make_double2(sign * c.x, sign * c.y);
    }
  }
  TM_FSTAMP(1);
  __syncthreads();
  TM_FSTAMP(2);
  double nrm = 0.0;
#pragma unroll
  for (int k = 0; k < EPT; ++k) {
    const int e = threadIdx.x + k * TM_VT;
    if (e < ch.count) {
      const size_t g = (size_t)ch.start + e;
      double ar = (double)w[g].re, ai = (double)w[g].im;
      int i = 0;
      if (VC == 2) {
        const int nc_ = min(nvec, vcap);
#pragma unroll 8
        for (; i < nc_; ++i) {
          const double2 c = s_c[i];
          const Cx<R> v = s_V[(size_t)i * (EPT * TM_VT) + e];
          ar += c.x * (double)v.re - c.y * (double)v.im;
          ai += c.x * (double)v.im + c.y * (double)v.re;
        }
      }
#pragma unroll (EPT == 1 ? 16 : 8)
      for (; i < nvec; ++i) {
        const double2 c = s_c[i];
        const Cx<R> v = V[(size_t)i * stride + g];
        ar += c.x * (double)v.re - c.y * (double)v.im;
        ai += c.x * (double)v.im + c.y * (double)v.re;
      }
      w[g] = cx<RW>((RW)ar, (RW)ai);
      nrm += ar * ar + ai * ai;
    }
  }
  TM_FSTAMP(3);
  if (normpart != nullptr) {
    nrm = warp_sum(nrm);
    if ((threadIdx.x & 31) == 0) s_n[threadIdx.x >> 5] = nrm;
    __syncthreads();
    if (threadIdx.x == 0) {
      double t = 0.0;
#pragma unroll
      for (int k = 0; k < TM_VT / 32; ++k) t += s_n[k];
      normpart[cidx] = t;
    }
  }
}

template <typename R, int EPT, typename RW = R>
__global__ void __launch_bounds__(TM_VT)
k_axpy(const Cx<R>* __restrict__ V, size_t stride, int nvec, double2* __restrict__ coef, int ldc, double sign,
       Cx<RW>* __restrict__ w, const TmChunk* __restrict__ chunks, double* __restrict__ normpart,
       const double2* __restrict__ part, int n_chunks, const int* __restrict__ win_chunk_ptr,
       const int* __restrict__ n_active) {
  if (n_active != nullptr && *n_active == 0) return;
  extern __shared__ double2 s_c[];                   // [nvec]
  __shared__ double s_n[TM_VT / 32];
  axpy_body<R, EPT, RW>(V, stride, nvec, coef, ldc, sign, w, chunks[blockIdx.x], blockIdx.x, normpart, part, n_chunks,
                        win_chunk_ptr, s_c, s_n);
}

// normpart[c] = sum |v|^2 over chunk c
template <typename R>
__global__ void __launch_bounds__(TM_VT)
k_norm2(const Cx<R>* __restrict__ v, const TmChunk* __restrict__ chunks, double* __restrict__ normpart) {
  const TmChunk ch = chunks[blockIdx.x];
  double nrm = 0.0;
  for (int e = threadIdx.x; e < ch.count; e += TM_VT) {
    const Cx<R> a = v[(size_t)ch.start + e];
    nrm += (double)a.re * (double)a.re + (double)a.im * (double)a.im;
  }
  __shared__ double s_n[TM_VT / 32];
  nrm = warp_sum(nrm);
  if ((threadIdx.x & 31) == 0) s_n[threadIdx.x >> 5] = nrm;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
#pragma unroll
    for (int k = 0; k < TM_VT / 32; ++k) t += s_n[k];
    normpart[blockIdx.x] = t;
  }
}

// out[win] = sqrt(sum of the window's normpart).  One block (64 threads) per window.
__global__ void k_reduce_norm(const double* __restrict__ normpart, const int* __restrict__ win_chunk_ptr,
                              double* __restrict__ out) {
  const int w = blockIdx.x;
  double s = 0.0;
  for (int c = win_chunk_ptr[w] + threadIdx.x; c < win_chunk_ptr[w + 1]; c += blockDim.x) s += normpart[c];
  __shared__ double sh[2];
  s = warp_sum(s);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) out[w] = sqrt(sh[0] + sh[1]);
}

// dst = a * scale[win]  (V_{j+1} = w / h_{j+1,j});  dst = a - b when b != nullptr (scale ignored).
// R: precision of a and b, RD: precision of dst (mixed-precision solves normalise an fp64 residual into an fp32 basis).
template <typename R, typename RD = R>
__global__ void __launch_bounds__(TM_VT)
k_scale_or_sub(const Cx<R>* __restrict__ a, const Cx<R>* __restrict__ b, const double* __restrict__ scale,
               Cx<RD>* __restrict__ dst, const TmChunk* __restrict__ chunks, const int* __restrict__ n_active) {
  if (n_active != nullptr && *n_active == 0) return;
  const TmChunk ch = chunks[blockIdx.x];
  const double sc = (b == nullptr) ? scale[ch.win] : 1.0;
  for (int e = threadIdx.x; e < ch.count; e += TM_VT) {
    const size_t g = (size_t)ch.start + e;
    if (b == nullptr) dst[g] = cx<RD>((RD)(sc * (double)a[g].re), (RD)(sc * (double)a[g].im));
    else dst[g] = cx<RD>((RD)((double)a[g].re - (double)b[g].re), (RD)((double)a[g].im - (double)b[g].im));
  }
}

// ------------------------------------------------------------------------------------------------ sensitivities
// out[j] = lambda_j^T dT_{type(j)} (p_j + (A s)_j)   (Eq. IV8 with Omega = T^{-1}(I - T A)).
// One warp per scatterer; `as` holds A s.
template <typename R>
__global__ void __launch_bounds__(128)
k_grad_tmatrix(int L, int n_scat, const Cx<R>* __restrict__ as, const double2* __restrict__ p, const Cx<R>* __restrict__ lam,
               const Cx<R>* __restrict__ dT, int diag, const int* __restrict__ type_of, double2* __restrict__ out) {
  const int j = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (j >= n_scat) return;
  const int ty = type_of[j];
  double sr = 0.0, si = 0.0;
  for (int a = lane; a < L; a += 32) {
    double rr, ri;                                     // (dT q)_a,  q = p + A s
    if (diag) {
      const Cx<R> d = dT[(size_t)ty * L + a];
      const double qr = p[(size_t)j * L + a].x + (double)as[(size_t)j * L + a].re, qi = p[(size_t)j * L + a].y + (double)as[(size_t)j * L + a].im;
      rr = (double)d.re * qr - (double)d.im * qi; ri = (double)d.re * qi + (double)d.im * qr;
    } else {
      rr = 0.0; ri = 0.0;
      const Cx<R>* row = dT + ((size_t)ty * L + a) * L;
      for (int b = 0; b < L; ++b) {
        const double qr = p[(size_t)j * L + b].x + (double)as[(size_t)j * L + b].re, qi = p[(size_t)j * L + b].y + (double)as[(size_t)j * L + b].im;
        rr += (double)row[b].re * qr - (double)row[b].im * qi; ri += (double)row[b].re * qi + (double)row[b].im * qr;
      }
    }
    const Cx<R> l = lam[(size_t)j * L + a];
    sr += (double)l.re * rr - (double)l.im * ri;
    si += (double)l.re * ri + (double)l.im * rr;
  }
  sr = warp_sum(sr); si = warp_sum(si);
  if (lane == 0) out[j] = make_double2(sr, si);
}

// acc = (init ? 0 : acc) + c * y
template <typename R>
__global__ void k_acc_scaled(Cx<R>* __restrict__ acc, const Cx<R>* __restrict__ y, double c, size_t n, int init) {
  for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
    const double ar = init ? 0.0 : (double)acc[e].re, ai = init ? 0.0 : (double)acc[e].im;
    acc[e] = cx<R>((R)(ar + c * (double)y[e].re), (R)(ai + c * (double)y[e].im));
  }
}

// out[j * out_stride] += sum_a left_j[perm a] * D_j[a]   (bilinear, no conjugation; P = the m -> -m permutation).
// D_j starts at D + j * d_stride.  One warp per scatterer.
template <typename R, typename RD>
__global__ void __launch_bounds__(128)
k_bilinear_rows(int L, int n_scat, const Cx<R>* __restrict__ left, const Cx<RD>* __restrict__ D, size_t d_stride,
                const TmConst* __restrict__ cst, double2* __restrict__ out, int out_stride) {
  const int j = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (j >= n_scat) return;
  double sr = 0.0, si = 0.0;
  for (int a = lane; a < L; a += 32) {
    const Cx<R> l = left[(size_t)j * L + cst->perm_neg_m[a]];
    const Cx<RD> d = D[(size_t)j * d_stride + a];
    sr += (double)l.re * (double)d.re - (double)l.im * (double)d.im;
    si += (double)l.re * (double)d.im + (double)l.im * (double)d.re;
  }
  sr = warp_sum(sr); si = warp_sum(si);
  if (lane == 0) { out[(size_t)j * out_stride].x += sr; out[(size_t)j * out_stride].y += si; }
}

// ------------------------------------------------------------------------------------------------ analytic position gradient
// dA/dd_alpha = k D^alpha A^ext (gen_tables.py: gradient_entries).  k_pad_modes embeds a coefficient
// vector of truncation lmax into the mode order of lmax + 1 (zeros for l = lmax + 1; xp is cleared by the caller);
// k_grad_contract adds  out[j][alpha] += k * sum_e left_j[perm(row_e)] D_e v_j[col_e]  (alpha = alpha_e), v = A^ext (padded x).
struct TmGradDev { int n; const uint8_t* alpha; const uint8_t* row; const uint8_t* col; const double* re; const double* im; };

template <typename R>
__global__ void k_pad_modes(const Cx<R>* __restrict__ x, Cx<R>* __restrict__ xp, int L, int Le, size_t n) {
  const size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (e >= n) return;
  const size_t j = e / L;
  const int a = (int)(e - j * L);
  const int ae = a < L / 2 ? a : a - L / 2 + Le / 2;            // flat index p * (L/2) + l (l + 1) - 1 + m (reading R1)
  xp[j * Le + ae] = x[e];
}

template <typename R>
__global__ void __launch_bounds__(128)
k_grad_contract(int L, int Le, int n_scat, const Cx<R>* __restrict__ left, const Cx<R>* __restrict__ v,
                const TmConst* __restrict__ cst, TmGradDev tab, double k, double2* __restrict__ out) {
  const int j = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (j >= n_scat) return;
  double sr[3] = {0.0, 0.0, 0.0}, si[3] = {0.0, 0.0, 0.0};
  for (int e = lane; e < tab.n; e += 32) {
    const Cx<R> l = left[(size_t)j * L + cst->perm_neg_m[tab.row[e]]];
    const Cx<R> w = v[(size_t)j * Le + tab.col[e]];
    const double dr = tab.re[e], di = tab.im[e];
    const double tr = dr * (double)w.re - di * (double)w.im, ti = dr * (double)w.im + di * (double)w.re;      // D_e v
    const double pr = (double)l.re * tr - (double)l.im * ti, pi = (double)l.re * ti + (double)l.im * tr;
    const int a = tab.alpha[e];
#pragma unroll
    for (int q = 0; q < 3; ++q) if (a == q) { sr[q] += pr; si[q] += pi; }
  }
#pragma unroll
  for (int q = 0; q < 3; ++q) {
    const double a = warp_sum(sr[q]), b = warp_sum(si[q]);
    if (lane == 0) { out[(size_t)j * 3 + q].x += k * a; out[(size_t)j * 3 + q].y += k * b; }
  }
}
