// One Arnoldi step after the operator application, as ONE cooperative launch (small / medium problems):
//   CGS2 orthogonalisation (dots -> axpy -> dots -> axpy + norm), Givens update per window, normalisation of the new
//   basis vector - the phases of tm_vecops.cuh / tm_gmres.cuh separated by grid-wide barriers instead of kernel
//   boundaries; for diagonal T the T application (and the transposed operator's permutations) is folded in too.  On the 32x32 lattice the seven dependent launches cost more than their work (profiles/
//   r01_recorded_runs.md, kernel history); here block c keeps chunk c for the whole step.  Used when all chunks are co-resident.
#pragma once
#include <cooperative_groups.h>

#include "tm_gmres.cuh"
#include "tm_vecops.cuh"

namespace cg = cooperative_groups;

// Optional fusion of the T application around the all-pairs product (diagonal T only):
//   mode 1 (forward):    w = x - T (sum_c u_c)                                     (Eq. I25)
//   mode 2 (transposed): w = x - P (sum_c u_c), and z_next = P T^T v_{j+1} for the next all-pairs product (identity S3)
template <typename R> struct TmFuseT {
  int mode;                     // 0: w was produced by k_tapply
  const Cx<R>* x;               // v_j
  const Cx<R>* u_part; int n_part; size_t n;
  const Cx<R>* T; const int* type_of; const int* perm; int L;
  Cx<R>* z_next;
};

#ifdef TM_ARN_STAMPS                // debug build: phase time stamps of block 0 of the last launch (clock64 of its SM, globaltimer)
__device__ unsigned long long g_arn_stamps[32];
#define TM_STAMP(k) do { if (blockIdx.x == 0 && threadIdx.x == 0) { g_arn_stamps[k] = clock64(); unsigned long long gt_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt_)); g_arn_stamps[16 + (k)] = gt_; } } while (0)
#define TM_FBASE(b) do { if (blockIdx.x == 0 && threadIdx.x == 0) g_fine_base = (b); } while (0)
#else
#define TM_STAMP(k) do { } while (0)
#define TM_FBASE(b) do { } while (0)
#endif

template <typename R, int EPT>
__global__ void __launch_bounds__(TM_VT, 2)          // 2 blocks per SM: problems of up to 296 chunks stay on this path
k_arnoldi_fused(const Cx<R>* __restrict__ V, size_t stride, int j, Cx<R>* __restrict__ W, const TmChunk* __restrict__ chunks,
                int n_chunks, double2* __restrict__ part, double* __restrict__ normpart,
                const int* __restrict__ win_chunk_ptr, TmGmresDev S, int n_win, double tol, TmFuseT<R> ft, int vcap, int voff, int do_givens) {
  if (*S.n_active == 0) return;                       // grid-uniform: nothing below changes it before the Givens phase
#ifdef TM_ARN_STAMPS
  if (blockIdx.x == 0 && threadIdx.x == 0) { g_arn_stamps[15] = g_arn_stamps[16 + 9]; g_arn_stamps[14] = (unsigned long long)j; }
#endif
  TM_STAMP(0);
  cg::grid_group grid = cg::this_grid();
  extern __shared__ double2 s_dyn[];                  // max(j+1 coefficients, Givens scratch), then the basis-vector cache
  // The block's chunk of the basis vectors i < vcap stays in shared memory for the whole step (voff: byte offset of
  // the cache in s_dyn): the first projection reads them from L2 once, the two updates and the second projection read
  // the cache - three of the four passes over V[0..j] no longer wait for L2.  Same values, same order of operations.
  Cx<R>* s_V = reinterpret_cast<Cx<R>*>(reinterpret_cast<char*>(s_dyn) + voff);
  __shared__ Cx<R> s_w[EPT * TM_VT];
  __shared__ double s_n[TM_VT / 32];
  const int nvec = j + 1, c = blockIdx.x;
  const TmChunk ch = chunks[c];

  if (ft.mode != 0) {                                 // the block produces its own chunk of w, then only reads that chunk
    for (int e = threadIdx.x; e < ch.count; e += TM_VT) {
      const size_t g = (size_t)ch.start + e;
      const int sj = (int)(g / ft.L), a = (int)(g - (size_t)sj * ft.L);
      const size_t gu = ft.mode == 2 ? (size_t)sj * ft.L + ft.perm[a] : g;
      Cx<R> u = ft.u_part[gu];
      int k = 1;
      for (; k + 8 <= ft.n_part; k += 8) {            // 8 loads in flight, added in fixed order
        Cx<R> t[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) t[q] = ft.u_part[(size_t)(k + q) * ft.n + gu];
#pragma unroll
        for (int q = 0; q < 8; ++q) u = cadd(u, t[q]);
      }
      for (; k < ft.n_part; ++k) u = cadd(u, ft.u_part[(size_t)k * ft.n + gu]);
      W[g] = ft.mode == 1 ? csub(ft.x[g], cmul(ft.T[(size_t)ft.type_of[sj] * ft.L + a], u)) : csub(ft.x[g], u);
    }
    __syncthreads();
  }
  TM_STAMP(1);
  // CGS2 with three grid barriers: the second projection of a chunk needs only that chunk of w after the first update, so
  // it follows the update without a barrier; its partial sums go to a second buffer because slower blocks may still be
  // reducing the first one.
  double2* part2 = part + (size_t)S.ldh * n_chunks;
  TM_FBASE(0);
  dots_body<R, EPT, 1>(V, stride, nvec, W, ch, c, n_chunks, part, 0, 1, s_w, s_V, vcap);
  TM_STAMP(2);
  grid.sync();
  TM_STAMP(3);
  TM_FBASE(8);
  axpy_body<R, EPT, R, 2>(V, stride, nvec, S.h1, S.ldh, -1.0, W, ch, c, nullptr, part, n_chunks, win_chunk_ptr, s_dyn, s_n, s_V, vcap);
  __syncthreads();
  TM_STAMP(4);
  TM_FBASE(16);
  dots_body<R, EPT, 2>(V, stride, nvec, W, ch, c, n_chunks, part2, 0, 1, s_w, s_V, vcap);
  TM_STAMP(5);
  grid.sync();
  TM_STAMP(6);
  TM_FBASE(24);
  axpy_body<R, EPT, R, 2>(V, stride, nvec, S.h2, S.ldh, -1.0, W, ch, c, normpart, part2, n_chunks, win_chunk_ptr, s_dyn, s_n, s_V, vcap);
  TM_STAMP(7);
  grid.sync();
  TM_STAMP(8);
  // Givens update (one warp per window) runs alongside the normalisation: every block recomputes its window's norm
  // from the chunk norms (same fixed order as the Givens warp), so no further barrier is needed.  A window that
  // finishes in this step keeps iterating harmlessly: its later columns are ignored (kcols is frozen, y is zero there).
  if (do_givens && threadIdx.x < 32)
    for (int w = c; w < n_win; w += gridDim.x) givens_body(S, w, j, tol, normpart, win_chunk_ptr, threadIdx.x, s_dyn);
  double nn = 0.0;
  if (threadIdx.x >= 32 && threadIdx.x < 64) {
    const int lane = threadIdx.x - 32;
    for (int k = win_chunk_ptr[ch.win] + lane; k < win_chunk_ptr[ch.win + 1]; k += 32) nn += normpart[k];
    nn = warp_sum(nn);
    if (lane == 0) s_n[0] = nn;
  }
  __syncthreads();
  const double hn = sqrt(s_n[0]);
  const double sc = hn > 0.0 ? 1.0 / hn : 0.0;        // V_{j+1} = w / h_{j+1,j}
  Cx<R>* dst = const_cast<Cx<R>*>(V) + (size_t)(j + 1) * stride;
  for (int e = threadIdx.x; e < ch.count; e += TM_VT) {
    const size_t g = (size_t)ch.start + e;
    dst[g] = cx<R>((R)(sc * (double)W[g].re), (R)(sc * (double)W[g].im));
    if (ft.mode == 2) {                               // z_next[a] = T[perm a] * v_{j+1}[perm a]
      const int sj = (int)(g / ft.L), a = (int)(g - (size_t)sj * ft.L), ap = ft.perm[a];
      const Cx<R> wv = W[(size_t)sj * ft.L + ap];
      const Cx<R> v = cx<R>((R)(sc * (double)wv.re), (R)(sc * (double)wv.im));
      ft.z_next[g] = cmul(ft.T[(size_t)ft.type_of[sj] * ft.L + ap], v);
    }
  }
#ifdef TM_ARN_STAMPS
  __syncthreads();
  TM_STAMP(9);
#endif
}
