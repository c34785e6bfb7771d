// One Arnoldi step after the operator application, as ONE cooperative launch (small / medium problems):
//   CGS2 orthogonalisation (dots -> axpy -> dots -> axpy + norm), Givens update per window, normalisation of the new
//   basis vector - the phases of tm_vecops.cuh / tm_gmres.cuh separated by grid-wide barriers instead of kernel
//   boundaries.  On the 32x32 lattice the seven dependent launches cost more than their work (profiles/
//   r01_launches_cfg2_v3.md); here block c keeps chunk c for the whole step.  Used when all chunks are co-resident.
#pragma once
#include <cooperative_groups.h>

#include "tm_gmres.cuh"
#include "tm_vecops.cuh"

namespace cg = cooperative_groups;

template <typename R, int EPT>
__global__ void __launch_bounds__(TM_VT)
k_arnoldi_fused(const Cx<R>* __restrict__ V, size_t stride, int j, Cx<R>* __restrict__ W, const TmChunk* __restrict__ chunks,
                int n_chunks, double2* __restrict__ part, double* __restrict__ normpart,
                const int* __restrict__ win_chunk_ptr, TmGmresDev S, int n_win, double tol) {
  if (*S.n_active == 0) return;                       // grid-uniform: nothing below changes it before the Givens phase
  cg::grid_group grid = cg::this_grid();
  extern __shared__ double2 s_dyn[];                  // max(j+1 coefficients, Givens scratch)
  __shared__ Cx<R> s_w[EPT * TM_VT];
  __shared__ double s_n[TM_VT / 32];
  const int nvec = j + 1, c = blockIdx.x;
  const TmChunk ch = chunks[c];

  dots_body<R, EPT>(V, stride, nvec, W, ch, c, n_chunks, part, 0, 1, s_w);
  grid.sync();
  axpy_body<R, EPT>(V, stride, nvec, S.h1, S.ldh, -1.0, W, ch, c, nullptr, part, n_chunks, win_chunk_ptr, s_dyn, s_n);
  grid.sync();
  dots_body<R, EPT>(V, stride, nvec, W, ch, c, n_chunks, part, 0, 1, s_w);
  grid.sync();
  axpy_body<R, EPT>(V, stride, nvec, S.h2, S.ldh, -1.0, W, ch, c, normpart, part, n_chunks, win_chunk_ptr, s_dyn, s_n);
  grid.sync();
  if (threadIdx.x < 32)
    for (int w = c; w < n_win; w += gridDim.x) givens_body(S, w, j, tol, normpart, win_chunk_ptr, threadIdx.x, s_dyn);
  grid.sync();
  const double sc = S.inv_norm[ch.win];               // V_{j+1} = w / h_{j+1,j}  (0 for finished windows)
  Cx<R>* dst = const_cast<Cx<R>*>(V) + (size_t)(j + 1) * stride;
  for (int e = threadIdx.x; e < ch.count; e += TM_VT) {
    const size_t g = (size_t)ch.start + e;
    dst[g] = cx<R>((R)(sc * (double)W[g].re), (R)(sc * (double)W[g].im));
  }
}
