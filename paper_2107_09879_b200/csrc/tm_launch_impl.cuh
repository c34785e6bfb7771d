// Definitions of the launch functions of tm_launch.h, one section per kernel family (selected by the TM_SEC_* / TM_RANGE_*
// macros of the including translation unit).
#pragma once
#include "tm_launch.h"
#include "tm_allpairs.cuh"

#ifdef TM_SEC_COP
// cluster launch of the coplanar kernel: CL blocks along the chunk dimension reduce their partials through distributed shared memory
template <typename R, int LM, int CL>
cudaError_t launch_coplanar_cluster(const TmLaunch& a, dim3 grid, const Cx<R>* x, Cx<R>* up, TmShift shift) {
  constexpr int L = 2 * LM * (LM + 2);
  const size_t sm = sizeof(Cx<R>) * (size_t)128 * L;  // staging rows [128 targets][L]
  auto kern = k_allpairs_coplanar<R, LM, 128, TM_COP_SS, CL>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = dim3(128); cfg.dynamicSmemBytes = sm; cfg.stream = a.stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = 1; at[0].val.clusterDim.y = CL; at[0].val.clusterDim.z = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, a.pos, x, up, a.tiles, a.n_scat, a.k_over_pi, a.inv_k, a.n_active, shift);
}

template <typename R> cudaError_t tm_launch_coplanar(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, int tj, int cl, TmShift shift) {
  dim3 grid = a.grid;
  grid.z = 2;                                         // mirror-parity half: slowest grid dimension
  if (cl > 1 && tj == 128 && grid.y % cl == 0) {
    cudaError_t e;
    if (cl == 4) e = a.lmax == 1 ? launch_coplanar_cluster<R, 1, 4>(a, grid, x, up, shift)
                   : (a.lmax == 2 ? launch_coplanar_cluster<R, 2, 4>(a, grid, x, up, shift) : launch_coplanar_cluster<R, 3, 4>(a, grid, x, up, shift));
    else e = a.lmax == 1 ? launch_coplanar_cluster<R, 1, 2>(a, grid, x, up, shift)
             : (a.lmax == 2 ? launch_coplanar_cluster<R, 2, 2>(a, grid, x, up, shift) : launch_coplanar_cluster<R, 3, 2>(a, grid, x, up, shift));
    return e != cudaSuccess ? e : cudaGetLastError();
  }
#define TM_LAUNCH_COP2(LM, TJ)                                                                              \
  k_allpairs_coplanar<R, LM, TJ, TM_COP_SS><<<grid, TJ, 0, a.stream>>>(a.pos, x, up, a.tiles, a.n_scat,     \
                                                                       a.k_over_pi, a.inv_k, a.n_active, shift)
#define TM_LAUNCH_COP(LM)                                                                                   \
  do { if (tj == 256) TM_LAUNCH_COP2(LM, 256); else TM_LAUNCH_COP2(LM, 128); } while (0)
  switch (a.lmax) {
    case 1: TM_LAUNCH_COP(1); break;
    case 2: TM_LAUNCH_COP(2); break;
    default: TM_LAUNCH_COP(3); break;
  }
#undef TM_LAUNCH_COP
#undef TM_LAUNCH_COP2
  return cudaGetLastError();
}
template cudaError_t tm_launch_coplanar<double>(const TmLaunch&, const Cx<double>*, Cx<double>*, int, int, TmShift);
template cudaError_t tm_launch_coplanar<float>(const TmLaunch&, const Cx<float>*, Cx<float>*, int, int, TmShift);
#endif

#ifdef TM_SEC_COP4
#define TM_LAUNCH_C4(LM, TJ_)                                                                                   \
  {                                                                                                             \
    const size_t sm = Cop4Smem<R, LM, TJ_, TM_COP4_SS>::bytes;                                                  \
    cudaFuncSetAttribute(k_allpairs_coplanar4<R, LM, TJ_, TM_COP4_SS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm); \
    k_allpairs_coplanar4<R, LM, TJ_, TM_COP4_SS><<<grid, TJ_, sm, a.stream>>>(a.pos, x, up, a.tiles, a.n_scat,  \
                                                                              a.k_over_pi, a.inv_k, a.n_active, shift); \
  }
#ifdef TM_RANGE_LO
template <typename R> cudaError_t tm_launch_coplanar4_lo(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, TmShift shift) {
  dim3 grid = a.grid;
  grid.z = 4 * (a.lmax == 4 ? Cop4Max<4>::ng : Cop4Max<5>::ng);   // (z-mirror parity, y'-mirror sector) x row group: slowest grid dimension
  if (a.lmax == 4) TM_LAUNCH_C4(4, 128) else TM_LAUNCH_C4(5, 128)
  return cudaGetLastError();
}
template cudaError_t tm_launch_coplanar4_lo<double>(const TmLaunch&, const Cx<double>*, Cx<double>*, TmShift);
template cudaError_t tm_launch_coplanar4_lo<float>(const TmLaunch&, const Cx<float>*, Cx<float>*, TmShift);
int tm_cop4_groups(int lmax) {
  return lmax == 4 ? Cop4Max<4>::ng : (lmax == 5 ? Cop4Max<5>::ng : (lmax == 6 ? Cop4Max<6>::ng : Cop4Max<7>::ng));
}
#endif
#ifdef TM_RANGE_HI
template <typename R> cudaError_t tm_launch_coplanar4_hi(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, TmShift shift) {
  dim3 grid = a.grid;
  grid.z = 4 * (a.lmax == 6 ? Cop4Max<6>::ng : Cop4Max<7>::ng);
  if (a.lmax == 6) TM_LAUNCH_C4(6, 256) else TM_LAUNCH_C4(7, 128)
  return cudaGetLastError();
}
template cudaError_t tm_launch_coplanar4_hi<double>(const TmLaunch&, const Cx<double>*, Cx<double>*, TmShift);
template cudaError_t tm_launch_coplanar4_hi<float>(const TmLaunch&, const Cx<float>*, Cx<float>*, TmShift);
#endif
#undef TM_LAUNCH_C4
#endif

#ifdef TM_SEC_SYM3D
template <typename R> cudaError_t tm_launch_sym3d(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, TmShift shift) {
  dim3 grid = a.grid;
  grid.z = 2;                                         // y'-mirror sector: slowest grid dimension
#define TM_LAUNCH_S3(LM)                                                                                        \
  {                                                                                                             \
    const size_t sm = Sym3dSmem<R, LM, TM_SYM3D_TJ, TM_SYM3D_SS>::bytes;                                        \
    cudaFuncSetAttribute(k_allpairs_sym3d<R, LM, TM_SYM3D_TJ, TM_SYM3D_SS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm); \
    k_allpairs_sym3d<R, LM, TM_SYM3D_TJ, TM_SYM3D_SS><<<grid, TM_SYM3D_TJ, sm, a.stream>>>(a.pos, x, up, a.tiles, a.n_scat, \
                                                                                           a.k_over_pi, a.inv_k, a.n_active, shift); \
  }
  switch (a.lmax) {
    case 1: TM_LAUNCH_S3(1) break;
    case 2: TM_LAUNCH_S3(2) break;
    default: TM_LAUNCH_S3(3) break;
  }
#undef TM_LAUNCH_S3
  return cudaGetLastError();
}
template cudaError_t tm_launch_sym3d<double>(const TmLaunch&, const Cx<double>*, Cx<double>*, TmShift);
template cudaError_t tm_launch_sym3d<float>(const TmLaunch&, const Cx<float>*, Cx<float>*, TmShift);
void tm_cost_sym3d(int lmax, double* inst, double* flop) {
  const int I[4] = {0, TM_G3D_FPINST_L1, TM_G3D_FPINST_L2, TM_G3D_FPINST_L3};
  const int F[4] = {0, TM_G3D_FLOP_L1, TM_G3D_FLOP_L2, TM_G3D_FLOP_L3};
  *inst = I[lmax]; *flop = F[lmax];
}
#endif

#ifdef TM_SEC_ROT3D
#define TM_LAUNCH_R3(LM, TJ_, SS_)                                                                              \
  {                                                                                                             \
    constexpr int PG_ = tm_rot3d_pg_level(LM);                                                                  \
    const size_t sm = Rot3dSmem<R, LM, TJ_, SS_, PG_>::bytes;                                                   \
    cudaFuncSetAttribute(k_allpairs_rot3d<R, LM, TJ_, SS_, PG_>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm); \
    k_allpairs_rot3d<R, LM, TJ_, SS_, PG_><<<grid, TJ_, sm, a.stream>>>(a.pos, x, up, a.tiles, a.n_scat,        \
                                                                        a.k_over_pi, a.inv_k, a.n_active, pacc); \
  }
#ifdef TM_RANGE_LO
template <typename R> cudaError_t tm_launch_rot3d_lo(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, R* pacc) {
  dim3 grid = a.grid;
  grid.z = 2;                                         // y'-mirror sector: slowest grid dimension
  switch (a.lmax) {
    case 1: TM_LAUNCH_R3(1, 128, 16) break;
    case 2: TM_LAUNCH_R3(2, 128, 16) break;
    case 3: TM_LAUNCH_R3(3, 128, 16) break;
    case 4: TM_LAUNCH_R3(4, 64, 4) break;
    default: TM_LAUNCH_R3(5, 64, 4) break;
  }
  return cudaGetLastError();
}
template cudaError_t tm_launch_rot3d_lo<double>(const TmLaunch&, const Cx<double>*, Cx<double>*, double*);
template cudaError_t tm_launch_rot3d_lo<float>(const TmLaunch&, const Cx<float>*, Cx<float>*, float*);
void tm_cost_rot3d(int lmax, double* inst, double* flop) {
  const int I[8] = {0, TM_R3D_FPINST_L1, TM_R3D_FPINST_L2, TM_R3D_FPINST_L3, TM_R3D_FPINST_L4, TM_R3D_FPINST_L5, TM_R3D_FPINST_L6, TM_R3D_FPINST_L7};
  const int F[8] = {0, TM_R3D_FLOP_L1, TM_R3D_FLOP_L2, TM_R3D_FLOP_L3, TM_R3D_FLOP_L4, TM_R3D_FLOP_L5, TM_R3D_FLOP_L6, TM_R3D_FLOP_L7};
  *inst = I[lmax]; *flop = F[lmax];
}
#endif
#ifdef TM_RANGE_6
template <typename R> cudaError_t tm_launch_rot3d_6(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, R* pacc) {
  dim3 grid = a.grid;
  grid.z = 2;
  TM_LAUNCH_R3(6, TM_R3D_TJ6, 4)
  return cudaGetLastError();
}
template cudaError_t tm_launch_rot3d_6<double>(const TmLaunch&, const Cx<double>*, Cx<double>*, double*);
template cudaError_t tm_launch_rot3d_6<float>(const TmLaunch&, const Cx<float>*, Cx<float>*, float*);
#endif
#ifdef TM_RANGE_7
template <typename R> cudaError_t tm_launch_rot3d_7(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, R* pacc) {
  dim3 grid = a.grid;
  grid.z = 2;
  TM_LAUNCH_R3(7, 64, 4)
  return cudaGetLastError();
}
template cudaError_t tm_launch_rot3d_7<double>(const TmLaunch&, const Cx<double>*, Cx<double>*, double*);
template cudaError_t tm_launch_rot3d_7<float>(const TmLaunch&, const Cx<float>*, Cx<float>*, float*);
#endif
#undef TM_LAUNCH_R3
#endif

#ifdef TM_SEC_ROT3DW
template <typename R> cudaError_t tm_launch_rot3d_ws(const TmLaunch& a, const Cx<R>* x, Cx<R>* up) {
  dim3 grid = a.grid;
  grid.z = 2;                                         // y'-mirror sector: slowest grid dimension
#define TM_LAUNCH_R3W(LM)                                                                                      \
  {                                                                                                             \
    constexpr int SS_ = LM >= 6 ? 4 : 8;              /* sources per stage: 2 blocks per SM must fit 4 scratch vectors each */ \
    const size_t sm = Rot3dWsSmem<R, LM, SS_>::bytes;                                                           \
    cudaFuncSetAttribute(k_allpairs_rot3d_ws<R, LM, SS_>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm); \
    k_allpairs_rot3d_ws<R, LM, SS_><<<grid, 128, sm, a.stream>>>(a.pos, x, up, a.tiles, a.n_scat, a.k_over_pi, a.inv_k, a.n_active); \
  }
  switch (a.lmax) {
    case 4: TM_LAUNCH_R3W(4) break;
    case 5: TM_LAUNCH_R3W(5) break;
    default: TM_LAUNCH_R3W(6) break;
  }
#undef TM_LAUNCH_R3W
  return cudaGetLastError();
}
template cudaError_t tm_launch_rot3d_ws<double>(const TmLaunch&, const Cx<double>*, Cx<double>*);
template cudaError_t tm_launch_rot3d_ws<float>(const TmLaunch&, const Cx<float>*, Cx<float>*);
void tm_cost_rot3d_ws(int lmax, double* inst, double* flop) {
  const int I[7] = {0, 0, 0, 0, TM_R3W_FPINST_L4, TM_R3W_FPINST_L5, TM_R3W_FPINST_L6};
  const int F[7] = {0, 0, 0, 0, TM_R3W_FLOP_L4, TM_R3W_FLOP_L5, TM_R3W_FLOP_L6};
  *inst = I[lmax]; *flop = F[lmax];
}
#endif

#ifdef TM_SEC_GEN
template <typename R> cudaError_t tm_launch_general(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, const TmConst* cst, TmTermsDev tb) {
  const dim3 grid = a.grid;
#define TM_LAUNCH_GEN(LM)                                                                                         \
  {                                                                                                               \
    const size_t sm = GenCfg<LM>::template smem<R>();                                                             \
    cudaFuncSetAttribute(k_allpairs_general<R, LM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);        \
    k_allpairs_general<R, LM><<<grid, 32 * GenCfg<LM>::WJ, sm, a.stream>>>(a.pos, x, up, a.tiles, cst, tb, a.n_scat, \
                                                                           a.k_over_pi, a.inv_k, a.n_active);     \
  }
  switch (a.lmax) {
    case 1: TM_LAUNCH_GEN(1) break;
    case 2: TM_LAUNCH_GEN(2) break;
    case 3: TM_LAUNCH_GEN(3) break;
    case 4: TM_LAUNCH_GEN(4) break;
    case 5: TM_LAUNCH_GEN(5) break;
    case 6: TM_LAUNCH_GEN(6) break;
    default: TM_LAUNCH_GEN(7) break;
  }
#undef TM_LAUNCH_GEN
  return cudaGetLastError();
}
template cudaError_t tm_launch_general<double>(const TmLaunch&, const Cx<double>*, Cx<double>*, const TmConst*, TmTermsDev);
template cudaError_t tm_launch_general<float>(const TmLaunch&, const Cx<float>*, Cx<float>*, const TmConst*, TmTermsDev);
#endif
