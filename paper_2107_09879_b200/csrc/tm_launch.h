// Launch functions of the all-pairs kernel families.  Each family is compiled in its own translation unit
// (tm_tu_*.cu: the generated straight-line code makes ptxas the long pole of the build, so the families build in
// parallel); the host code (tm_api.cu) sees only these declarations.
#pragma once
#include "tm_common.cuh"

struct TmLaunch {                // what every all-pairs launch needs
  const double* pos; const TmTile* tiles; int n_scat; double k_over_pi, inv_k; const int* n_active;
  cudaStream_t stream; dim3 grid; int lmax;
};

// launch configuration constants shared by the launch code and the host-side planning (configure_kernel)
constexpr int TM_COP_SS = 64;        // coplanar kernel: sources per shared-memory stage
constexpr int TM_SYM3D_TJ = 128;     // direct generated 3-D kernel: targets per block
constexpr int TM_SYM3D_SS = 32;      //   sources per stage
constexpr int TM_COP4_SS = 16;       // four-sector coplanar kernel (lmax 4..7): sources per stage
// four-sector coplanar kernel: targets per block.  lmax 6: ONE 8-warp block per SM, so that all warps of an SM run the
// same sector's code (a sector's loop body is 42 KB > the 32 KB L1.5 instruction cache; two co-resident 4-warp blocks
// of DIFFERENT sectors double the footprint; measured 6.80 -> 6.50 ms on the 56x56 lattice)
inline int tm_cop4_tj(int lmax) { return lmax == 6 ? 256 : 128; }
// rotation-based 3-D kernel: targets per block (shared memory per thread grows with L: scratch L/2 + accumulators L complex)
#ifndef TM_R3D_PG_FROM
#define TM_R3D_PG_FROM 6             // lmax from which accumulators live in global memory (L2-resident)
#endif
#ifndef TM_R3D_PG_LEVEL
#define TM_R3D_PG_LEVEL 2            // 1: the partner sector's share; 2: the own sector's accumulators too
#endif
#ifndef TM_R3D_TJ6
#define TM_R3D_TJ6 128               // targets per block at lmax 6 (64 with PG level 1: shared memory)
#endif
inline int tm_rot3d_tj(int lmax) { return lmax <= 3 ? 128 : (lmax == 6 ? TM_R3D_TJ6 : 64); }
// lmax 7 (internal: the gradient at lmax 6) stays at level 1 with 64-target blocks: at level 2 its compile time explodes
constexpr int tm_rot3d_pg_level(int lmax) { return lmax < TM_R3D_PG_FROM ? 0 : (lmax == 6 ? TM_R3D_PG_LEVEL : 1); }
inline int tm_rot3d_pg(int lmax) { return tm_rot3d_pg_level(lmax); }
inline int tm_general_tj(int lmax) { return lmax <= 3 ? 4 : 2; }      // table-driven kernel: targets (warps) per block

// cl: cluster size along the chunk dimension (1: none; 2 or 4: chunk partials reduced through distributed shared memory, grid.y / cl partial buffers)
template <typename R> cudaError_t tm_launch_coplanar(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, int tj, int cl, TmShift shift);   // lmax 1..3
template <typename R> cudaError_t tm_launch_coplanar4_lo(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, TmShift shift);      // lmax 4, 5
template <typename R> cudaError_t tm_launch_coplanar4_hi(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, TmShift shift);      // lmax 6, 7
template <typename R> cudaError_t tm_launch_sym3d(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, TmShift shift);             // lmax 1..3
template <typename R> cudaError_t tm_launch_rot3d_lo(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, R* pacc);                // lmax 1..5
template <typename R> cudaError_t tm_launch_rot3d_6(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, R* pacc);
template <typename R> cudaError_t tm_launch_rot3d_7(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, R* pacc);
// warp-split rotation-based kernel (lmax 4..6): 32 targets per tile, 4 warps = 4 parts of the sector's code
#ifndef TM_R3D_WS
#define TM_R3D_WS 1                  // build switch: 0 = keep the one-thread-per-target rotation-based kernel at lmax 4..6
#endif
inline bool tm_rot3d_ws(int lmax) { return TM_R3D_WS && lmax >= 4 && lmax <= 6; }
template <typename R> cudaError_t tm_launch_rot3d_ws(const TmLaunch& a, const Cx<R>* x, Cx<R>* up);
void tm_cost_rot3d_ws(int lmax, double* inst, double* flop);
template <typename R> cudaError_t tm_launch_general(const TmLaunch& a, const Cx<R>* x, Cx<R>* up, const TmConst* cst, TmTermsDev tb);   // lmax 1..7

int tm_cop4_groups(int lmax);                                  // row groups per sector (generated constant)
// executed FP work per ordered pair of the generated code (FP-pipe instructions, flop with FMA = 2)
void tm_cost_coplanar(int lmax, double* inst, double* flop);   // lmax 1..7 (four-sector code above 3)
void tm_cost_sym3d(int lmax, double* inst, double* flop);
void tm_cost_rot3d(int lmax, double* inst, double* flop);
