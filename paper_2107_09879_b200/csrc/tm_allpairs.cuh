// All-pairs translation + block matvec  u_j = sum_{i != j, same window} A_ji x_i
// (PAPER.md:336 Eq. I21: blocks are built on the fly and never stored).
//
// Two variants:
//   k_allpairs_coplanar  lmax <= 3, all scatterers in one plane z = const (every experiment of the paper):
//                        straight-line generated code, thread = target, block = one mirror-parity half,
//                        register accumulators, FP64/FP32 FMA-pipe bound.
//   k_allpairs_general   any lmax <= 6, arbitrary 3-D positions: table-driven, warp per target.
// Both write per-source-chunk partial sums u_part[chunk][n_scat][L]; the finishing kernel (tm_vecops.cuh)
// adds the chunks in a fixed order (deterministic) and applies T.
#pragma once
#include <cooperative_groups.h>

#include "tm_common.cuh"
// Sections (one per kernel family): a translation unit defines the TM_SEC_* it compiles (csrc/tm_tu_*.cu) so that the
// families build in parallel; the host code (tm_api.cu) sees only the launch functions of tm_launch.h.
#ifdef TM_SEC_COP
#include "generated/tm_coplanar_gen.cuh"
#include "generated/tm_coplanar_f2_gen.cuh"
#endif

// ---------------------------------------------------------------------------------------------------
// h_q^(1)(x), q = 0..NQ-1, by upward recurrence from h_{-1} = e^{ix}/x, h_0 = -i e^{ix}/x  (stable upward for
// the outgoing function); t = 1/x, (c, s) = (cos x, sin x).  t = 0 (self pair) gives h_q = 0 for all q.
template <typename R, int NQ>
__device__ __forceinline__ void hankel_up(R t, R c, R s, R* hr, R* hi) {
  R pr = c * t, pi = s * t;            // h_{-1}
  hr[0] = s * t; hi[0] = -c * t;       // h_0
#pragma unroll
  for (int q = 0; q + 1 < NQ; ++q) {
    const R f = R(2 * q + 1) * t;
    const R nr = fma(f, hr[q], -pr), ni = fma(f, hi[q], -pi);
    pr = hr[q]; pi = hi[q];
    hr[q + 1] = nr; hi[q + 1] = ni;
  }
}

// cos/sin of k*r with the range reduction done in double (fp32 hazard: k r reaches ~900).
template <typename R> __device__ __forceinline__ void phase_kr(double k_over_pi, double r, R& c, R& s);
template <> __device__ __forceinline__ void phase_kr<double>(double k_over_pi, double r, double& c, double& s) {
  sincospi(k_over_pi * r, &s, &c);
}
template <> __device__ __forceinline__ void phase_kr<float>(double k_over_pi, double r, float& c, float& s) {
  double t = k_over_pi * r;
  t -= 2.0 * rint(0.5 * t);            // exact: t in [-1, 1]
  sincospif((float)t, &s, &c);
}

// Optional rigid displacement of all TARGETS against the sources (tm_grad_positions: numerical differentiation of the
// translation operator in its displacement argument).  With a non-zero shift the self pair no longer has r = 0 and is
// excluded by index instead.

#ifdef TM_SEC_COP
// Accumulators of one parity half: two real arrays in fp64; one float2 per complex number in fp32, where the generated
// code uses Blackwell's packed FFMA2 arithmetic (generated/tm_coplanar_f2_gen.cuh) to halve the FP issue slots.
template <typename R, int NH> struct CopAcc {
  R ar[NH], ai[NH];
  __device__ __forceinline__ void clear() {
#pragma unroll
    for (int b = 0; b < NH; ++b) { ar[b] = R(0); ai[b] = R(0); }
  }
};
template <int NH> struct CopAcc<float, NH> {
  float2 a[NH];
  __device__ __forceinline__ void clear() {
#pragma unroll
    for (int b = 0; b < NH; ++b) a[b] = make_float2(0.f, 0.f);
  }
};

template <typename R, int LMAX, int H> struct CopPair;
#define TM_COP_SPEC(LM, HH)                                                                              \
  template <> struct CopPair<double, LM, HH> {                                                           \
    static constexpr int NH = TM_COP_NH_L##LM;                                                           \
    static __device__ __forceinline__ void run(const double* xs, const double* cm, const double* sm,     \
                                               const double* hr, const double* hi, CopAcc<double, NH>& A) { \
      tm_cop_pair_L##LM##_H##HH<double>(xs, cm, sm, hr, hi, A.ar, A.ai);                                 \
    }                                                                                                    \
    template <typename HK>                                                                               \
    static __device__ __forceinline__ void run_hk(const double* xs, const double* cm, const double* sm,  \
                                                  const double* hr, const double* hi, CopAcc<double, NH>& A, const HK& hk) { \
      tm_cop_pair_L##LM##_H##HH##_hk<double, HK>(xs, cm, sm, hr, hi, A.ar, A.ai, hk);                    \
    }                                                                                                    \
    static __device__ __forceinline__ void unmix(const CopAcc<double, NH>& A, Cx<double>* out) {         \
      tm_cop_unmix_L##LM##_H##HH<double, Cx<double>>(A.ar, A.ai, out);                                   \
    }                                                                                                    \
    static __device__ __forceinline__ void stage_entry(int k, int& a, int& b, int& sg) {                 \
      a = tm_cop_sa_L##LM##_H##HH[k]; b = tm_cop_sb_L##LM##_H##HH[k]; sg = tm_cop_ss_L##LM##_H##HH[k];   \
    }                                                                                                    \
  };                                                                                                     \
  template <> struct CopPair<float, LM, HH> {                                                            \
    static constexpr int NH = TM_COP_NH_L##LM;                                                           \
    static __device__ __forceinline__ void run(const float* xs, const float* cm, const float* sm,        \
                                               const float* hr, const float* hi, CopAcc<float, NH>& A) { \
      tm_cop_pair_f2_L##LM##_H##HH(reinterpret_cast<const float2*>(xs), cm, sm, hr, hi, A.a);            \
    }                                                                                                    \
    template <typename HK>                                                                               \
    static __device__ __forceinline__ void run_hk(const float* xs, const float* cm, const float* sm,     \
                                                  const float* hr, const float* hi, CopAcc<float, NH>& A, const HK& hk) { \
      hk.template at<0>(); hk.template at<HK::B>();                /* packed-fp32 code has no hook points */ \
      tm_cop_pair_f2_L##LM##_H##HH(reinterpret_cast<const float2*>(xs), cm, sm, hr, hi, A.a);            \
    }                                                                                                    \
    static __device__ __forceinline__ void unmix(const CopAcc<float, NH>& A, Cx<float>* out) {           \
      tm_cop_unmix_f2_L##LM##_H##HH<Cx<float>>(A.a, out);                                                \
    }                                                                                                    \
    static __device__ __forceinline__ void stage_entry(int k, int& a, int& b, int& sg) {                 \
      a = tm_cop_sa_L##LM##_H##HH[k]; b = tm_cop_sb_L##LM##_H##HH[k]; sg = tm_cop_ss_L##LM##_H##HH[k];   \
    }                                                                                                    \
  };
TM_COP_SPEC(1, 0) TM_COP_SPEC(1, 1) TM_COP_SPEC(2, 0) TM_COP_SPEC(2, 1) TM_COP_SPEC(3, 0) TM_COP_SPEC(3, 1)
#undef TM_COP_SPEC

// ---------------------------------------------------------------------------------------------------
// Coplanar kernel.  grid = (n_tiles, n_chunk, 2); block = TJ threads.  blockIdx.z selects the mirror-parity
// half: it is the SLOWEST grid dimension, so at any time (almost) all resident blocks of an SM run the same
// half and its ~30 KB of straight-line code stays within the 32 KB L1.5 instruction cache (ncu showed the
// two-halves-per-block version stalled on instruction fetch: profiles/r01_recorded_runs.md, kernel history).
// Thread t handles target tile.tgt_start + t.  Sources of the tile's window are split into n_chunk contiguous
// chunks (blockIdx.y) so that small problems still fill 148 SMs; each chunk is streamed through shared memory
// SS sources at a time (positions + this half's d-values in the tilde basis x~ = i^p x).
#ifndef TM_COP_PIPE
#define TM_COP_PIPE 1            // 1: the head of the pair set-up (rsqrt, phase of k r) is computed one source ahead
#endif
#ifndef TM_COP_HOOK_NUM
#define TM_COP_HOOK_NUM 1        // the phase of the next pair is computed at hook point NH * NUM / DEN + 1 (row of the axial translation)
#define TM_COP_HOOK_DEN 2
#endif
// Set-up head of the NEXT pair, run from the hook points of the generated apply code (mutable: the hooks take it by const reference).
template <typename R, int B_> struct CopHead {
  static constexpr int B = B_;
  const double* px; const double* py; double xj, yj, k_over_pi; int self;   // self: stage index of the pair to annihilate (shifted targets), or -1
  mutable int sn;                                                             // stage index of the next source
  mutable double dx, dy, r2, rinv; mutable R ck, sk;
  template <int K> __device__ __forceinline__ void at() const {
    if constexpr (K == 0) {
      dx = xj - px[sn]; dy = yj - py[sn];                      // d = x_dest - x_source (reading R3)
      r2 = dx * dx + dy * dy;
      rinv = (r2 > 0.0 && sn != self) ? rsqrt(r2) : 0.0;       // self pair -> h_q = 0 -> nothing
    } else if constexpr (K == B) {
      phase_kr<R>(k_over_pi, r2 * rinv, ck, sk);
    }
  }
};
#ifndef TM_COP_MINBLOCKS
#define TM_COP_MINBLOCKS 1       // resident blocks per SM the register allocation is asked to allow (experiments: 3)
#endif
// CL > 1: the kernel is launched in thread-block CLUSTERS of CL blocks along the source-chunk dimension (grid.y % CL == 0).
// The CL chunk partials of a tile are then summed INSIDE the launch through distributed shared memory - every block stages its
// partial rows in its own shared memory, the cluster synchronises, and the blocks share the rows out and add the CL partials in
// the fixed order of the cluster ranks (deterministic) - so only grid.y / CL partial buffers of u reach memory instead of
// grid.y.  On config 5 (8 chunks) this takes the launch's DRAM traffic from 572 MB to the order of the algorithmic 43 MB.
// Clusters of 4, not 8: a GPC of 18 SMs has 36 block slots of this kernel, which clusters of 8 cannot fill.
template <typename R, int LMAX, int TJ, int SS, int CL = 1>
__global__ void __launch_bounds__(TJ, TM_COP_MINBLOCKS)
k_allpairs_coplanar(const double* __restrict__ pos, const Cx<R>* __restrict__ x, Cx<R>* __restrict__ u_part,
                    const TmTile* __restrict__ tiles, int n_scat, double k_over_pi, double inv_k,
                    const int* __restrict__ n_active, TmShift shift) {
  constexpr int L = 2 * LMAX * (LMAX + 2);
  constexpr int NH = L / 2;
  constexpr int NQ = 2 * LMAX + 1;
  if (n_active != nullptr && *n_active == 0) return;     // grid-uniform: all blocks of a cluster leave together

  __shared__ double s_px[SS], s_py[SS];
  __shared__ __align__(16) R s_x[SS * NH * 2];         // [source][NH] complex, tilde basis, this half only
  __shared__ int s_sa[NH], s_sb[NH], s_ss[NH];       // staging: d_k = x~[sa] + ss * x~[sb]

  const TmTile tile = tiles[blockIdx.x];
  const int tid = threadIdx.x;
  const int half = blockIdx.z;
  const bool live = tid < tile.tgt_count;
  const int j = tile.tgt_start + (live ? tid : tile.tgt_count - 1);
  const double xj = pos[3 * j] + shift.x, yj = pos[3 * j + 1] + shift.y;     // shift.z must be 0 for this kernel

  // this block's chunk of the window's sources
  const int per = (tile.src_count + gridDim.y - 1) / gridDim.y;
  const int c0 = tile.src_start + blockIdx.y * per;
  const int c1 = min(tile.src_start + tile.src_count, c0 + per);

  if (tid < NH) {
    int a, b, sg;
    if (half == 0) CopPair<R, LMAX, 0>::stage_entry(tid, a, b, sg); else CopPair<R, LMAX, 1>::stage_entry(tid, a, b, sg);
    s_sa[tid] = a; s_sb[tid] = b; s_ss[tid] = sg;
  }

  CopAcc<R, NH> acc;
  acc.clear();

  for (int s0 = c0; s0 < c1; s0 += SS) {
    const int ns = min(SS, c1 - s0);
    __syncthreads();                                   // previous stage fully consumed (also orders the staging tables)
    for (int e = tid; e < ns; e += TJ) { s_px[e] = pos[3 * (s0 + e)]; s_py[e] = pos[3 * (s0 + e) + 1]; }
    for (int e = tid; e < ns * NH; e += TJ) {
      const int src = e / NH, kk = e - src * NH;
      const Cx<R>* xrow = x + (size_t)(s0 + src) * L;
      const int ia = s_sa[kk], sg = s_ss[kk];
      Cx<R> v = xrow[ia];
      if (sg != 0) {                                   // d^+- = x_{l,m,p} +- x_{l,-m,p}  (pair's y'-mirror symmetry)
        const Cx<R> o = xrow[s_sb[kk]];
        v = sg > 0 ? cadd(v, o) : csub(v, o);
      }
      if (ia >= NH) v = cx<R>(-v.im, v.re);            // tilde basis: multiply p = 1 modes by i
      s_x[2 * e] = v.re;
      s_x[2 * e + 1] = v.im;
    }
    __syncthreads();
#if TM_COP_PIPE
    // Software pipeline over the sources of a stage: the serial head of a pair's set-up (rsqrt, then the phase of k r -
    // two long dependent chains with no parallelism of their own) is computed ONE SOURCE AHEAD, so that it interleaves
    // with the previous source's apply code instead of standing alone at the top of the loop body.
    // With the hook points of the generated code (tm_cop_pair_*_hk) the two chains sit INSIDE the previous source's apply
    // code: the rsqrt after its frame change (hook 0), the phase after row TM_COP_HOOK_B - 1 of its axial translation.
    using Head = CopHead<R, NH * TM_COP_HOOK_NUM / TM_COP_HOOK_DEN + 1>;
    Head hd{s_px, s_py, xj, yj, k_over_pi, shift.on ? j - s0 : -1, 0, 0.0, 0.0, 0.0, 0.0, R(0), R(0)};
    hd.template at<0>(); hd.template at<Head::B>();
#pragma unroll 1
    for (int s = 0; s < ns; ++s) {
      const double dx = hd.dx, dy = hd.dy, rinv = hd.rinv;
      const R ck = hd.ck, sk = hd.sk;
      hd.sn = min(s + 1, ns - 1);
      R cm[LMAX + 1], sm[LMAX + 1];
      cm[0] = R(1); sm[0] = R(0);
      cm[1] = (R)(dx * rinv); sm[1] = (R)(dy * rinv);
      if (rinv == 0.0 && dx == 0.0 && dy == 0.0) cm[1] = R(1);
#pragma unroll
      for (int m = 2; m <= LMAX; ++m) {
        cm[m] = cm[m - 1] * cm[1] - sm[m - 1] * sm[1];
        sm[m] = sm[m - 1] * cm[1] + cm[m - 1] * sm[1];
      }
      R hr[NQ], hi[NQ];
      hankel_up<R, NQ>((R)(rinv * inv_k), ck, sk, hr, hi);
      const R* xs = &s_x[s * NH * 2];
      if (half == 0) CopPair<R, LMAX, 0>::run_hk(xs, cm, sm, hr, hi, acc, hd);
      else           CopPair<R, LMAX, 1>::run_hk(xs, cm, sm, hr, hi, acc, hd);
    }
#else
#pragma unroll 1
    for (int s = 0; s < ns; ++s) {
      const double dx = xj - s_px[s], dy = yj - s_py[s];        // d = x_dest - x_source (reading R3)
      const double r2 = dx * dx + dy * dy;
      const double rinv = (r2 > 0.0 && !(shift.on && s0 + s == j)) ? rsqrt(r2) : 0.0;   // self pair -> h_q = 0 -> nothing
      const double r = r2 * rinv;
      R cm[LMAX + 1], sm[LMAX + 1];
      cm[0] = R(1); sm[0] = R(0);
      cm[1] = (R)(dx * rinv); sm[1] = (R)(dy * rinv);
      if (r2 == 0.0) cm[1] = R(1);
#pragma unroll
      for (int m = 2; m <= LMAX; ++m) {
        cm[m] = cm[m - 1] * cm[1] - sm[m - 1] * sm[1];
        sm[m] = sm[m - 1] * cm[1] + cm[m - 1] * sm[1];
      }
      R ck, sk;
      phase_kr<R>(k_over_pi, r, ck, sk);
      R hr[NQ], hi[NQ];
      hankel_up<R, NQ>((R)(rinv * inv_k), ck, sk, hr, hi);
      const R* xs = &s_x[s * NH * 2];
      if (half == 0) CopPair<R, LMAX, 0>::run(xs, cm, sm, hr, hi, acc);
      else           CopPair<R, LMAX, 1>::run(xs, cm, sm, hr, hi, acc);
    }
#endif
  }

  // this chunk's partial sums of this half, back in the standard basis:
  // u~_{l,+-m,p} = (A^+ +- A^-)/2,  u_b = (-i)^{p_b} u~_b
  if constexpr (CL <= 1) {
    if (live) {
      Cx<R>* out = u_part + ((size_t)blockIdx.y * n_scat + j) * L;
      if (half == 0) CopPair<R, LMAX, 0>::unmix(acc, out);
      else           CopPair<R, LMAX, 1>::unmix(acc, out);
    }
  } else {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(16) unsigned char s_dyn_cl[];
    Cx<R>* s_part = reinterpret_cast<Cx<R>*>(s_dyn_cl);          // [TJ][L]: this block's partial rows (only this half's entries are written)
    __shared__ int s_hidx[NH];                                    // flat indices of this half's NH modes
    if (tid == 0) {
      int n = 0;
      for (int k = 0; k < NH; ++k) {
        if (s_ss[k] >= 0) s_hidx[n++] = s_sa[k];                  // kinds '0' and '+': (l, |m|, p)
        if (s_ss[k] > 0) s_hidx[n++] = s_sb[k];                   // kind '+': (l, -|m|, p) too
      }
    }
    if (half == 0) CopPair<R, LMAX, 0>::unmix(acc, s_part + (size_t)tid * L);
    else           CopPair<R, LMAX, 1>::unmix(acc, s_part + (size_t)tid * L);
    cluster.sync();                                               // every block's rows are staged (also orders s_hidx)
    const unsigned rank = cluster.block_rank();
    const Cx<R>* peer[CL];
#pragma unroll
    for (int c = 0; c < CL; ++c) peer[c] = cluster.map_shared_rank(s_part, c);
    Cx<R>* out = u_part + ((size_t)(blockIdx.y / CL) * n_scat + tile.tgt_start) * L;
    for (int e = rank * TJ + tid; e < TJ * NH; e += CL * TJ) {
      const int t = e / NH, a = s_hidx[e - t * NH];
      if (t >= tile.tgt_count) continue;
      Cx<R> sum = peer[0][t * L + a];
#pragma unroll
      for (int c = 1; c < CL; ++c) sum = cadd(sum, peer[c][t * L + a]);          // fixed order: cluster rank = chunk index mod CL
      out[(size_t)t * L + a] = sum;
    }
    cluster.sync();                                               // no block leaves while a peer still reads its rows
  }
}

#endif  // TM_SEC_COP
#ifdef TM_SEC_GEN
// ---------------------------------------------------------------------------------------------------
// General 3-D kernel (any lmax <= 6).  Term table on the device: for destination row b, terms
// row_ptr[b] <= t < row_ptr[b+1] with source column col[t], scalar-wave index widx[t] = q^2 + q + mu
// (mu = m_col - m_b) and coefficient coef[t] (real part if !imag[t], imaginary part otherwise):
//      A[b][col] += coef * h_q(kr) Pbar_q^{|mu|}(cos theta) e^{i mu phi}                 (Eq. I17)

template <int LMAX> struct GenCfg {
  static constexpr int L = 2 * LMAX * (LMAX + 2);
  static constexpr int NQ = 2 * LMAX + 1;
  static constexpr int NW2 = NQ * NQ;
  static constexpr int SG = 16;                         // sources per stage
  static constexpr int WJ = (LMAX <= 3) ? 4 : 2;        // targets (warps) per block
  static constexpr int RB = (L + 31) / 32;              // rows per lane
  template <typename R> static constexpr size_t smem() { return sizeof(Cx<R>) * (size_t)(SG * L + WJ * SG * NW2); }
};

template <typename R, int LMAX>
__global__ void __launch_bounds__(32 * GenCfg<LMAX>::WJ)
k_allpairs_general(const double* __restrict__ pos, const Cx<R>* __restrict__ x, Cx<R>* __restrict__ u_part,
                   const TmTile* __restrict__ tiles, const TmConst* __restrict__ cst, TmTermsDev tb, int n_scat,
                   double k_over_pi, double inv_k, const int* __restrict__ n_active) {
  using G = GenCfg<LMAX>;
  constexpr int L = G::L, NQ = G::NQ, NW2 = G::NW2, SG = G::SG, WJ = G::WJ, RB = G::RB;
  if (n_active != nullptr && *n_active == 0) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Cx<R>* s_x = reinterpret_cast<Cx<R>*>(smem_raw);                 // [SG][L]
  Cx<R>* s_w = s_x + SG * L;                                       // [WJ][SG][NW2]

  const TmTile tile = tiles[blockIdx.x];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const bool live = warp < tile.tgt_count;
  const int j = tile.tgt_start + (live ? warp : 0);
  const double xj = pos[3 * j], yj = pos[3 * j + 1], zj = pos[3 * j + 2];
  const int per = (tile.src_count + gridDim.y - 1) / gridDim.y;
  const int c0 = tile.src_start + blockIdx.y * per;
  const int c1 = min(tile.src_start + tile.src_count, c0 + per);

  Cx<R> acc[RB];
  int m_b[RB];
#pragma unroll
  for (int rb = 0; rb < RB; ++rb) { acc[rb] = cx<R>(R(0), R(0)); const int b = lane + 32 * rb; m_b[rb] = b < L ? cst->mode_m[b] : 0; }

  for (int s0 = c0; s0 < c1; s0 += SG) {
    const int ns = min(SG, c1 - s0);
    __syncthreads();
    for (int e = threadIdx.x; e < ns * L; e += 32 * WJ) s_x[e] = x[(size_t)s0 * L + e];
    // phase 1: lane s builds the (2 lmax + 1)^2 scalar outgoing waves of pair (j, s0 + s)
    if (lane < ns) {
      const int i = s0 + lane;
      const double dx = xj - pos[3 * i], dy = yj - pos[3 * i + 1], dz = zj - pos[3 * i + 2];
      const double rho2 = dx * dx + dy * dy, r2 = rho2 + dz * dz;
      const double rinv = r2 > 0.0 ? rsqrt(r2) : 0.0;
      const double r = r2 * rinv;
      const double rhoinv = rho2 > 0.0 ? rsqrt(rho2) : 0.0;
      const R ct = (R)(dz * rinv), st = (R)(rho2 * rhoinv * rinv);
      const R cph = rho2 > 0.0 ? (R)(dx * rhoinv) : R(1), sph = (R)(dy * rhoinv);
      R ck, sk;
      phase_kr<R>(k_over_pi, r, ck, sk);
      R hr[NQ], hi[NQ];
      hankel_up<R, NQ>((R)(rinv * inv_k), ck, sk, hr, hi);
      Cx<R>* w = s_w + (size_t)(warp * SG + lane) * NW2;
      R pmm = R(0.70710678118654752440);                 // Pbar_0^0
      R em_r = R(1), em_i = R(0);                        // e^{i mu phi}
#pragma unroll
      for (int mu = 0; mu < NQ; ++mu) {
        if (mu > 0) {
          pmm *= (R)cst->leg_d[mu] * st;
          const R t = em_r * cph - em_i * sph; em_i = em_i * cph + em_r * sph; em_r = t;
        }
        R p2 = R(0), p1 = pmm;                           // Pbar_{q-2}^mu, Pbar_{q-1}^mu
#pragma unroll
        for (int q = mu; q < NQ; ++q) {
          R pq;
          if (q == mu) pq = pmm;
          else { pq = (R)cst->leg_a[q][mu] * (ct * p1 - (R)cst->leg_b[q][mu] * p2); p2 = p1; p1 = pq; }
          const R gr = hr[q] * pq, gi = hi[q] * pq;      // h_q Pbar_q^mu
          w[q * q + q + mu] = cx<R>(gr * em_r - gi * em_i, gr * em_i + gi * em_r);
          if (mu > 0) w[q * q + q - mu] = cx<R>(gr * em_r + gi * em_i, -gr * em_i + gi * em_r);
        }
      }
    }
    __syncthreads();
    // phase 2: lane = destination row(s) b; loop terms of the row, then the staged sources
    if (live) {
      const Cx<R>* wj = s_w + (size_t)warp * SG * NW2;
#pragma unroll
      for (int rb = 0; rb < RB; ++rb) {
        const int b = lane + 32 * rb;
        if (b >= L) continue;
        const int t0 = tb.row_ptr[b], t1 = tb.row_ptr[b + 1];
        Cx<R> a = acc[rb];
        for (int t = t0; t < t1; ++t) {
          const int col = tb.col[t], wi = tb.widx[t];
          const R cf = (R)tb.coef[t];
          const bool im = tb.imag[t] != 0;
          for (int s = 0; s < ns; ++s) {
            const Cx<R> wv = wj[s * NW2 + wi];
            const Cx<R> e = im ? cx<R>(-cf * wv.im, cf * wv.re) : cx<R>(cf * wv.re, cf * wv.im);
            a = cfma(e, s_x[s * L + col], a);
          }
        }
        acc[rb] = a;
      }
    }
  }
  if (live) {
    Cx<R>* out = u_part + ((size_t)blockIdx.y * n_scat + j) * L;
#pragma unroll
    for (int rb = 0; rb < RB; ++rb) { const int b = lane + 32 * rb; if (b < L) out[b] = acc[rb]; }
  }
  (void)m_b;
}

#endif  // TM_SEC_GEN
#ifdef TM_SEC_SYM3D
// ---------------------------------------------------------------------------------------------------
// Generated 3-D kernel (arbitrary positions, lmax <= 3).  Same scheme as the coplanar kernel - rotate about z onto
// the pair's azimuth, exploit the mirror y' -> -y' of the rotated pair (+- basis), never form the block:
//     u^new_r = sum_q h_q(kr) sum_c ( sum_mu kappa Pbar_q^mu(cos theta) ) x^new_c      (kappa real constants)
// but without the z-mirror: the L modes split into two SECTORS of L/2 (blockIdx.z, slowest grid dimension).
// Thread = target; x^new (L/2 complex), the row sums, h_q and two levels of the Legendre recurrence in registers; the accumulators
// (own sector's A and the partner sector's share produced by the output rotation: L complex) live in shared memory
// [slot][thread] (conflict-free).  Each sector writes its share of u to its own partial buffer
// u_part[(chunk * 2 + sector)][n_scat][L]; the finishing kernel adds them in fixed order.
#include "generated/tm_general3d_gen.cuh"

template <typename R, int LMAX, int S> struct G3dPair;
#define TM_G3D_SPEC(LM, SS_)                                                                             \
  template <typename R> struct G3dPair<R, LM, SS_> {                                                     \
    template <int AS>                                                                                    \
    static __device__ __forceinline__ void run(const R* xs, const R* cm, const R* sm, const R* hr,       \
                                               const R* hi, R ct, R st, R* ar, R* ai) {                  \
      tm_g3d_pair_L##LM##_S##SS_<R, AS>(xs, cm, sm, hr, hi, ct, st, ar, ai);                             \
    }                                                                                                    \
    template <int AS>                                                                                    \
    static __device__ __forceinline__ void unmix(const R* ar, const R* ai, Cx<R>* out) {                 \
      tm_g3d_unmix_L##LM##_S##SS_<R, Cx<R>, AS>(ar, ai, out);                                            \
    }                                                                                                    \
    static __device__ __forceinline__ void stage_entry(int k, int& a, int& b, int& sg) {                 \
      a = tm_g3d_sa_L##LM##_S##SS_[k]; b = tm_g3d_sb_L##LM##_S##SS_[k]; sg = tm_g3d_ss_L##LM##_S##SS_[k]; \
    }                                                                                                    \
  };
TM_G3D_SPEC(1, 0) TM_G3D_SPEC(1, 1) TM_G3D_SPEC(2, 0) TM_G3D_SPEC(2, 1) TM_G3D_SPEC(3, 0) TM_G3D_SPEC(3, 1)
#undef TM_G3D_SPEC

template <typename R, int LMAX, int TJ, int SS> struct Sym3dSmem {
  static constexpr int L = 2 * LMAX * (LMAX + 2);
  static constexpr size_t bytes = sizeof(double) * 3 * SS + sizeof(R) * (size_t)(SS * L * 2 + 2 * L * TJ) + sizeof(int) * 3 * L;
};

template <typename R, int LMAX, int TJ, int SS>
__global__ void __launch_bounds__(TJ)
k_allpairs_sym3d(const double* __restrict__ pos, const Cx<R>* __restrict__ x, Cx<R>* __restrict__ u_part,
                 const TmTile* __restrict__ tiles, int n_scat, double k_over_pi, double inv_k,
                 const int* __restrict__ n_active, TmShift shift) {
  constexpr int L = 2 * LMAX * (LMAX + 2);
  constexpr int NS = L / 2;                 // slots per sector
  constexpr int NQ = 2 * LMAX + 1;
  if (n_active != nullptr && *n_active == 0) return;

  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* s_px = reinterpret_cast<double*>(smem_raw);
  double* s_py = s_px + SS;
  double* s_pz = s_py + SS;
  R* s_x = reinterpret_cast<R*>(s_pz + SS);          // [source][2 NS] complex: own slots then partner slots
  R* s_acc = s_x + SS * L * 2;                       // [re/im][2 NS][TJ]
  int* s_sa = reinterpret_cast<int*>(s_acc + 2 * L * TJ);
  int* s_sb = s_sa + L;
  int* s_ss = s_sb + L;

  const TmTile tile = tiles[blockIdx.x];
  const int tid = threadIdx.x;
  const int sct = blockIdx.z;
  const bool live = tid < tile.tgt_count;
  const int j = tile.tgt_start + (live ? tid : tile.tgt_count - 1);
  const double xj = pos[3 * j] + shift.x, yj = pos[3 * j + 1] + shift.y, zj = pos[3 * j + 2] + shift.z;
  const int per = (tile.src_count + gridDim.y - 1) / gridDim.y;
  const int c0 = tile.src_start + blockIdx.y * per;
  const int c1 = min(tile.src_start + tile.src_count, c0 + per);

  if (tid < L) {
    int a, b, sg;
    if (sct == 0) G3dPair<R, LMAX, 0>::stage_entry(tid, a, b, sg); else G3dPair<R, LMAX, 1>::stage_entry(tid, a, b, sg);
    s_sa[tid] = a; s_sb[tid] = b; s_ss[tid] = sg;
  }
  R* ar = s_acc + tid;
  R* ai = s_acc + L * TJ + tid;
#pragma unroll
  for (int b = 0; b < L; ++b) { ar[b * TJ] = R(0); ai[b * TJ] = R(0); }

  for (int s0 = c0; s0 < c1; s0 += SS) {
    const int ns = min(SS, c1 - s0);
    __syncthreads();
    for (int e = tid; e < ns; e += TJ) {
      s_px[e] = pos[3 * (s0 + e)]; s_py[e] = pos[3 * (s0 + e) + 1]; s_pz[e] = pos[3 * (s0 + e) + 2];
    }
    for (int e = tid; e < ns * L; e += TJ) {
      const int src = e / L, kk = e - src * L;
      const Cx<R>* xrow = x + (size_t)(s0 + src) * L;
      const int ia = s_sa[kk], sg = s_ss[kk];
      Cx<R> v = xrow[ia];
      if (sg != 0) {
        const Cx<R> o = xrow[s_sb[kk]];
        v = sg > 0 ? cadd(v, o) : csub(v, o);
      }
      if (ia >= NS) v = cx<R>(-v.im, v.re);            // tilde basis: multiply p = 1 modes by i
      s_x[2 * e] = v.re;
      s_x[2 * e + 1] = v.im;
    }
    __syncthreads();
#pragma unroll 1
    for (int s = 0; s < ns; ++s) {
      const double dx = xj - s_px[s], dy = yj - s_py[s], dz = zj - s_pz[s];   // d = x_dest - x_source (reading R3)
      const double rho2 = dx * dx + dy * dy, r2 = rho2 + dz * dz;
      const double rinv = (r2 > 0.0 && !(shift.on && s0 + s == j)) ? rsqrt(r2) : 0.0;   // self pair -> h_q = 0 -> nothing
      const double rhoinv = rho2 > 0.0 ? rsqrt(rho2) : 0.0;
      const double r = r2 * rinv;
      R cm[LMAX + 1], sm[LMAX + 1];
      cm[0] = R(1); sm[0] = R(0);
      cm[1] = rho2 > 0.0 ? (R)(dx * rhoinv) : R(1); sm[1] = (R)(dy * rhoinv);
#pragma unroll
      for (int m = 2; m <= LMAX; ++m) {
        cm[m] = cm[m - 1] * cm[1] - sm[m - 1] * sm[1];
        sm[m] = sm[m - 1] * cm[1] + cm[m - 1] * sm[1];
      }
      R ck, sk;
      phase_kr<R>(k_over_pi, r, ck, sk);
      R hr[NQ], hi[NQ];
      hankel_up<R, NQ>((R)(rinv * inv_k), ck, sk, hr, hi);
      const R ct = (R)(dz * rinv), st = (R)(rho2 * rhoinv * rinv);      // cos / sin of the polar angle of d
      const R* xs = &s_x[s * L * 2];
      if (sct == 0) G3dPair<R, LMAX, 0>::template run<TJ>(xs, cm, sm, hr, hi, ct, st, ar, ai);
      else          G3dPair<R, LMAX, 1>::template run<TJ>(xs, cm, sm, hr, hi, ct, st, ar, ai);
    }
  }
  if (live) {
    Cx<R>* out = u_part + ((size_t)(blockIdx.y * 2 + sct) * n_scat + j) * L;
    if (sct == 0) G3dPair<R, LMAX, 0>::template unmix<TJ>(ar, ai, out);
    else          G3dPair<R, LMAX, 1>::template unmix<TJ>(ar, ai, out);
  }
}

#endif  // TM_SEC_SYM3D
#ifdef TM_SEC_ROT3D
// ---------------------------------------------------------------------------------------------------
// Rotation-based 3-D kernel (arbitrary positions, any lmax 1..7): rotation - axial translation - rotation with the theta
// rotation written as  constant frame change . phase rotation . constant frame change  (gen_tables.py: rot3d_sectors), so
// the per-pair work is O(L^1.5) for every pair direction: 1516 FP instructions per ordered pair at lmax 3 (sym3d: 4094),
// ~7000 at lmax 6 (table-driven kernel: ~150 000).  Thread = target, one y'-mirror sector per block (blockIdx.z); the
// sector's vector in the pair-axis frame (n = L/2 complex) lives in a per-thread shared-memory scratch [slot][thread]
// because the frame changes are block diagonal in (l, p) and the axial translation in |m''|; accumulators (own sector +
// partner share) in shared memory as in k_allpairs_sym3d.  Partial buffers and the finishing kernel as for sym3d.
// zero-cost scheduling pin: the compiler must treat v as modified here (keeps a value's consumers after this point)
#ifndef TM_PIN
__device__ __forceinline__ void tm_pin(double& v) { asm volatile("" : "+d"(v)); }
__device__ __forceinline__ void tm_pin(float& v) { asm volatile("" : "+f"(v)); }
#define TM_PIN(v) tm_pin(v)
#endif
#include "generated/tm_rot3d_gen.cuh"

template <typename R, int LMAX, int S> struct R3dPair;
#define TM_R3D_SPEC(LM, SS_)                                                                             \
  template <typename R> struct R3dPair<R, LM, SS_> {                                                     \
    template <int AS>                                                                                    \
    static __device__ __forceinline__ void run(const R* xs, R cph, R sph, R cth, R sth, R* hr, R* hi,    \
                                               R* sr, R* si, R* ar, R* ai, R* pr, R* pi) {               \
      tm_r3d_pair_L##LM##_S##SS_<R, AS>(xs, cph, sph, cth, sth, hr, hi, sr, si, ar, ai, pr, pi);         \
    }                                                                                                    \
    template <int AS>                                                                                    \
    static __device__ __forceinline__ void unmix(const R* ar, const R* ai, const R* pr, const R* pi, Cx<R>* out) { \
      tm_r3d_unmix_L##LM##_S##SS_<R, Cx<R>, AS>(ar, ai, pr, pi, out);                                    \
    }                                                                                                    \
    static __device__ __forceinline__ void stage_entry(int k, int& a, int& b, int& sg) {                 \
      a = tm_r3d_sa_L##LM##_S##SS_[k]; b = tm_r3d_sb_L##LM##_S##SS_[k]; sg = tm_r3d_ss_L##LM##_S##SS_[k]; \
    }                                                                                                    \
  };
TM_R3D_SPEC(1, 0) TM_R3D_SPEC(1, 1) TM_R3D_SPEC(2, 0) TM_R3D_SPEC(2, 1) TM_R3D_SPEC(3, 0) TM_R3D_SPEC(3, 1) TM_R3D_SPEC(4, 0)
TM_R3D_SPEC(4, 1) TM_R3D_SPEC(5, 0) TM_R3D_SPEC(5, 1) TM_R3D_SPEC(6, 0) TM_R3D_SPEC(6, 1) TM_R3D_SPEC(7, 0) TM_R3D_SPEC(7, 1)
#undef TM_R3D_SPEC

// PG: the partner sector's share of the accumulators lives in GLOBAL memory (L2-resident, [block][re/im][slot][thread],
// coalesced) instead of shared memory: at lmax >= 6 the three per-thread vectors (scratch, own and partner accumulators)
// leave room for a single 2-warp block per SM; with the partner share in L2 two blocks fit and every scheduler has a warp.
// PG = 2: the own sector's accumulators too (shared memory then holds only the scratch vector: 128-thread blocks, 8 warps per SM;
// measured at lmax 6 on the 56x56 lattice: 27.4 ms (PG 1, 64 targets) -> 24.3 ms (PG 2, 128 targets); PG 2 with 64 targets: 33.0 ms).
template <typename R, int LMAX, int TJ, int SS, int PG> struct Rot3dSmem {
  static constexpr int L = 2 * LMAX * (LMAX + 2);
  // positions | staged d-values (own + partner = L slots) | scratch (L/2 slots) | accumulators (L, L/2 or 0 slots) | staging tables
  static constexpr size_t bytes = sizeof(double) * 3 * SS + sizeof(R) * (size_t)(SS * L * 2 + L * TJ + (2 - PG) * L * TJ) + sizeof(int) * 3 * L;
};

template <typename R, int LMAX, int TJ, int SS, int PG>
__global__ void __launch_bounds__(TJ)
k_allpairs_rot3d(const double* __restrict__ pos, const Cx<R>* __restrict__ x, Cx<R>* __restrict__ u_part,
                 const TmTile* __restrict__ tiles, int n_scat, double k_over_pi, double inv_k,
                 const int* __restrict__ n_active, R* __restrict__ g_pacc) {
  constexpr int L = 2 * LMAX * (LMAX + 2);
  constexpr int NS = L / 2;                 // slots per sector
  constexpr int NQ = 2 * LMAX + 1;
  if (n_active != nullptr && *n_active == 0) return;

  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* s_px = reinterpret_cast<double*>(smem_raw);
  double* s_py = s_px + SS;
  double* s_pz = s_py + SS;
  R* s_x = reinterpret_cast<R*>(s_pz + SS);          // [source][2 NS] complex: own slots then partner slots
  R* s_scr = s_x + SS * L * 2;                       // [re/im][NS][TJ]
  R* s_acc = s_scr + L * TJ;                         // [re/im][NS][TJ] own sector, then (unless PG) [re/im][NS][TJ] partner share
  int* s_sa = reinterpret_cast<int*>(s_acc + (2 - PG) * L * TJ);
  int* s_sb = s_sa + L;
  int* s_ss = s_sb + L;

  const TmTile tile = tiles[blockIdx.x];
  const int tid = threadIdx.x;
  const int sct = blockIdx.z;
  const bool live = tid < tile.tgt_count;
  const int j = tile.tgt_start + (live ? tid : tile.tgt_count - 1);
  const double xj = pos[3 * j], yj = pos[3 * j + 1], zj = pos[3 * j + 2];
  const int per = (tile.src_count + gridDim.y - 1) / gridDim.y;
  const int c0 = tile.src_start + blockIdx.y * per;
  const int c1 = min(tile.src_start + tile.src_count, c0 + per);

  for (int e = tid; e < L; e += TJ) {
    int a, b, sg;
    if (sct == 0) R3dPair<R, LMAX, 0>::stage_entry(e, a, b, sg); else R3dPair<R, LMAX, 1>::stage_entry(e, a, b, sg);
    s_sa[e] = a; s_sb[e] = b; s_ss[e] = sg;
  }
  R* sr = s_scr + tid;
  R* si = s_scr + NS * TJ + tid;
  R* ar = s_acc + tid;
  R* ai = s_acc + NS * TJ + tid;
  R* pr = s_acc + L * TJ + tid;
  R* pi = s_acc + (L + NS) * TJ + tid;
  if (PG >= 1) {
    const size_t blk = ((size_t)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
    pr = g_pacc + blk * (size_t)(PG * L * TJ) + tid;
    pi = pr + NS * TJ;
    if (PG >= 2) { ar = pr + L * TJ; ai = ar + NS * TJ; }
  }
#pragma unroll
  for (int b = 0; b < NS; ++b) { ar[b * TJ] = R(0); ai[b * TJ] = R(0); pr[b * TJ] = R(0); pi[b * TJ] = R(0); }

  for (int s0 = c0; s0 < c1; s0 += SS) {
    const int ns = min(SS, c1 - s0);
    __syncthreads();
    for (int e = tid; e < ns; e += TJ) {
      s_px[e] = pos[3 * (s0 + e)]; s_py[e] = pos[3 * (s0 + e) + 1]; s_pz[e] = pos[3 * (s0 + e) + 2];
    }
    for (int e = tid; e < ns * L; e += TJ) {
      const int src = e / L, kk = e - src * L;
      const Cx<R>* xrow = x + (size_t)(s0 + src) * L;
      const int ia = s_sa[kk], sg = s_ss[kk];
      Cx<R> v = xrow[ia];
      if (sg != 0) {
        const Cx<R> o = xrow[s_sb[kk]];
        v = sg > 0 ? cadd(v, o) : csub(v, o);
      }
      if (ia >= NS) v = cx<R>(-v.im, v.re);            // tilde basis: multiply p = 1 modes by i
      s_x[2 * e] = v.re;
      s_x[2 * e + 1] = v.im;
    }
    __syncthreads();
#pragma unroll 1
    for (int s = 0; s < ns; ++s) {
      const double dx = xj - s_px[s], dy = yj - s_py[s], dz = zj - s_pz[s];   // d = x_dest - x_source (reading R3)
      const double rho2 = dx * dx + dy * dy, r2 = rho2 + dz * dz;
      const double rinv = r2 > 0.0 ? rsqrt(r2) : 0.0;                          // self pair -> h_q = 0 -> nothing  [rot3d]
      const double rhoinv = rho2 > 0.0 ? rsqrt(rho2) : 0.0;
      const double r = r2 * rinv;
      const R cph = rho2 > 0.0 ? (R)(dx * rhoinv) : R(1), sph = (R)(dy * rhoinv);         // azimuth of d (pair along z: phi := 0)
      const R cth = r2 > 0.0 ? (R)(dz * rinv) : R(1), sth = (R)(rho2 * rhoinv * rinv);     // polar angle of d
      R ck, sk;
      phase_kr<R>(k_over_pi, r, ck, sk);
      R hr[NQ], hi[NQ];
      hankel_up<R, NQ>((R)(rinv * inv_k), ck, sk, hr, hi);
      const R* xs = &s_x[s * L * 2];
      if (sct == 0) R3dPair<R, LMAX, 0>::template run<TJ>(xs, cph, sph, cth, sth, hr, hi, sr, si, ar, ai, pr, pi);
      else          R3dPair<R, LMAX, 1>::template run<TJ>(xs, cph, sph, cth, sth, hr, hi, sr, si, ar, ai, pr, pi);
    }
  }
  if (live) {
    Cx<R>* out = u_part + ((size_t)(blockIdx.y * 2 + sct) * n_scat + j) * L;
    if (sct == 0) R3dPair<R, LMAX, 0>::template unmix<TJ>(ar, ai, pr, pi, out);
    else          R3dPair<R, LMAX, 1>::template unmix<TJ>(ar, ai, pr, pi, out);
  }
}

#endif  // TM_SEC_ROT3D
#ifdef TM_SEC_ROT3DW
// ---------------------------------------------------------------------------------------------------
// Rotation-based 3-D kernel, WARP-SPLIT (lmax 4..6; gen_tables.py: emit_rot3d_ws).  Block = 4 warps x 32 targets: lane = target.
// A round handles 4 sources: warp g runs phases A + B (into the pair-axis frame, axial translation) - the SAME straight-line code
// in all warps, so the instruction stream is shared - for source s + g of its lane's target and leaves t in ITS scratch vector
// [slot][lane]; block barrier; warp g then runs phase C (back into the pair-azimuth frame, accumulation) of the (l, p) blocks it
// OWNS for each of the 4 sources, into REGISTER accumulators (n / 4 slots, own sector + partner share); block barrier.
// The pair angles travel with t (4 values per lane and source in shared memory).
#ifndef TM_PIN
__device__ __forceinline__ void tm_pin(double& v) { asm volatile("" : "+d"(v)); }
__device__ __forceinline__ void tm_pin(float& v) { asm volatile("" : "+f"(v)); }
#define TM_PIN(v) tm_pin(v)
#endif
#include "generated/tm_rot3d_ws_gen.cuh"

template <int LMAX, int S> struct R3wTab;
#define TM_R3W_TAB(LM, SS_)                                                                               \
  template <> struct R3wTab<LM, SS_> {                                                                    \
    static __device__ __forceinline__ void entry(int k, int& a, int& b, int& sg) {                        \
      a = tm_r3w_sa_L##LM##_S##SS_[k]; b = tm_r3w_sb_L##LM##_S##SS_[k]; sg = tm_r3w_ss_L##LM##_S##SS_[k]; \
    }                                                                                                     \
  };
TM_R3W_TAB(4, 0) TM_R3W_TAB(4, 1) TM_R3W_TAB(5, 0) TM_R3W_TAB(5, 1) TM_R3W_TAB(6, 0) TM_R3W_TAB(6, 1)
#undef TM_R3W_TAB

template <typename R, int LMAX, int S> struct R3wSec;
#define TM_R3W_SEC(LM, SS_)                                                                               \
  template <typename R> struct R3wSec<R, LM, SS_> {                                                       \
    template <int AS> static __device__ __forceinline__ void A(const R* xs, R cph, R sph, R cth, R sth, R* wr, R* wi) { \
      tm_r3w_A_L##LM##_S##SS_<R, AS>(xs, cph, sph, cth, sth, wr, wi);                                     \
    }                                                                                                     \
    template <int AS> static __device__ __forceinline__ void B(R* hr, R* hi, R* wr, R* wi) {              \
      tm_r3w_B_L##LM##_S##SS_<R, AS>(hr, hi, wr, wi, wr, wi);                                             \
    }                                                                                                     \
  };
TM_R3W_SEC(4, 0) TM_R3W_SEC(4, 1) TM_R3W_SEC(5, 0) TM_R3W_SEC(5, 1) TM_R3W_SEC(6, 0) TM_R3W_SEC(6, 1)
#undef TM_R3W_SEC
template <typename R, int LMAX, int S, int P> struct R3wPart;
#define TM_R3W_SPEC(LM, SS_, PP)                                                                          \
  template <typename R> struct R3wPart<R, LM, SS_, PP> {                                                  \
    template <int AS> static __device__ __forceinline__ void Cc(R cph, R sph, R cth, R sth, const R* tr, const R* ti, \
                                                                R* ar, R* ai, R* pr, R* pi) {             \
      tm_r3w_C_L##LM##_S##SS_##_P##PP<R, AS>(cph, sph, cth, sth, tr, ti, ar, ai, pr, pi);                 \
    }                                                                                                     \
    static __device__ __forceinline__ void unmix(const R* ar, const R* ai, const R* pr, const R* pi, Cx<R>* out) { \
      tm_r3w_unmix_L##LM##_S##SS_##_P##PP<R, Cx<R>>(ar, ai, pr, pi, out);                                 \
    }                                                                                                     \
  };
#define TM_R3W_SPEC_S(LM, SS_) TM_R3W_SPEC(LM, SS_, 0) TM_R3W_SPEC(LM, SS_, 1) TM_R3W_SPEC(LM, SS_, 2) TM_R3W_SPEC(LM, SS_, 3)
TM_R3W_SPEC_S(4, 0) TM_R3W_SPEC_S(4, 1) TM_R3W_SPEC_S(5, 0) TM_R3W_SPEC_S(5, 1) TM_R3W_SPEC_S(6, 0) TM_R3W_SPEC_S(6, 1)
#undef TM_R3W_SPEC_S
#undef TM_R3W_SPEC
template <int LMAX> struct R3wMax;
template <> struct R3wMax<4> { static constexpr int nsl = TM_R3W_NSLMAX_L4; };
template <> struct R3wMax<5> { static constexpr int nsl = TM_R3W_NSLMAX_L5; };
template <> struct R3wMax<6> { static constexpr int nsl = TM_R3W_NSLMAX_L6; };

template <typename R, int LMAX, int SS> struct Rot3dWsSmem {
  static constexpr int L = 2 * LMAX * (LMAX + 2);
  // positions | staged d-values (own + partner = L slots per source) | 4 scratch vectors ([re/im][L/2 slots][32 lanes], one per warp) |
  // pair angles [warp][4][32 lanes] | staging tables
  static constexpr size_t bytes = sizeof(double) * 3 * SS + sizeof(R) * (size_t)(SS * L * 2 + 4 * L * 32 + 4 * 4 * 32) + sizeof(int) * 3 * L;
};

// one sector (compile time) of the warp-split kernel; `warp` selects the part at run time (warp-uniform branch)
template <typename R, int LMAX, int S, int SS>
__device__ __forceinline__ void rot3d_ws_sector(const double* __restrict__ pos, const Cx<R>* __restrict__ x, Cx<R>* __restrict__ u_part,
                                                const TmTile tile, int n_scat, double k_over_pi, double inv_k, unsigned char* smem_raw) {
  constexpr int L = 2 * LMAX * (LMAX + 2), NS = L / 2, NQ = 2 * LMAX + 1, TJ = 32, NT = 128, NSL = R3wMax<LMAX>::nsl;
  double* s_px = reinterpret_cast<double*>(smem_raw);
  double* s_py = s_px + SS;
  double* s_pz = s_py + SS;
  R* s_x = reinterpret_cast<R*>(s_pz + SS);          // [source][2 NS] complex: own slots then partner slots
  R* s_scr = s_x + SS * L * 2;                       // [warp][re/im][NS][TJ]: t of the warp's source of the round
  R* s_ang = s_scr + 4 * L * TJ;                     // [warp][4][TJ]: cos / sin of the pair's azimuth and polar angle
  int* s_sa = reinterpret_cast<int*>(s_ang + 4 * 4 * TJ);
  int* s_sb = s_sa + L;
  int* s_ss = s_sb + L;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const bool live = lane < tile.tgt_count;
  const int j = tile.tgt_start + (live ? lane : tile.tgt_count - 1);
  const double xj = pos[3 * j], yj = pos[3 * j + 1], zj = pos[3 * j + 2];
  const int per = (tile.src_count + gridDim.y - 1) / gridDim.y;
  const int c0 = tile.src_start + blockIdx.y * per;
  const int c1 = min(tile.src_start + tile.src_count, c0 + per);
  for (int e = tid; e < L; e += NT) {
    int a, b, sg;
    R3wTab<LMAX, S>::entry(e, a, b, sg);
    s_sa[e] = a; s_sb[e] = b; s_ss[e] = sg;
  }
  R* wr = s_scr + (size_t)warp * L * TJ + lane;      // this warp's scratch vector
  R* wi = wr + NS * TJ;
  R ar[NSL], ai[NSL], pr[NSL], pi[NSL];
#pragma unroll
  for (int q = 0; q < NSL; ++q) { ar[q] = R(0); ai[q] = R(0); pr[q] = R(0); pi[q] = R(0); }

  for (int s0 = c0; s0 < c1; s0 += SS) {
    const int ns = min(SS, c1 - s0);
    __syncthreads();                                   // previous stage consumed (also orders the staging tables)
    for (int e = tid; e < ns; e += NT) {
      s_px[e] = pos[3 * (s0 + e)]; s_py[e] = pos[3 * (s0 + e) + 1]; s_pz[e] = pos[3 * (s0 + e) + 2];
    }
    for (int e = tid; e < ns * L; e += NT) {
      const int src = e / L, kk = e - src * L;
      const Cx<R>* xrow = x + (size_t)(s0 + src) * L;
      const int ia = s_sa[kk], sg = s_ss[kk];
      Cx<R> v = xrow[ia];
      if (sg != 0) {
        const Cx<R> o = xrow[s_sb[kk]];
        v = sg > 0 ? cadd(v, o) : csub(v, o);
      }
      if (ia >= NS) v = cx<R>(-v.im, v.re);            // tilde basis: multiply p = 1 modes by i
      s_x[2 * e] = v.re;
      s_x[2 * e + 1] = v.im;
    }
    __syncthreads();
#pragma unroll 1
    for (int s = 0; s < ns; s += 4) {
      const int sg = s + warp;                       // this warp's source of the round
      if (sg < ns) {
        const double dx = xj - s_px[sg], dy = yj - s_py[sg], dz = zj - s_pz[sg];   // d = x_dest - x_source (reading R3)
        const double rho2 = dx * dx + dy * dy, r2 = rho2 + dz * dz;
        const double rinv = r2 > 0.0 ? rsqrt(r2) : 0.0;                            // self pair -> h_q = 0 -> t = 0
        const double rhoinv = rho2 > 0.0 ? rsqrt(rho2) : 0.0;
        const double r = r2 * rinv;
        const R cph = rho2 > 0.0 ? (R)(dx * rhoinv) : R(1), sph = (R)(dy * rhoinv);
        const R cth = r2 > 0.0 ? (R)(dz * rinv) : R(1), sth = (R)(rho2 * rhoinv * rinv);
        R* ang = s_ang + (size_t)warp * 4 * TJ + lane;
        ang[0] = cph; ang[TJ] = sph; ang[2 * TJ] = cth; ang[3 * TJ] = sth;
        R3wSec<R, LMAX, S>::template A<TJ>(&s_x[sg * L * 2], cph, sph, cth, sth, wr, wi);
        R ck, sk;
        phase_kr<R>(k_over_pi, r, ck, sk);
        R hr[NQ], hi[NQ];
        hankel_up<R, NQ>((R)(rinv * inv_k), ck, sk, hr, hi);
        R3wSec<R, LMAX, S>::template B<TJ>(hr, hi, wr, wi);
      }
      __syncthreads();                               // the round's t vectors are complete
      const int nq = min(4, ns - s);
#pragma unroll 1
      for (int q = 0; q < nq; ++q) {
        const R* ang = s_ang + (size_t)q * 4 * TJ + lane;
        const R cph = ang[0], sph = ang[TJ], cth = ang[2 * TJ], sth = ang[3 * TJ];
        const R* tr = s_scr + (size_t)q * L * TJ + lane;
        const R* ti = tr + NS * TJ;
        switch (warp) {
          case 0: R3wPart<R, LMAX, S, 0>::template Cc<TJ>(cph, sph, cth, sth, tr, ti, ar, ai, pr, pi); break;
          case 1: R3wPart<R, LMAX, S, 1>::template Cc<TJ>(cph, sph, cth, sth, tr, ti, ar, ai, pr, pi); break;
          case 2: R3wPart<R, LMAX, S, 2>::template Cc<TJ>(cph, sph, cth, sth, tr, ti, ar, ai, pr, pi); break;
          default: R3wPart<R, LMAX, S, 3>::template Cc<TJ>(cph, sph, cth, sth, tr, ti, ar, ai, pr, pi); break;
        }
      }
      __syncthreads();                               // every owner has consumed the round before the scratch is rewritten
    }
  }
  if (live) {
    Cx<R>* out = u_part + ((size_t)(blockIdx.y * 2 + S) * n_scat + j) * L;
    switch (warp) {
      case 0: R3wPart<R, LMAX, S, 0>::unmix(ar, ai, pr, pi, out); break;
      case 1: R3wPart<R, LMAX, S, 1>::unmix(ar, ai, pr, pi, out); break;
      case 2: R3wPart<R, LMAX, S, 2>::unmix(ar, ai, pr, pi, out); break;
      default: R3wPart<R, LMAX, S, 3>::unmix(ar, ai, pr, pi, out); break;
    }
  }
}

#ifndef TM_R3W_MINBLOCKS
#define TM_R3W_MINBLOCKS 2
#endif
template <typename R, int LMAX, int SS>
__global__ void __launch_bounds__(128, TM_R3W_MINBLOCKS)
k_allpairs_rot3d_ws(const double* __restrict__ pos, const Cx<R>* __restrict__ x, Cx<R>* __restrict__ u_part,
                    const TmTile* __restrict__ tiles, int n_scat, double k_over_pi, double inv_k,
                    const int* __restrict__ n_active) {
  if (n_active != nullptr && *n_active == 0) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const TmTile tile = tiles[blockIdx.x];
  if (blockIdx.z == 0) rot3d_ws_sector<R, LMAX, 0, SS>(pos, x, u_part, tile, n_scat, k_over_pi, inv_k, smem_raw);
  else                 rot3d_ws_sector<R, LMAX, 1, SS>(pos, x, u_part, tile, n_scat, k_over_pi, inv_k, smem_raw);
}
#endif  // TM_SEC_ROT3DW
#ifdef TM_SEC_COP4
// ---------------------------------------------------------------------------------------------------
// Coplanar kernel for lmax 4..6 (the paper's truncation is lmax = 6).  Same mathematics as
// k_allpairs_coplanar, but the two mirrors split the operator into FOUR uncoupled sectors (blockIdx.z = 2 h + t,
// slowest grid dimension), the accumulators (own sector + the partner sector's share from the output rotation) live in
// shared memory [slot][thread], and only the sector's own x^new (<= 24 complex at lmax 6) and h_q stay in registers.
// At lmax 6 a sector's straight-line code is ~120 KB, far beyond the instruction caches: the kernel is
// instruction-fetch bound there, still an order of magnitude ahead of the table-driven kernel.
// Phase barriers inside the generated pair code (gen_tables.py: emit_axial_core): bit k of TM_COP4_SYNC_L<lmax> enables
// barrier k.  All threads of a block run the same straight-line code with a uniform trip count, so the barriers are legal.
#ifndef TM_COP4_SYNC_L4
#define TM_COP4_SYNC_L4 0
#endif
#ifndef TM_COP4_SYNC_L5
#define TM_COP4_SYNC_L5 0
#endif
#ifndef TM_COP4_SYNC_L6
#define TM_COP4_SYNC_L6 0
#endif
#ifndef TM_COP4_SYNC_L7
#define TM_COP4_SYNC_L7 0
#endif
#define TM_PHASE_SYNC(lmax, k) do { if ((TM_COP4_SYNC_L##lmax >> (k)) & 1) __syncthreads(); } while (0)
#include "generated/tm_coplanar4_gen.cuh"

template <typename R, int LMAX, int Z, int G> struct Cop4;
#define TM_COP4_SPEC(LM, ZZ, GG)                                                                         \
  template <typename R> struct Cop4<R, LM, ZZ, GG> {                                                     \
    static constexpr int n = TM_COP4_N_L##LM##_Z##ZZ;                                                    \
    static constexpr int nr = TM_COP4_NR_L##LM##_Z##ZZ##_G##GG;                                          \
    template <int AS>                                                                                    \
    static __device__ __forceinline__ void run(const R* xs, const R* cm, const R* sm, const R* hr,       \
                                               const R* hi, R* ar, R* ai) {                              \
      tm_cop4_pair_L##LM##_Z##ZZ##_G##GG<R, AS>(xs, cm, sm, hr, hi, ar, ai);                             \
    }                                                                                                    \
    template <int AS>                                                                                    \
    static __device__ __forceinline__ void unmix(const R* ar, const R* ai, Cx<R>* out) {                 \
      tm_cop4_unmix_L##LM##_Z##ZZ##_G##GG<R, Cx<R>, AS>(ar, ai, out);                                    \
    }                                                                                                    \
    static __device__ __forceinline__ void stage_entry(int k, int& a, int& b, int& sg) {                 \
      a = tm_cop4_sa_L##LM##_Z##ZZ[k]; b = tm_cop4_sb_L##LM##_Z##ZZ[k]; sg = tm_cop4_ss_L##LM##_Z##ZZ[k]; \
    }                                                                                                    \
  };
#define TM_COP4_SPEC_Z(LM, GG) TM_COP4_SPEC(LM, 0, GG) TM_COP4_SPEC(LM, 1, GG) TM_COP4_SPEC(LM, 2, GG) TM_COP4_SPEC(LM, 3, GG)
#define TM_COP4_SPEC_L(LM)                                                            \
  TM_COP4_SPEC_Z(LM, 0) TM_COP4_SPEC_G2(LM) TM_COP4_SPEC_G4(LM) TM_COP4_SPEC_G8(LM)
#define TM_COP4_SPEC_G2(LM) TM_COP4_IF2_L##LM(TM_COP4_SPEC_Z(LM, 1))
#define TM_COP4_SPEC_G4(LM) TM_COP4_IF4_L##LM(TM_COP4_SPEC_Z(LM, 2) TM_COP4_SPEC_Z(LM, 3))
#define TM_COP4_SPEC_G8(LM) TM_COP4_IF8_L##LM(TM_COP4_SPEC_Z(LM, 4) TM_COP4_SPEC_Z(LM, 5) TM_COP4_SPEC_Z(LM, 6) TM_COP4_SPEC_Z(LM, 7))
TM_COP4_SPEC_L(4) TM_COP4_SPEC_L(5) TM_COP4_SPEC_L(6) TM_COP4_SPEC_L(7)
#undef TM_COP4_SPEC_L
#undef TM_COP4_SPEC_Z
#undef TM_COP4_SPEC

template <int LMAX> struct Cop4Max;      // n: slots of the largest sector; nr: rows of the largest row group; ng: row groups per sector
template <> struct Cop4Max<4> { static constexpr int n = TM_COP4_NMAX_L4, nr = TM_COP4_NRMAX_L4, ng = TM_COP4_G_L4; };
template <> struct Cop4Max<5> { static constexpr int n = TM_COP4_NMAX_L5, nr = TM_COP4_NRMAX_L5, ng = TM_COP4_G_L5; };
template <> struct Cop4Max<6> { static constexpr int n = TM_COP4_NMAX_L6, nr = TM_COP4_NRMAX_L6, ng = TM_COP4_G_L6; };
template <> struct Cop4Max<7> { static constexpr int n = TM_COP4_NMAX_L7, nr = TM_COP4_NRMAX_L7, ng = TM_COP4_G_L7; };

template <typename R, int LMAX, int TJ, int SS> struct Cop4Smem {
  static constexpr int NM = Cop4Max<LMAX>::n;
  static constexpr int NR = Cop4Max<LMAX>::nr;
  static constexpr size_t bytes = sizeof(double) * 2 * SS + sizeof(R) * (size_t)(SS * 2 * NM * 2 + 2 * 2 * NR * TJ) + sizeof(int) * 3 * 2 * NM;
};

template <typename R, int LMAX, int Z, int G, int TJ, int SS>
__device__ __forceinline__ void cop4_sector(const double* __restrict__ pos, const Cx<R>* __restrict__ x, Cx<R>* __restrict__ u_part,
                                            const TmTile tile, int n_scat, double k_over_pi, double inv_k, TmShift shift,
                                            unsigned char* smem_raw) {
  using S = Cop4<R, LMAX, Z, G>;
  constexpr int L = 2 * LMAX * (LMAX + 2);
  constexpr int NQ = 2 * LMAX + 1;
  constexpr int NM = Cop4Max<LMAX>::n;
  constexpr int NR = Cop4Max<LMAX>::nr;
  constexpr int n = S::n;
  constexpr int nr = S::nr;
  double* s_px = reinterpret_cast<double*>(smem_raw);
  double* s_py = s_px + SS;
  R* s_x = reinterpret_cast<R*>(s_py + SS);          // [source][2 n] complex: own slots then partner slots
  R* s_acc = s_x + SS * 2 * NM * 2;                  // [re/im][2 nr][TJ]: the group's own rows, then their partner share
  int* s_sa = reinterpret_cast<int*>(s_acc + 2 * 2 * NR * TJ);
  int* s_sb = s_sa + 2 * NM;
  int* s_ss = s_sb + 2 * NM;
  const int tid = threadIdx.x;
  const bool live = tid < tile.tgt_count;
  const int j = tile.tgt_start + (live ? tid : tile.tgt_count - 1);
  const double xj = pos[3 * j] + shift.x, yj = pos[3 * j + 1] + shift.y;
  const int per = (tile.src_count + gridDim.y - 1) / gridDim.y;
  const int c0 = tile.src_start + blockIdx.y * per;
  const int c1 = min(tile.src_start + tile.src_count, c0 + per);
  if (tid < 2 * n) {
    int a, b, sg;
    S::stage_entry(tid, a, b, sg);
    s_sa[tid] = a; s_sb[tid] = b; s_ss[tid] = sg;
  }
  R* ar = s_acc + tid;
  R* ai = s_acc + 2 * NR * TJ + tid;
#pragma unroll
  for (int b = 0; b < 2 * nr; ++b) { ar[b * TJ] = R(0); ai[b * TJ] = R(0); }
  for (int s0 = c0; s0 < c1; s0 += SS) {
    const int ns = min(SS, c1 - s0);
    __syncthreads();
    for (int e = tid; e < ns; e += TJ) { s_px[e] = pos[3 * (s0 + e)]; s_py[e] = pos[3 * (s0 + e) + 1]; }
    for (int e = tid; e < ns * 2 * n; e += TJ) {
      const int src = e / (2 * n), kk = e - src * 2 * n;
      const Cx<R>* xrow = x + (size_t)(s0 + src) * L;
      const int ia = s_sa[kk], sg = s_ss[kk];
      Cx<R> v = xrow[ia];
      if (sg != 0) {
        const Cx<R> o = xrow[s_sb[kk]];
        v = sg > 0 ? cadd(v, o) : csub(v, o);
      }
      if (ia >= L / 2) v = cx<R>(-v.im, v.re);         // tilde basis: multiply p = 1 modes by i
      s_x[2 * e] = v.re;
      s_x[2 * e + 1] = v.im;
    }
    __syncthreads();
#pragma unroll 1
    for (int s = 0; s < ns; ++s) {
      const double dx = xj - s_px[s], dy = yj - s_py[s];
      const double r2 = dx * dx + dy * dy;
      const double rinv = (r2 > 0.0 && !(shift.on && s0 + s == j)) ? rsqrt(r2) : 0.0;
      const double r = r2 * rinv;
      R cm[LMAX + 1], sm[LMAX + 1];
      cm[0] = R(1); sm[0] = R(0);
      cm[1] = r2 > 0.0 ? (R)(dx * rinv) : R(1); sm[1] = (R)(dy * rinv);
#pragma unroll
      for (int m = 2; m <= LMAX; ++m) {
        cm[m] = cm[m - 1] * cm[1] - sm[m - 1] * sm[1];
        sm[m] = sm[m - 1] * cm[1] + cm[m - 1] * sm[1];
      }
      R ck, sk;
      phase_kr<R>(k_over_pi, r, ck, sk);
      R hr[NQ], hi[NQ];
      hankel_up<R, NQ>((R)(rinv * inv_k), ck, sk, hr, hi);
      S::template run<TJ>(&s_x[s * 2 * n * 2], cm, sm, hr, hi, ar, ai);
      // lmax 5 only: the warps of a block stay within one pass of the sector's code and share its instruction fetches
      // (measured 4.41 -> 4.04 ms; lmax 4: 2.10 -> 2.17, lmax 6: 6.76 -> 6.78, so not there)
      if constexpr (LMAX == 5) __syncthreads();
    }
  }
  if (live) {
    Cx<R>* out = u_part + ((size_t)(blockIdx.y * 2 + (Z & 1)) * n_scat + j) * L;
    S::template unmix<TJ>(ar, ai, out);
  }
}

// blockIdx.z = z * NG + g (sector-major, slowest grid dimension: co-resident blocks run the same code)
template <typename R, int LMAX, int ZG, int TJ, int SS>
__device__ __forceinline__ void cop4_dispatch(const double* __restrict__ pos, const Cx<R>* __restrict__ x, Cx<R>* __restrict__ u_part,
                                              const TmTile tile, int n_scat, double k_over_pi, double inv_k, TmShift shift,
                                              unsigned char* smem_raw) {
  constexpr int NG = Cop4Max<LMAX>::ng;
  if (blockIdx.z == ZG) cop4_sector<R, LMAX, ZG / NG, ZG % NG, TJ, SS>(pos, x, u_part, tile, n_scat, k_over_pi, inv_k, shift, smem_raw);
  else if constexpr (ZG + 1 < 4 * NG) cop4_dispatch<R, LMAX, ZG + 1, TJ, SS>(pos, x, u_part, tile, n_scat, k_over_pi, inv_k, shift, smem_raw);
}

template <typename R, int LMAX, int TJ, int SS>
__global__ void __launch_bounds__(TJ)
k_allpairs_coplanar4(const double* __restrict__ pos, const Cx<R>* __restrict__ x, Cx<R>* __restrict__ u_part,
                     const TmTile* __restrict__ tiles, int n_scat, double k_over_pi, double inv_k,
                     const int* __restrict__ n_active, TmShift shift) {
  if (n_active != nullptr && *n_active == 0) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const TmTile tile = tiles[blockIdx.x];
  cop4_dispatch<R, LMAX, 0, TJ, SS>(pos, x, u_part, tile, n_scat, k_over_pi, inv_k, shift, smem_raw);
}
#endif  // TM_SEC_COP4
