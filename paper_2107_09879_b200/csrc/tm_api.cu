// libtm: C-ABI entry points (include/tm.h) and host orchestration.  sm_100a only, no CPU fallback.
#include "../../include/tm.h"

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <type_traits>
#include <unordered_map>
#include <vector>

#include "tm_launch.h"
#include "tm_arnoldi.cuh"
#include "tm_common.cuh"
#include "tm_fields.cuh"
#include "tm_gmres.cuh"
#include "tm_incident.cuh"
#include "tm_nullfield.cuh"
#include "tm_special.cuh"
#include "tm_ttable.cuh"
#include "tm_vecops.cuh"
#include "generated/tm_tables_gen.h"

namespace {

std::string g_create_error;

// Device memory comes from the device's stream-ordered pool with an unlimited release threshold: a context that is
// created and destroyed once per step (an optimisation loop, the end-to-end bench leg) gets the same physical memory
// back instead of paying the driver's map / unmap on every cudaMalloc / cudaFree (measured: 1-60 ms per call, at
// random).  tm_release_cached_memory() returns the cached memory to the driver.
// Debug aid (tm_debug_guards; compute-sanitizer is not available everywhere): with guards ON every block handed out below
// carries a 4 KiB margin of 0xA5 bytes on each side; the margins are compared when the block is freed and whenever
// tm_debug_guards is asked, so a kernel that writes outside ANY internal buffer (chunk partials, Krylov basis, tables,
// quadrature scratch, ...) is caught.  Off (the default) the allocator is exactly what it was.
constexpr size_t GUARD_BYTES = 4096;
struct GuardRegistry {
  std::mutex mu;
  bool on = false;
  std::unordered_map<void*, size_t> live;      // user pointer -> user bytes, guarded blocks only
  long long violations = 0, blocks = 0;
};
GuardRegistry& guards() { static GuardRegistry g; return g; }

// Number of margins of one block that no longer hold the sentinel (0, 1 or 2); the device is idle when this runs.
int guard_damage(void* user, size_t bytes) {
  static std::vector<unsigned char> h(2 * GUARD_BYTES);
  char* u = static_cast<char*>(user);
  if (cudaMemcpy(h.data(), u - GUARD_BYTES, GUARD_BYTES, cudaMemcpyDeviceToHost) != cudaSuccess ||
      cudaMemcpy(h.data() + GUARD_BYTES, u + bytes, GUARD_BYTES, cudaMemcpyDeviceToHost) != cudaSuccess) { cudaGetLastError(); return 2; }
  int bad = 0;
  for (int side = 0; side < 2; ++side)
    for (size_t i = 0; i < GUARD_BYTES; ++i)
      if (h[side * GUARD_BYTES + i] != 0xA5) { ++bad; break; }
  return bad;
}

template <typename T>
cudaError_t tm_dev_alloc(T** p, size_t bytes) {
  *p = nullptr;
  if (bytes == 0) return cudaSuccess;
  static bool pool_set[64] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev >= 0 && dev < 64 && !pool_set[dev]) {
    cudaMemPool_t pool;
    unsigned long long keep = ~0ULL;
    if ((e = cudaDeviceGetDefaultMemPool(&pool, dev)) != cudaSuccess) return e;
    if ((e = cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep)) != cudaSuccess) return e;
    pool_set[dev] = true;
  }
  GuardRegistry& g = guards();
  std::lock_guard<std::mutex> lock(g.mu);
  const size_t pad = g.on ? GUARD_BYTES : 0;
  void* q = nullptr;
  if ((e = cudaMallocAsync(&q, bytes + 2 * pad, (cudaStream_t)0)) != cudaSuccess) return e;
  if (pad) {
    char* c = static_cast<char*>(q);
    if ((e = cudaMemsetAsync(c, 0xA5, pad, (cudaStream_t)0)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(c + pad + bytes, 0xA5, pad, (cudaStream_t)0)) != cudaSuccess) return e;
    q = c + pad;
    g.live[q] = bytes;
    ++g.blocks;
  }
  *p = static_cast<T*>(q);
  return cudaStreamSynchronize((cudaStream_t)0);      // usable from any stream on return
}

// Like cudaFree: every kernel that may still use the block has finished before it goes back to the pool.
inline cudaError_t tm_dev_free(void* p) {
  if (!p) return cudaSuccess;
  cudaError_t e = cudaDeviceSynchronize();
  GuardRegistry& g = guards();
  std::lock_guard<std::mutex> lock(g.mu);
  const auto it = g.live.find(p);
  if (it != g.live.end()) {                          // a guarded block: check its margins, free from its true start
    g.violations += guard_damage(p, it->second);
    g.live.erase(it);
    p = static_cast<char*>(p) - GUARD_BYTES;
  }
  const cudaError_t f = cudaFreeAsync(p, (cudaStream_t)0);
  return e != cudaSuccess ? e : f;
}

constexpr int MAX_RESTART = 300;
static_assert(MAX_RESTART + 1 <= TM_MAX_LDH, "k_gmres_solve_y keeps y in shared memory");

struct Gmres {                   // device scalars of the Krylov solver, sized for `restart`
  int restart = 0;
  TmGmresDev dev{};
  double2* part = nullptr;       // [(restart+1)][n_chunks]
  double* normpart = nullptr;    // [n_chunks]
  void* blob = nullptr;
};

}  // namespace

struct tm_ctx {
  int n_scat = 0, n_win = 0, lmax = 0, L = 0, precision = TM_FP64;
  double k = 0.0;
  size_t n = 0;                  // n_scat * L
  cudaStream_t stream = nullptr;
  std::vector<int> win_ptr;
  bool coplanar = false;
  int kernel_req = TM_KERNEL_AUTO, kernel = TM_KERNEL_GENERAL;
  TmShift shift{0.0, 0.0, 0.0, 0};      // target displacement (unused by the library: kept for A/B experiments)
  tm_ctx* grad_aux = nullptr;           // tm_grad_positions: the same layout at lmax + 1 (all-pairs product A^ext)
  tm_ctx* multi_aux = nullptr;          // tm_solve_multi: the same geometry replicated as one set of windows per right-hand side
  int multi_rhs = 0; long long multi_T_version = -1;
  long long T_version = 0;              // bumped by tm_set_tmatrices
  void* d_grad_tab = nullptr; TmGradDev grad_tab{};
  int cop_tj = 128;                     // coplanar kernel: targets per block (-DTM_COP_TJ=256 for experiments)
  int cop_cl = 1;                       // coplanar kernel: cluster size along the chunk dimension (chunk partials reduced in DSMEM)

  double* d_pos = nullptr;
  std::vector<double> h_pos;      // host copy (quadrature sizing of the angular-spectrum sources)
  int* d_win_of = nullptr;
  int* d_type_of = nullptr;
  void* d_T = nullptr;           // Cx<R> [n_types][L] or [n_types][L][L]
  void* d_T32 = nullptr;         // TM_MIXED only: fp32 copy of T for the inner Krylov cycles
  int n_types = 0, diag = 1;
  bool has_T = false, has_inc = false;
  double2* d_p = nullptr;        // incident coefficients, fp64 [n]
  // description of the last tm_set_incident (for TM_FIELD_E_INC)
  int inc_kind = -1;
  double inc_kvec[3] = {0, 0, 0}; double2 inc_e0[3] = {};            // plane wave
  std::vector<double> inc_src; std::vector<double2> inc_amp;         // beams / jinc sources (all windows)
  double inc_kw = -1.0, inc_bmax = 0.0; int inc_nb = 0;
  TmConst* d_const = nullptr;
  TmConst h_const{};
  int* d_rowptr = nullptr; uint8_t* d_col = nullptr; uint8_t* d_widx = nullptr; uint8_t* d_imag = nullptr; double* d_coef = nullptr;

  TmTile* d_tiles = nullptr; int n_tiles = 0, n_chunk = 1, n_part = 1;   // n_part: partial-sum buffers the finishing kernel adds
  void* d_upart = nullptr; size_t upart_bytes = 0;
  void* d_pacc = nullptr; size_t pacc_bytes = 0;       // rotation-based 3-D kernel, lmax >= 6: partner accumulators [block][L][TJ]
  TmChunk* d_chunks = nullptr; int n_chunks = 0; int* d_win_chunk_ptr = nullptr;
  int ept = 4;                   // vector kernels: elements per thread (chunk = ept * TM_VT)
  int max_chunks_per_win = 0;

  void* d_v[3] = {nullptr, nullptr, nullptr};   // Cx<R> work vectors [n]: X, B, Z
  double2* d_io = nullptr;                      // fp64 staging [n]

  void* ws = nullptr; size_t ws_bytes = 0; bool ws_owned = false;
  Gmres gm;

  // One restart cycle (all-pairs + fused Arnoldi step, m times) as a CUDA graph: window-sized problems are launch-bound
  // (the paper's windows are ~31^2 scatterers).  Keyed on everything the captured launches bake in.
  struct CycleGraph {
    cudaGraphExec_t exec = nullptr;
    int transpose = -1, m = 0, rbytes = 0, n_part = 0, kernel = 0, launches = 0;
    double tol = 0.0;
    const void *ws = nullptr, *T = nullptr, *upart = nullptr, *blob = nullptr, *tiles = nullptr, *pacc = nullptr;
    int n_tiles = 0, n_chunk = 0, diag = -1;
  } cyc[2];
  bool graphs_ok = true;          // cleared when a capture fails (direct launches from then on)
  bool capturing = false;
  // side branch of the captured cycle: the Givens update of step j runs beside the all-pairs product of step j + 1
  cudaStream_t side = nullptr;
  cudaEvent_t fork_ev = nullptr, join_ev = nullptr;

  // timing of the all-pairs kernel
  bool time_kernels = false;
  std::vector<cudaEvent_t> ev;   // pairs
  size_t ev_used = 0;
  long long allpairs_launches = 0, total_launches = 0;

  // cached device scratch of the per-call paths (tm_set_incident, tm_fields): cudaMalloc / cudaFree synchronise the device and
  // occasionally take hundreds of ms on a busy host, so nothing on the per-step path allocates
  void* scratch[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  size_t scratch_cap[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  cudaEvent_t t0_ev = nullptr, t1_ev = nullptr;   // solve timing
  cudaEvent_t sync_ev = nullptr; // blocking-sync event: the host thread sleeps instead of spinning while the GPU works

  std::string err;
};

namespace {

int fail(tm_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg; else g_create_error = msg;
  return code;
}

#define TM_CUDA(call)                                                                       \
  do {                                                                                      \
    cudaError_t e_ = (call);                                                                \
    if (e_ != cudaSuccess)                                                                  \
      return fail(ctx, e_ == cudaErrorMemoryAllocation ? TM_E_NOMEM : TM_E_CUDA,            \
                  std::string(#call) + ": " + cudaGetErrorString(e_));                      \
  } while (0)

bool is_device_ptr(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

cudaError_t copy_in(void* dst_dev, const void* src, size_t bytes, cudaStream_t s) {
  return cudaMemcpyAsync(dst_dev, src, bytes, is_device_ptr(src) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s);
}
cudaError_t copy_out(void* dst, const void* src_dev, size_t bytes, cudaStream_t s) {
  return cudaMemcpyAsync(dst, src_dev, bytes, is_device_ptr(dst) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, s);
}

// bytes of one element of the context's main vectors / T: fp64 in TM_FP64 and TM_MIXED, fp32 in TM_FP32
// Wait for the context's stream without spinning (a spinning host thread burns the container's CPU quota during
// multi-second solves; seen as occasional 2-3x outlier steps on shared hosts).
// Device scratch slot `i` of at least `bytes` bytes (grown on demand, freed in tm_destroy).
cudaError_t scratch_get(tm_ctx* c, int i, size_t bytes, void** out) {
  if (c->scratch_cap[i] < bytes) {
    if (c->scratch[i]) tm_dev_free(c->scratch[i]);
    c->scratch[i] = nullptr; c->scratch_cap[i] = 0;
    const size_t cap = bytes + bytes / 4 + 256;
    cudaError_t e = tm_dev_alloc(&c->scratch[i], cap);
    if (e != cudaSuccess) return e;
    c->scratch_cap[i] = cap;
  }
  *out = c->scratch[i];
  return cudaSuccess;
}

cudaError_t stream_wait(tm_ctx* c) {
  if (c->sync_ev == nullptr) {
    cudaError_t e = cudaEventCreateWithFlags(&c->sync_ev, cudaEventBlockingSync | cudaEventDisableTiming);
    if (e != cudaSuccess) { c->sync_ev = nullptr; return cudaStreamSynchronize(c->stream); }
  }
  cudaError_t e = cudaEventRecord(c->sync_ev, c->stream);
  if (e != cudaSuccess) return e;
  return cudaEventSynchronize(c->sync_ev);
}

size_t elem_bytes(const tm_ctx* c) { return c->precision == TM_FP32 ? sizeof(Cx<float>) : sizeof(Cx<double>); }

// ---------------------------------------------------------------------------------------- host math
// Gauss-Legendre nodes/weights on [-1, 1] by Newton iteration on P_n.
void gauss_legendre(int n, std::vector<double>& x, std::vector<double>& w) {
  x.resize(n); w.resize(n);
  for (int i = 0; i < (n + 1) / 2; ++i) {
    double z = std::cos(M_PI * (i + 0.75) / (n + 0.5)), pp = 0.0;
    for (int it = 0; it < 100; ++it) {
      double p1 = 1.0, p2 = 0.0;
      for (int j = 1; j <= n; ++j) { const double p3 = p2; p2 = p1; p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j; }
      pp = n * (z * p1 - p2) / (z * z - 1.0);
      const double dz = p1 / pp;
      z -= dz;
      if (std::fabs(dz) < 1e-16) break;
    }
    // one more evaluation of P_n' at the converged root for the weight
    double p1 = 1.0, p2 = 0.0;
    for (int j = 1; j <= n; ++j) { const double p3 = p2; p2 = p1; p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j; }
    pp = n * (z * p1 - p2) / (z * z - 1.0);
    x[i] = -z; x[n - 1 - i] = z;
    w[i] = w[n - 1 - i] = 2.0 / ((1.0 - z * z) * pp * pp);
  }
}

typedef std::complex<double> cd;

// spherical Bessel j_0..j_lmax at complex z (Miller backward recurrence, normalised with j_0 or j_1)
void sph_jn_complex(int lmax, cd z, std::vector<cd>& j) {
  j.assign(lmax + 1, cd(0));
  if (std::abs(z) < 1e-12) { j[0] = 1.0; return; }
  const int N = lmax + 40 + (int)std::abs(z) * 2;
  std::vector<cd> f(N + 2, cd(0));
  f[N + 1] = 0.0; f[N] = 1e-280;
  for (int n = N; n >= 1; --n) {
    f[n - 1] = (2.0 * n + 1.0) / z * f[n] - f[n + 1];
    if (std::abs(f[n - 1]) > 1e200) for (int q = n - 1; q <= N; ++q) f[q] *= 1e-200;
  }
  const cd j0 = std::sin(z) / z, j1 = std::sin(z) / (z * z) - std::cos(z) / z;
  const cd sc = (std::abs(j0) >= std::abs(j1)) ? j0 / f[0] : j1 / f[1];
  for (int l = 0; l <= lmax; ++l) j[l] = f[l] * sc;
}

// spherical Neumann y_0..y_lmax at real x > 0 (upward recurrence, stable)
void sph_yn_real(int lmax, double x, std::vector<double>& y) {
  y.assign(lmax + 2, 0.0);
  y[0] = -std::cos(x) / x;
  y[1] = -std::cos(x) / (x * x) - std::sin(x) / x;
  for (int l = 1; l < lmax + 1; ++l) y[l + 1] = (2.0 * l + 1.0) / x * y[l] - y[l - 1];
}

}  // namespace

// ============================================================================================ typed launches
namespace {

template <typename R> Cx<R>* vec(tm_ctx* c, int i) { return reinterpret_cast<Cx<R>*>(c->d_v[i]); }
// T in precision R: in TM_MIXED the context holds an fp64 copy (d_T) and an fp32 copy (d_T32)
template <typename R> const Cx<R>* Tptr(const tm_ctx* c) {
  return reinterpret_cast<const Cx<R>*>((sizeof(R) == 4 && c->precision == TM_MIXED) ? c->d_T32 : c->d_T);
}

int grid_for(size_t n, int block) { return (int)std::min<size_t>((n + block - 1) / block, 148 * 32); }

void tick(tm_ctx* c, bool allpairs_begin) {
  if (!c->time_kernels || c->capturing) return;
  if (c->ev_used + 2 > c->ev.size()) return;
  if (allpairs_begin) cudaEventRecord(c->ev[c->ev_used], c->stream);
  else { cudaEventRecord(c->ev[c->ev_used + 1], c->stream); c->ev_used += 2; }
}

// u_part <- A x   (all chunks)
template <typename R>
cudaError_t launch_allpairs(tm_ctx* c, const Cx<R>* x, const int* n_active) {
  Cx<R>* up = reinterpret_cast<Cx<R>*>(c->d_upart);
  const TmLaunch a{c->d_pos, c->d_tiles, c->n_scat, c->k / M_PI, 1.0 / c->k, n_active, c->stream, dim3(c->n_tiles, c->n_chunk), c->lmax};
  tick(c, true);
  cudaError_t e;
  if (c->kernel == TM_KERNEL_COPLANAR && c->lmax > 3)
    e = c->lmax <= 5 ? tm_launch_coplanar4_lo<R>(a, x, up, c->shift) : tm_launch_coplanar4_hi<R>(a, x, up, c->shift);
  else if (c->kernel == TM_KERNEL_COPLANAR) e = tm_launch_coplanar<R>(a, x, up, c->cop_tj, c->cop_cl, c->shift);
  else if (c->kernel == TM_KERNEL_ROT3D) {
    R* pacc = reinterpret_cast<R*>(c->d_pacc);
    if (tm_rot3d_ws(c->lmax)) e = tm_launch_rot3d_ws<R>(a, x, up);
    else e = c->lmax <= 5 ? tm_launch_rot3d_lo<R>(a, x, up, pacc) : (c->lmax == 6 ? tm_launch_rot3d_6<R>(a, x, up, pacc) : tm_launch_rot3d_7<R>(a, x, up, pacc));
  } else if (c->kernel == TM_KERNEL_SYM3D) e = tm_launch_sym3d<R>(a, x, up, c->shift);
  else e = tm_launch_general<R>(a, x, up, c->d_const, TmTermsDev{c->d_rowptr, c->d_col, c->d_widx, c->d_imag, c->d_coef});
  tick(c, false);
  c->allpairs_launches++; c->total_launches++;
  return e;
}

template <typename R>
cudaError_t launch_tapply(tm_ctx* c, int mode, const Cx<R>* x, Cx<R>* y, const int* n_active) {
  constexpr int JB = 8;
  const int grid = (c->n_scat + JB - 1) / JB;
  k_tapply<R, JB><<<grid, 256, 0, c->stream>>>(mode, c->L, c->n_scat, c->n_part, x, reinterpret_cast<Cx<R>*>(c->d_upart), y,
                                               Tptr<R>(c), c->diag, c->d_type_of, c->d_const, n_active);
  c->total_launches++;
  return cudaGetLastError();
}

// y = op(x): transpose 0: (I - T A) x; 1: (I - T A)^T x; 2: A x.   z = scratch vector for the transposed pre-step.
template <typename R>
cudaError_t apply_operator(tm_ctx* c, int transpose, const Cx<R>* x, Cx<R>* y, Cx<R>* z, const int* n_active) {
  cudaError_t e;
  if (transpose == 1) {
    if ((e = launch_tapply<R>(c, 4, x, z, n_active)) != cudaSuccess) return e;       // z = P T^T x
    if ((e = launch_allpairs<R>(c, z, n_active)) != cudaSuccess) return e;           // u = A z
    return launch_tapply<R>(c, 1, x, y, n_active);                                    // y = x - P u
  }
  if ((e = launch_allpairs<R>(c, x, n_active)) != cudaSuccess) return e;
  return launch_tapply<R>(c, transpose == 2 ? 2 : 0, x, y, n_active);
}

template <typename R>
cudaError_t load_c64(tm_ctx* c, const tm_c64* src, Cx<R>* dst) {     // host/device fp64 -> device Cx<R>
  cudaError_t e = copy_in(c->d_io, src, c->n * sizeof(double2), c->stream);
  if (e != cudaSuccess) return e;
  k_from_c64<R><<<grid_for(c->n, 256), 256, 0, c->stream>>>(reinterpret_cast<const double*>(c->d_io), dst, c->n);
  c->total_launches++;
  return cudaGetLastError();
}
template <typename R>
cudaError_t store_c64(tm_ctx* c, const Cx<R>* src, tm_c64* dst) {
  k_to_c64<R><<<grid_for(c->n, 256), 256, 0, c->stream>>>(src, reinterpret_cast<double*>(c->d_io), c->n);
  c->total_launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  return copy_out(dst, c->d_io, c->n * sizeof(double2), c->stream);
}

// ---------------------------------------------------------------------------------------- GMRES driver
// R  = precision of the Krylov cycles (all-pairs kernel, basis V, work vector W, orthogonalisation),
// RX = precision of the iterate x, the right-hand side b and the TRUE residual recomputed at every restart.
// R == RX: plain restarted GMRES.  R = float, RX = double (TM_MIXED): GMRES with iterative refinement - every cycle
// solves the correction equation M d = r for the fp64 residual r in fp32 and adds d to the fp64 iterate.
template <typename R, typename RX>
int gmres_solve(tm_ctx* ctx, int transpose, const tm_solve_opts& o, tm_solve_info* info) {
  // on entry: d_v[1] = right-hand side b (and, with o.warm_start, d_v[0] = initial guess x0); on exit d_v[0] = x.
  constexpr bool mixed = !std::is_same<R, RX>::value;
  Cx<RX>* X = vec<RX>(ctx, 0); Cx<RX>* B = vec<RX>(ctx, 1); Cx<RX>* ZX = vec<RX>(ctx, 2);
  const size_t n = ctx->n;
  const int m = o.restart, nw = ctx->n_win, nc = ctx->n_chunks;
  Cx<R>* V = reinterpret_cast<Cx<R>*>(ctx->ws);
  Cx<R>* W = V + (size_t)(m + 1) * n;
  // scratch of the transposed operator in the cycle precision, and the vector that receives M x / the true residual
  Cx<R>* ZV = mixed ? W + n : reinterpret_cast<Cx<R>*>(ZX);
  Cx<RX>* RXv = mixed ? reinterpret_cast<Cx<RX>*>((reinterpret_cast<uintptr_t>(ZV + n) + 255) & ~(uintptr_t)255)
                      : reinterpret_cast<Cx<RX>*>(W);
  TmGmresDev& S = ctx->gm.dev;
  S.inner_floor = mixed ? 1e-5 : 0.0;                 // an fp32 cycle cannot usefully reduce its residual further
  cudaStream_t st = ctx->stream;
  const int wb = (nw + 63) / 64;
  if (!ctx->t0_ev) { TM_CUDA(cudaEventCreate(&ctx->t0_ev)); TM_CUDA(cudaEventCreate(&ctx->t1_ev)); }
  cudaEvent_t e0 = ctx->t0_ev, e1 = ctx->t1_ev;
  TM_CUDA(cudaEventRecord(e0, st));
  const bool warm = o.warm_start != 0;
  if (!warm) TM_CUDA(cudaMemsetAsync(X, 0, n * sizeof(Cx<RX>), st));
  TM_CUDA(cudaMemsetAsync(V, 0, (size_t)(m + 2) * n * sizeof(Cx<R>), st));   // basis vectors must be finite (k_axpy)

  std::vector<int> h_k(nw), h_done(nw), iters(nw, 0), restarts(nw, 0);
  std::vector<double> h_res(nw, 0.0);
  int matvecs = 0, total = 0, cycle = 0, stagnant = 0, last_mc = 0;
  std::vector<double> prev_res(nw, 1e300);
  bool all_ok = false;
  // cooperative single-launch Arnoldi step: only when every chunk's block can be resident at once
  bool coop = false;
  int vcap = 0;                      // basis vectors whose chunk a block of k_arnoldi_fused keeps in shared memory
#ifndef TM_NO_COOP                 // build switch (-DTM_NO_COOP): multi-kernel Arnoldi step everywhere, for A/B measurements
  if (ctx->max_chunks_per_win <= 512) {
    int per_sm = 0, dev = 0, n_sm = 0, can = 0, smem_sm = 0, smem_blk = 0;
    const void* fn = ctx->ept == 1 ? (const void*)k_arnoldi_fused<R, 1> : (const void*)k_arnoldi_fused<R, 4>;
    const size_t sm_max = (size_t)(2 * m + 2) * sizeof(double2) + (size_t)(m + 1) * sizeof(double);
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&can, cudaDevAttrCooperativeLaunch, dev);
    cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev);
    cudaDeviceGetAttribute(&smem_blk, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    auto occ = [&](size_t dyn) {
      per_sm = 0;
      if (ctx->ept == 1) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_arnoldi_fused<R, 1>, TM_VT, dyn);
      else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_arnoldi_fused<R, 4>, TM_VT, dyn);
      return can && (long long)per_sm * n_sm >= nc;
    };
    coop = occ(sm_max);
#ifndef TM_NO_VCACHE               // build switch (-DTM_NO_VCACHE): every pass over the basis reads global memory
    if (coop) {                      // shared memory left per block when all nc blocks are co-resident -> cached vectors
      cudaFuncAttributes fa;
      cudaFuncGetAttributes(&fa, fn);
      const int bps = (nc + n_sm - 1) / n_sm;
      const long long per_blk = std::min<long long>(smem_blk, smem_sm / bps - 1024) - (long long)fa.sharedSizeBytes;
      const long long vbytes = (long long)ctx->ept * TM_VT * (long long)sizeof(Cx<R>);
      const long long room = per_blk - (long long)((sm_max + 15) & ~(size_t)15);
      vcap = room > 0 ? (int)std::min<long long>(m + 1, room / vbytes) : 0;
      if (vcap < 4) vcap = 0;
      if (vcap > 0) {
        const size_t dyn = ((sm_max + 15) & ~(size_t)15) + (size_t)vcap * vbytes;
        if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn) != cudaSuccess || !occ(dyn)) {
          cudaGetLastError();
          vcap = 0;
          coop = occ(sm_max);
        }
      }
    }
#endif
  }
#endif
  const Cx<RX>* resid_vec = B;                        // first cycle: x0 = 0 so r = b
  if (warm) {                                         // ||b|| is the reference norm; r0 = b - M x0 starts the first cycle
    k_norm2<RX><<<nc, TM_VT, 0, st>>>(B, ctx->d_chunks, ctx->gm.normpart);
    k_reduce_norm<<<nw, 64, 0, st>>>(ctx->gm.normpart, ctx->d_win_chunk_ptr, S.bnorm);
    TM_CUDA(apply_operator<RX>(ctx, transpose, X, RXv, ZX, nullptr));
    matvecs++;
    k_scale_or_sub<RX, RX><<<nc, TM_VT, 0, st>>>(B, RXv, nullptr, RXv, ctx->d_chunks, nullptr);
    ctx->total_launches += 3;
    resid_vec = RXv;
  }
  while (true) {
    // beta = ||r|| per window
    k_norm2<RX><<<nc, TM_VT, 0, st>>>(resid_vec, ctx->d_chunks, ctx->gm.normpart);
    k_reduce_norm<<<nw, 64, 0, st>>>(ctx->gm.normpart, ctx->d_win_chunk_ptr, S.normw);
    if (cycle > 0) {
      k_gmres_true_resid<<<wb, 64, 0, st>>>(S, nw);
      TM_CUDA(cudaMemcpyAsync(h_res.data(), S.resid, nw * sizeof(double), cudaMemcpyDeviceToHost, st));
      TM_CUDA(cudaMemcpyAsync(h_k.data(), S.kcols, nw * sizeof(int), cudaMemcpyDeviceToHost, st));
      TM_CUDA(stream_wait(ctx));
      int kmax = 0;
      all_ok = true;
      for (int w = 0; w < nw; ++w) {
        iters[w] += h_k[w]; kmax = std::max(kmax, h_k[w]);
        if (h_k[w] > 0) restarts[w]++;
        if (!(h_res[w] <= o.tol)) all_ok = false;
      }
      total += kmax;
      if (all_ok || total >= o.max_iter || kmax == 0) break;
      // Precision floor (fp32 mode): every window met the ESTIMATED residual before the cycle ended, yet the true
      // residual of the unconverged ones no longer improves - further cycles only repeat that.  Stop (soft status).
      bool floor_hit = kmax < last_mc;
      for (int w = 0; w < nw && floor_hit; ++w)
        if (!(h_res[w] <= o.tol) && h_res[w] < 0.9 * prev_res[w]) floor_hit = false;
      stagnant = floor_hit ? stagnant + 1 : 0;
      prev_res = h_res;
      if (stagnant >= 2) break;
    }
    TM_CUDA(cudaMemsetAsync(S.n_active, 0, sizeof(int), st));
    k_gmres_init_cycle<<<wb, 64, 0, st>>>(S, nw, (cycle == 0 && !warm) ? 1 : 0, o.tol);
    k_scale_or_sub<RX, R><<<nc, TM_VT, 0, st>>>(resid_vec, nullptr, S.inv_norm, V, ctx->d_chunks, nullptr);   // V_0 = r / beta
    ctx->total_launches += 4;
    const int mc = std::min(m, o.max_iter - total);
    last_mc = mc;
    // the Arnoldi steps of this cycle: enqueue(j0, j1) issues steps j0..j1-1 (directly or into a stream capture)
    auto enqueue = [&](int j0, int j1) -> int {
    for (int j = j0; j < j1; ++j) {
      Cx<R>* Vj = V + (size_t)j * n;
      const bool fuse_t = coop && ctx->diag;       // T application folded into the cooperative step
      if (fuse_t) {
        if (transpose == 1 && j == 0) TM_CUDA(launch_tapply<R>(ctx, 4, Vj, ZV, S.n_active));   // z = P T^T v_0
        TM_CUDA(launch_allpairs<R>(ctx, transpose == 1 ? ZV : Vj, S.n_active));
      } else {
        TM_CUDA(apply_operator<R>(ctx, transpose, Vj, W, ZV, S.n_active));
      }
      // split the basis vectors of a dot-product pass over gridDim.y when there are few chunks
      const int G = std::max(1, std::min((j + 1 + 7) / 8, (148 * 4 + nc - 1) / nc));
      const size_t sm_a = (size_t)(j + 1) * sizeof(double2);
      // small windows: the axpy blocks reduce the partial dots themselves (saves a launch per pass)
      const bool fuse = ctx->max_chunks_per_win <= 512;
#define TM_DOTS(H)                                                                                              \
  do {                                                                                                          \
    if (ctx->ept == 1) k_dots<R, 1><<<dim3(nc, G), TM_VT, 0, st>>>(V, n, j + 1, W, ctx->d_chunks, nc, ctx->gm.part, S.n_active); \
    else k_dots<R, 4><<<dim3(nc, G), TM_VT, 0, st>>>(V, n, j + 1, W, ctx->d_chunks, nc, ctx->gm.part, S.n_active); \
    if (!fuse) k_reduce_h<<<dim3(j + 1, nw), 64, 0, st>>>(ctx->gm.part, nc, ctx->d_win_chunk_ptr, H, S.ldh, 0, S.n_active); \
  } while (0)
#define TM_AXPY(H, NP)                                                                                          \
  do {                                                                                                          \
    const double2* pp = fuse ? ctx->gm.part : nullptr;                                                          \
    if (ctx->ept == 1) k_axpy<R, 1><<<nc, TM_VT, sm_a, st>>>(V, n, j + 1, H, S.ldh, -1.0, W, ctx->d_chunks, NP, pp, nc, ctx->d_win_chunk_ptr, S.n_active); \
    else k_axpy<R, 4><<<nc, TM_VT, sm_a, st>>>(V, n, j + 1, H, S.ldh, -1.0, W, ctx->d_chunks, NP, pp, nc, ctx->d_win_chunk_ptr, S.n_active); \
  } while (0)
      const size_t sm_g = (size_t)(2 * j + 2) * sizeof(double2) + (size_t)(j + 1) * sizeof(double);
      if (coop) {            // whole step in one cooperative launch (all chunks co-resident)
        const Cx<R>* Vc = V; size_t nn = n; int jj = j, ncc = nc, nww = nw; double tl = o.tol;
        Cx<R>* Wc = W; const TmChunk* chk = ctx->d_chunks; double2* prt = ctx->gm.part; double* npt = ctx->gm.normpart;
        const int* wcp = ctx->d_win_chunk_ptr; TmGmresDev Sc = S;
        TmFuseT<R> ft{fuse_t ? (transpose == 1 ? 2 : 1) : 0, Vj, reinterpret_cast<const Cx<R>*>(ctx->d_upart), ctx->n_part, n,
                      Tptr<R>(ctx), ctx->d_type_of, ctx->d_const->perm_neg_m, ctx->L, ZV};
        int vc = std::min(vcap, j + 1), voff = (int)((std::max(sm_a, sm_g) + 15) & ~(size_t)15);
        // Inside a captured cycle the Givens update (a long scalar recurrence run by ONE warp, ~5 us at the end of the step)
        // leaves the critical path: it becomes a node of its own on a side branch that only the NEXT Arnoldi step (and the
        // end of the cycle) waits for, so it runs beside the next all-pairs product.  That product may then read a stale
        // `n_active`; a window that has just converged costs one more product whose result nobody uses.  Same arithmetic.
        const bool side_givens = ctx->capturing && ctx->side != nullptr;
        int dg = side_givens ? 0 : 1;
        if (side_givens && j > j0) TM_CUDA(cudaStreamWaitEvent(st, ctx->join_ev, 0));
        void* args[] = {&Vc, &nn, &jj, &Wc, &chk, &ncc, &prt, &npt, &wcp, &Sc, &nww, &tl, &ft, &vc, &voff, &dg};
        const void* fn = ctx->ept == 1 ? (const void*)k_arnoldi_fused<R, 1> : (const void*)k_arnoldi_fused<R, 4>;
        const size_t sm_v = (size_t)voff + (size_t)vc * ctx->ept * TM_VT * sizeof(Cx<R>);
        TM_CUDA(cudaLaunchCooperativeKernel(fn, dim3(nc), dim3(TM_VT), args, sm_v, st));
        ctx->total_launches += 1;
        if (side_givens) {
          TM_CUDA(cudaEventRecord(ctx->fork_ev, st));
          TM_CUDA(cudaStreamWaitEvent(ctx->side, ctx->fork_ev, 0));
          k_gmres_givens<<<nw, 32, sm_g, ctx->side>>>(S, nw, j, o.tol, ctx->gm.normpart, ctx->d_win_chunk_ptr);
          TM_CUDA(cudaEventRecord(ctx->join_ev, ctx->side));
          if (j == j1 - 1) TM_CUDA(cudaStreamWaitEvent(st, ctx->join_ev, 0));
          ctx->total_launches += 1;
        }
      } else {
        TM_DOTS(S.h1);
        TM_AXPY(S.h1, nullptr);
        TM_DOTS(S.h2);
        TM_AXPY(S.h2, ctx->gm.normpart);
        k_gmres_givens<<<nw, 32, sm_g, st>>>(S, nw, j, o.tol, ctx->gm.normpart, ctx->d_win_chunk_ptr);
        k_scale_or_sub<R><<<nc, TM_VT, 0, st>>>(W, nullptr, S.inv_norm, V + (size_t)(j + 1) * n, ctx->d_chunks, S.n_active);
        ctx->total_launches += fuse ? 6 : 8;
      }
#undef TM_DOTS
#undef TM_AXPY
    }
    return TM_OK;
    };
    // CUDA graph of a full cycle (cooperative path only: small / medium problems, where the ~2 m launches of a cycle
    // cost more in launch gaps than in work).  Timing mode (tm_kernel_time) keeps direct launches: events per launch.
    bool launched = false;
    if (coop && ctx->graphs_ok && !ctx->time_kernels && mc == m && m >= 4) {
      tm_ctx::CycleGraph& G = ctx->cyc[transpose == 1 ? 1 : 0];
      const void* Tp = Tptr<R>(ctx);
      const bool hit = G.exec && G.transpose == transpose && G.m == m && G.rbytes == (int)sizeof(R) && G.n_part == ctx->n_part &&
                       G.kernel == ctx->kernel && G.tol == o.tol && G.ws == ctx->ws && G.T == Tp && G.upart == ctx->d_upart &&
                       G.blob == ctx->gm.blob && G.tiles == ctx->d_tiles && G.pacc == ctx->d_pacc && G.n_tiles == ctx->n_tiles &&
                       G.n_chunk == ctx->n_chunk && G.diag == ctx->diag;
      if (!hit) {
        if (G.exec) { cudaGraphExecDestroy(G.exec); G.exec = nullptr; }
        const long long l0 = ctx->total_launches, a0 = ctx->allpairs_launches;
        cudaGraph_t graph = nullptr;
#ifndef TM_NO_SIDE_GIVENS           // build switch (-DTM_NO_SIDE_GIVENS): Givens update inside the Arnoldi kernel in captured cycles too
        if (!ctx->side) {
          if (cudaStreamCreateWithFlags(&ctx->side, cudaStreamNonBlocking) != cudaSuccess ||
              cudaEventCreateWithFlags(&ctx->fork_ev, cudaEventDisableTiming) != cudaSuccess ||
              cudaEventCreateWithFlags(&ctx->join_ev, cudaEventDisableTiming) != cudaSuccess) {
            cudaGetLastError();
            if (ctx->side) { cudaStreamDestroy(ctx->side); ctx->side = nullptr; }
          }
        }
#endif
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
          ctx->capturing = true;
          const int rc_cap = enqueue(0, m);
          ctx->capturing = false;
          const cudaError_t ee = cudaStreamEndCapture(st, &graph);
          if (rc_cap == TM_OK && ee == cudaSuccess && graph && cudaGraphInstantiate(&G.exec, graph, 0) == cudaSuccess) {
            G.transpose = transpose; G.m = m; G.rbytes = (int)sizeof(R); G.n_part = ctx->n_part; G.kernel = ctx->kernel;
            G.tol = o.tol; G.ws = ctx->ws; G.T = Tp; G.upart = ctx->d_upart; G.blob = ctx->gm.blob; G.tiles = ctx->d_tiles; G.pacc = ctx->d_pacc; G.n_tiles = ctx->n_tiles; G.n_chunk = ctx->n_chunk; G.diag = ctx->diag;
            G.launches = (int)(ctx->total_launches - l0);
          } else {
            G.exec = nullptr; ctx->graphs_ok = false;
          }
          if (graph) cudaGraphDestroy(graph);
        } else {
          ctx->graphs_ok = false;
        }
        cudaGetLastError();
        ctx->total_launches = l0; ctx->allpairs_launches = a0;       // the capture pass launched nothing
      }
      if (G.exec) {
        TM_CUDA(cudaGraphLaunch(G.exec, st));
        ctx->total_launches += G.launches; ctx->allpairs_launches += m;
        launched = true;
      }
    }
    if (!launched) { const int rc_e = enqueue(0, mc); if (rc_e != TM_OK) return rc_e; }
    matvecs += mc;
    // x += V y ; r = b - M x
    k_gmres_solve_y<<<nw, 32, 0, st>>>(S, nw);
    if (ctx->ept == 1) k_axpy<R, 1, RX><<<nc, TM_VT, (size_t)m * sizeof(double2), st>>>(V, n, m, S.y, S.ldh, +1.0, X, ctx->d_chunks, nullptr, nullptr, nc, ctx->d_win_chunk_ptr, nullptr);
    else k_axpy<R, 4, RX><<<nc, TM_VT, (size_t)m * sizeof(double2), st>>>(V, n, m, S.y, S.ldh, +1.0, X, ctx->d_chunks, nullptr, nullptr, nc, ctx->d_win_chunk_ptr, nullptr);
    TM_CUDA(apply_operator<RX>(ctx, transpose, X, RXv, ZX, nullptr));                       // in the iterate's precision
    matvecs++;
    k_scale_or_sub<RX, RX><<<nc, TM_VT, 0, st>>>(B, RXv, nullptr, RXv, ctx->d_chunks, nullptr);   // r = b - M x
    ctx->total_launches += 3;
    TM_CUDA(cudaGetLastError());
    resid_vec = RXv;
    cycle++;
  }
  TM_CUDA(cudaEventRecord(e1, st));
  TM_CUDA(cudaEventSynchronize(e1));
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  if (info)
    for (int w = 0; w < nw; ++w) {
      info[w].iterations = iters[w]; info[w].restarts = restarts[w]; info[w].converged = h_res[w] <= o.tol ? 1 : 0;
      info[w].matvecs = matvecs; info[w].rel_residual = h_res[w]; info[w].seconds = ms * 1e-3;
    }
  return all_ok ? TM_OK : TM_NOT_CONVERGED;
}

}  // namespace

// ============================================================================================ setup helpers
namespace {

// min over same-window pairs of |x_i - x_j| - r_i - r_j  <= 0  -> flag (coincident centres when radii are null)
__global__ void k_check_overlap(const double* __restrict__ pos, const int* __restrict__ win_of, const int* __restrict__ win_ptr,
                                const int* __restrict__ type_of, const double* __restrict__ radii, int n_scat, int* flag) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n_scat) return;
  const int w = win_of[j];
  const double xj = pos[3 * j], yj = pos[3 * j + 1], zj = pos[3 * j + 2];
  const double rj = radii ? radii[type_of[j]] : 0.0;
  bool bad = false;
  for (int i = win_ptr[w]; i < win_ptr[w + 1]; ++i) {
    if (i == j) continue;
    const double dx = xj - pos[3 * i], dy = yj - pos[3 * i + 1], dz = zj - pos[3 * i + 2];
    const double ri = radii ? radii[type_of[i]] : 0.0;
    const double lim = ri + rj;
    const double d2 = dx * dx + dy * dy + dz * dz;
    if (radii ? (d2 < lim * lim) : (d2 == 0.0)) bad = true;
  }
  if (bad) atomicExch(flag, 1);
}

void fill_const(tm_ctx* c) {
  TmConst& t = c->h_const;
  std::memset(&t, 0, sizeof(t));
  const int lmax = c->lmax, L = c->L, LH = L / 2;
  for (int p = 0; p < 2; ++p)
    for (int l = 1; l <= lmax; ++l)
      for (int m = -l; m <= l; ++m) {
        const int idx = p * LH + l * (l + 1) - 1 + m;
        t.mode_l[idx] = l; t.mode_m[idx] = m; t.mode_p[idx] = p;
        t.perm_neg_m[idx] = p * LH + l * (l + 1) - 1 - m;
      }
  for (int q = 0; q <= TM_MAX_NQ; ++q)
    for (int mu = 0; mu <= q && mu <= TM_MAX_NQ; ++mu) {
      if (q > mu) {
        t.leg_a[q][mu] = std::sqrt((4.0 * q * q - 1.0) / ((double)q * q - (double)mu * mu));
        const double qq = (q - 1.0);
        t.leg_b[q][mu] = (q - 1 > mu) ? std::sqrt((qq * qq - (double)mu * mu) / (4.0 * qq * qq - 1.0)) : 0.0;
      }
    }
  for (int mu = 1; mu <= TM_MAX_NQ; ++mu) t.leg_d[mu] = std::sqrt((2.0 * mu + 1.0) / (2.0 * mu));
}

int configure_kernel(tm_ctx* ctx) {
  int want = ctx->kernel_req;
  if (want == TM_KERNEL_AUTO) want = ctx->coplanar ? TM_KERNEL_COPLANAR : TM_KERNEL_ROT3D;
  if (want == TM_KERNEL_COPLANAR && !ctx->coplanar)
    return fail(ctx, TM_E_INVALID, "coplanar kernel needs all z equal");
  if (want == TM_KERNEL_SYM3D && ctx->lmax > 3) return fail(ctx, TM_E_INVALID, "generated 3-D kernel needs lmax <= 3");
  ctx->kernel = want;
#ifdef TM_COP_TJ                   // build switch (-DTM_COP_TJ=256): 256 targets per block (measured +-1 %)
  ctx->cop_tj = TM_COP_TJ == 256 ? 256 : 128;
#endif
  int tgt_per_tile;
  const bool gen = want == TM_KERNEL_COPLANAR || want == TM_KERNEL_SYM3D || want == TM_KERNEL_ROT3D;   // generated kernels: thread = target
  switch (gen ? 0 : ctx->lmax) {
    case 0: tgt_per_tile = want == TM_KERNEL_ROT3D ? (tm_rot3d_ws(ctx->lmax) ? 32 : tm_rot3d_tj(ctx->lmax)) : (want == TM_KERNEL_SYM3D ? TM_SYM3D_TJ : (ctx->lmax > 3 ? tm_cop4_tj(ctx->lmax) : ctx->cop_tj)); break;
    default: tgt_per_tile = tm_general_tj(ctx->lmax); break;
  }
  std::vector<TmTile> tiles;
  int min_win = ctx->n_scat;
  for (int w = 0; w < ctx->n_win; ++w) {
    const int lo = ctx->win_ptr[w], hi = ctx->win_ptr[w + 1];
    if (hi > lo) min_win = std::min(min_win, hi - lo);
    for (int s = lo; s < hi; s += tgt_per_tile) tiles.push_back(TmTile{s, std::min(tgt_per_tile, hi - s), lo, hi - lo});
  }
  ctx->n_tiles = (int)tiles.size();
  // Source chunks: pick the chunk count that minimises (waves of resident blocks) x (sources per block), so that
  // small problems fill the 148 SMs (2 resident 128-thread blocks each at 255 registers) and large ones end
  // without a long tail; bounded by 64 chunks, >= 32 sources per chunk and 2 GB of partial sums.
  const bool cop4 = want == TM_KERNEL_COPLANAR && ctx->lmax > 3;   // four-sector coplanar kernel (lmax 4..6)
  const long long slots = 148LL * (cop4 ? 256 / tm_cop4_tj(ctx->lmax) : (want == TM_KERNEL_COPLANAR ? 256 / ctx->cop_tj :
                                   (want == TM_KERNEL_SYM3D ? 2 : (want == TM_KERNEL_ROT3D ? (tm_rot3d_ws(ctx->lmax) ? 2 : (ctx->lmax <= 6 ? 2 : 1)) : 4))));
  const int cop4_z = !cop4 ? 0 : 4 * tm_cop4_groups(ctx->lmax);
  const long long blocks1 = (long long)ctx->n_tiles * (cop4 ? cop4_z : (gen ? 2 : 1));
  const int part_mult = (want == TM_KERNEL_SYM3D || want == TM_KERNEL_ROT3D || cop4) ? 2 : 1;   // one partial buffer per (chunk, y'-sector)
  int max_win = 1;
  for (int w = 0; w < ctx->n_win; ++w) max_win = std::max(max_win, ctx->win_ptr[w + 1] - ctx->win_ptr[w]);
  const size_t vec_bytes = ctx->n * elem_bytes(ctx);
  long long nchunk = 1;
  double best = 1e300;
  for (long long cnd = 1; cnd <= 64; ++cnd) {
    if (cnd > 1 && (min_win / cnd < 32 || (size_t)cnd * part_mult * vec_bytes > ((size_t)2 << 30))) break;
    const long long waves = (blocks1 * cnd + slots - 1) / slots;
    const double cost = (double)waves * (double)((max_win + cnd - 1) / cnd + 8);     // +8: per-block fixed cost
    if (cost < best * 0.995) { best = cost; nchunk = cnd; }
  }
  ctx->n_chunk = (int)std::max<long long>(1, nchunk);
  if (ctx->d_tiles) tm_dev_free(ctx->d_tiles);
  TM_CUDA(tm_dev_alloc(&ctx->d_tiles, tiles.size() * sizeof(TmTile)));
  TM_CUDA(cudaMemcpy(ctx->d_tiles, tiles.data(), tiles.size() * sizeof(TmTile), cudaMemcpyHostToDevice));
  if (want == TM_KERNEL_ROT3D && tm_rot3d_pg(ctx->lmax) && !tm_rot3d_ws(ctx->lmax)) {
    const size_t per_block = (size_t)tm_rot3d_pg(ctx->lmax) * ctx->L * tm_rot3d_tj(ctx->lmax) * (ctx->precision == TM_FP32 ? sizeof(float) : sizeof(double));
    const size_t need_p = (size_t)ctx->n_tiles * ctx->n_chunk * 2 * per_block;
    if (need_p > ctx->pacc_bytes) {
      if (ctx->d_pacc) tm_dev_free(ctx->d_pacc);
      ctx->d_pacc = nullptr; ctx->pacc_bytes = 0;
      TM_CUDA(tm_dev_alloc(&ctx->d_pacc, need_p));
      ctx->pacc_bytes = need_p;
    }
  }
  // Optional (build switch, OFF by default): on large planar problems (lmax <= 3) clusters of 4 or 2 chunk blocks sum their partials
  // through distributed shared memory, so only n_chunk / cl partial buffers are written and read back.  Measured on config 5
  // (8 chunks; profiles/r02_cluster_reduction.md): DRAM traffic of the launch 572 MB -> 177 MB (clusters of 2) / 64 MB (clusters
  // of 4), launch time 132.6 -> 134.6 / 142.4 ms - the launch is ALU-bound, the traffic costs nothing, and only 71 of the 74
  // clusters of 4 that the 296 block slots could hold are co-resident.  Parity with clusters on: 1e-12 (same tests).
#ifndef TM_COP_CLUSTER
#define TM_COP_CLUSTER 0              // largest cluster size: 4, 2, or 0 = never launch clusters
#endif
  ctx->cop_cl = 1;
  if (TM_COP_CLUSTER >= 2 && want == TM_KERNEL_COPLANAR && !cop4 && ctx->cop_tj == 128 && ctx->n_chunk > 1 &&
      (size_t)ctx->n_chunk * vec_bytes >= ((size_t)32 << 20))
    ctx->cop_cl = (TM_COP_CLUSTER >= 4 && ctx->n_chunk % 4 == 0) ? 4 : (ctx->n_chunk % 2 == 0 ? 2 : 1);
  ctx->n_part = ctx->n_chunk * part_mult / ctx->cop_cl;
  const size_t need = (size_t)ctx->n_part * vec_bytes;
  if (need > ctx->upart_bytes) {
    if (ctx->d_upart) tm_dev_free(ctx->d_upart);
    ctx->d_upart = nullptr; ctx->upart_bytes = 0;
    TM_CUDA(tm_dev_alloc(&ctx->d_upart, need));
    ctx->upart_bytes = need;
  }
  return TM_OK;
}

int ensure_gmres(tm_ctx* ctx, int restart) {
  if (ctx->gm.restart >= restart && ctx->gm.blob) { ctx->gm.dev.ldh = restart + 1; ctx->gm.dev.m = restart; return TM_OK; }
  if (ctx->gm.blob) tm_dev_free(ctx->gm.blob);
  ctx->gm = Gmres{};
  const size_t nw = ctx->n_win, ldh = restart + 1, m = restart, nc = ctx->n_chunks;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += (bytes + 255) / 256 * 256; return o; };
  const size_t o_h1 = take(nw * ldh * 16), o_h2 = take(nw * ldh * 16), o_R = take(nw * m * ldh * 16), o_cs = take(nw * m * 8),
               o_sn = take(nw * m * 16), o_g = take(nw * ldh * 16), o_y = take(nw * ldh * 16), o_nw = take(nw * 8),
               o_bn = take(nw * 8), o_in = take(nw * 8), o_b0 = take(nw * 8), o_rs = take(nw * 8), o_k = take(nw * 4), o_d = take(nw * 4),
               o_na = take(4), o_part = take(2 * ldh * nc * 16) /* two buffers: k_arnoldi_fused */, o_np = take(nc * 8);
  TM_CUDA(tm_dev_alloc(&ctx->gm.blob, off));
  TM_CUDA(cudaMemset(ctx->gm.blob, 0, off));
  char* b = reinterpret_cast<char*>(ctx->gm.blob);
  TmGmresDev& S = ctx->gm.dev;
  S.h1 = (double2*)(b + o_h1); S.h2 = (double2*)(b + o_h2); S.Rm = (double2*)(b + o_R); S.cs = (double*)(b + o_cs);
  S.sn = (double2*)(b + o_sn); S.g = (double2*)(b + o_g); S.y = (double2*)(b + o_y); S.normw = (double*)(b + o_nw);
  S.bnorm = (double*)(b + o_bn); S.inv_norm = (double*)(b + o_in); S.beta0 = (double*)(b + o_b0); S.resid = (double*)(b + o_rs); S.kcols = (int*)(b + o_k);
  S.done = (int*)(b + o_d); S.n_active = (int*)(b + o_na);
  S.ldh = (int)ldh; S.m = (int)m; S.inner_floor = 0.0;
  ctx->gm.part = (double2*)(b + o_part); ctx->gm.normpart = (double*)(b + o_np);
  ctx->gm.restart = restart;
  return TM_OK;
}

size_t ws_bytes_for(const tm_ctx* c, int restart) {
  if (c->precision == TM_MIXED)     // fp32 basis + work vector + fp32 scratch, fp64 residual vector
    return (size_t)(restart + 3) * c->n * sizeof(Cx<float>) + c->n * sizeof(Cx<double>) + 1024;
  return (size_t)(restart + 2) * c->n * elem_bytes(c) + 256;
}

int ensure_workspace(tm_ctx* ctx, int restart) {
  const size_t need = ws_bytes_for(ctx, restart);
  if (ctx->ws && ctx->ws_bytes >= need) return TM_OK;
  if (ctx->ws && !ctx->ws_owned) return fail(ctx, TM_E_NOMEM, "caller workspace too small: see tm_workspace_bytes");
  if (ctx->ws) tm_dev_free(ctx->ws);
  ctx->ws = nullptr; ctx->ws_bytes = 0;
  TM_CUDA(tm_dev_alloc(&ctx->ws, need));
  ctx->ws_bytes = need; ctx->ws_owned = true;
  return TM_OK;
}

int check_opts(tm_ctx* ctx, const tm_solve_opts* o) {
  if (!o) return fail(ctx, TM_E_INVALID, "opts is NULL");
  if (!(o->tol > 0.0) || o->restart < 1 || o->restart > MAX_RESTART || o->max_iter < 1)
    return fail(ctx, TM_E_INVALID, "need tol > 0, 1 <= restart <= 300, max_iter >= 1");
  return TM_OK;
}

}  // namespace

// ============================================================================================ C ABI
extern "C" {

int tm_num_modes(int lmax) { return 2 * lmax * (lmax + 2); }

const char* tm_last_error(const tm_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

void tm_destroy(tm_ctx* c) {
  if (!c) return;
  cudaStreamSynchronize(c->stream);
  for (auto& g : c->cyc) if (g.exec) cudaGraphExecDestroy(g.exec);
  if (c->side) cudaStreamDestroy(c->side);
  if (c->fork_ev) cudaEventDestroy(c->fork_ev);
  if (c->join_ev) cudaEventDestroy(c->join_ev);
  if (c->grad_aux) tm_destroy(c->grad_aux);
  if (c->multi_aux) tm_destroy(c->multi_aux);
  tm_dev_free(c->d_grad_tab);
  tm_dev_free(c->d_pos); tm_dev_free(c->d_win_of); tm_dev_free(c->d_type_of); tm_dev_free(c->d_T); tm_dev_free(c->d_T32); tm_dev_free(c->d_p);
  tm_dev_free(c->d_const); tm_dev_free(c->d_rowptr); tm_dev_free(c->d_col); tm_dev_free(c->d_widx); tm_dev_free(c->d_imag);
  tm_dev_free(c->d_coef); tm_dev_free(c->d_tiles); tm_dev_free(c->d_upart); tm_dev_free(c->d_pacc); tm_dev_free(c->d_chunks); tm_dev_free(c->d_win_chunk_ptr);
  for (int i = 0; i < 3; ++i) tm_dev_free(c->d_v[i]);
  tm_dev_free(c->d_io);
  if (c->ws_owned) tm_dev_free(c->ws);
  tm_dev_free(c->gm.blob);
  for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
  if (c->sync_ev) cudaEventDestroy(c->sync_ev);
  if (c->t0_ev) cudaEventDestroy(c->t0_ev);
  if (c->t1_ev) cudaEventDestroy(c->t1_ev);
  for (int i = 0; i < 8; ++i) tm_dev_free(c->scratch[i]);
  delete c;
}

}  // extern "C"

namespace {
// tm_create with the truncation limit as a parameter: the public entry point allows lmax <= TM_MAX_LMAX, the position
// gradient builds its auxiliary context at lmax + 1 <= TM_INT_LMAX.
int create_ctx(tm_ctx** out, int n_scat, const double* pos_xyz, int n_win, const int* win_ptr, int lmax, double k_b,
               int precision, void* cuda_stream, int lmax_limit) {
  tm_ctx* ctx = nullptr;                                  // errors before allocation go to g_create_error
  if (!out) return fail(ctx, TM_E_INVALID, "out is NULL");
  *out = nullptr;
  if (n_scat < 1 || !pos_xyz) return fail(ctx, TM_E_INVALID, "need n_scat >= 1 and positions");
  static_assert(tm_max_table_lmax == TM_INT_LMAX, "term tables must reach the internal truncation");
  if (lmax < 1 || lmax > lmax_limit) return fail(ctx, TM_E_INVALID, "lmax must be in 1..6");
  if (!(k_b > 0.0) || !std::isfinite(k_b)) return fail(ctx, TM_E_INVALID, "k_b must be positive and finite");
  if (precision != TM_FP64 && precision != TM_FP32 && precision != TM_MIXED)
    return fail(ctx, TM_E_INVALID, "precision must be TM_FP64, TM_FP32 or TM_MIXED");
  if (n_win < 1) return fail(ctx, TM_E_INVALID, "n_win must be >= 1");
  std::vector<int> wp;
  if (win_ptr) {
    wp.assign(win_ptr, win_ptr + n_win + 1);
    if (wp[0] != 0 || wp[n_win] != n_scat) return fail(ctx, TM_E_INVALID, "win_ptr must start at 0 and end at n_scat");
    for (int w = 0; w < n_win; ++w)
      if (wp[w + 1] < wp[w]) return fail(ctx, TM_E_INVALID, "win_ptr must be monotone");
  } else {
    if (n_win != 1) return fail(ctx, TM_E_INVALID, "win_ptr is NULL but n_win != 1");
    wp = {0, n_scat};
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return fail(ctx, TM_E_CUDA, "no CUDA device: libtm has no CPU fallback");
  }
  std::vector<double> hpos((size_t)n_scat * 3);
  {
    cudaError_t e = cudaMemcpy(hpos.data(), pos_xyz, hpos.size() * sizeof(double),
                               is_device_ptr(pos_xyz) ? cudaMemcpyDeviceToHost : cudaMemcpyHostToHost);
    if (e != cudaSuccess) return fail(ctx, TM_E_CUDA, std::string("copy positions: ") + cudaGetErrorString(e));
  }
  bool coplanar = true;
  for (size_t i = 0; i < hpos.size(); ++i)
    if (!std::isfinite(hpos[i])) return fail(ctx, TM_E_INVALID, "non-finite position");
  for (int i = 1; i < n_scat; ++i)
    if (hpos[3 * (size_t)i + 2] != hpos[2]) { coplanar = false; break; }

  tm_ctx* c = new tm_ctx();
  c->n_scat = n_scat; c->n_win = n_win; c->lmax = lmax; c->L = tm_num_modes(lmax); c->precision = precision;
  c->k = k_b; c->n = (size_t)n_scat * c->L; c->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  c->win_ptr = wp; c->coplanar = coplanar; c->h_pos = hpos;
  ctx = c;
#define TM_CREATE_CUDA(call)                                                                  \
  do {                                                                                        \
    cudaError_t e_ = (call);                                                                  \
    if (e_ != cudaSuccess) {                                                                  \
      g_create_error = std::string(#call) + ": " + cudaGetErrorString(e_);                    \
      const int code_ = e_ == cudaErrorMemoryAllocation ? TM_E_NOMEM : TM_E_CUDA;             \
      tm_destroy(c);                                                                          \
      return code_;                                                                           \
    }                                                                                         \
  } while (0)
  TM_CREATE_CUDA(tm_dev_alloc(&c->d_pos, hpos.size() * sizeof(double)));
  TM_CREATE_CUDA(cudaMemcpy(c->d_pos, hpos.data(), hpos.size() * sizeof(double), cudaMemcpyHostToDevice));
  std::vector<int> win_of(n_scat);
  for (int w = 0; w < n_win; ++w) for (int i = wp[w]; i < wp[w + 1]; ++i) win_of[i] = w;
  TM_CREATE_CUDA(tm_dev_alloc(&c->d_win_of, n_scat * sizeof(int)));
  TM_CREATE_CUDA(cudaMemcpy(c->d_win_of, win_of.data(), n_scat * sizeof(int), cudaMemcpyHostToDevice));
  TM_CREATE_CUDA(tm_dev_alloc(&c->d_type_of, n_scat * sizeof(int)));
  fill_const(c);
  TM_CREATE_CUDA(tm_dev_alloc(&c->d_const, sizeof(TmConst)));
  TM_CREATE_CUDA(cudaMemcpy(c->d_const, &c->h_const, sizeof(TmConst), cudaMemcpyHostToDevice));
  {   // general-kernel term table of this lmax
    const TmTermTable& t = tm_term_tables[lmax - 1];
    const int nt = t.n_terms, L = c->L;
    std::vector<uint8_t> widx(nt), imag(nt);
    std::vector<double> coef(nt);
    for (int b = 0; b < L; ++b)
      for (int q = t.row_ptr[b]; q < t.row_ptr[b + 1]; ++q) {
        const int mu = c->h_const.mode_m[t.col[q]] - c->h_const.mode_m[b];
        const int qq = t.q[q];
        widx[q] = (uint8_t)(qq * qq + qq + mu);
        imag[q] = t.ipow[q] & 1;
        coef[q] = (t.ipow[q] & 2) ? -t.val[q] : t.val[q];
      }
    TM_CREATE_CUDA(tm_dev_alloc(&c->d_rowptr, (L + 1) * sizeof(int)));
    TM_CREATE_CUDA(cudaMemcpy(c->d_rowptr, t.row_ptr, (L + 1) * sizeof(int), cudaMemcpyHostToDevice));
    TM_CREATE_CUDA(tm_dev_alloc(&c->d_col, nt)); TM_CREATE_CUDA(cudaMemcpy(c->d_col, t.col, nt, cudaMemcpyHostToDevice));
    TM_CREATE_CUDA(tm_dev_alloc(&c->d_widx, nt)); TM_CREATE_CUDA(cudaMemcpy(c->d_widx, widx.data(), nt, cudaMemcpyHostToDevice));
    TM_CREATE_CUDA(tm_dev_alloc(&c->d_imag, nt)); TM_CREATE_CUDA(cudaMemcpy(c->d_imag, imag.data(), nt, cudaMemcpyHostToDevice));
    TM_CREATE_CUDA(tm_dev_alloc(&c->d_coef, nt * sizeof(double)));
    TM_CREATE_CUDA(cudaMemcpy(c->d_coef, coef.data(), nt * sizeof(double), cudaMemcpyHostToDevice));
  }
  {   // vector chunks: every chunk inside one window
    std::vector<TmChunk> ch;
    std::vector<int> wcp(n_win + 1, 0);
    c->ept = (c->n < (size_t)148 * 2 * 4 * TM_VT) ? 1 : 4;       // small vectors: more, smaller blocks
    const long long chunk = (long long)c->ept * TM_VT;
    for (int w = 0; w < n_win; ++w) {
      const long long e0 = (long long)wp[w] * c->L, e1 = (long long)wp[w + 1] * c->L;
      for (long long s = e0; s < e1; s += chunk) ch.push_back(TmChunk{w, (int)s, (int)std::min<long long>(chunk, e1 - s)});
      wcp[w + 1] = (int)ch.size();
      c->max_chunks_per_win = std::max(c->max_chunks_per_win, wcp[w + 1] - wcp[w]);
    }
    if (c->n > (size_t)0x7fffffff) { g_create_error = "problem too large (n_scat * L must fit in int32)"; tm_destroy(c); return TM_E_INVALID; }
    c->n_chunks = (int)ch.size();
    TM_CREATE_CUDA(tm_dev_alloc(&c->d_chunks, ch.size() * sizeof(TmChunk)));
    TM_CREATE_CUDA(cudaMemcpy(c->d_chunks, ch.data(), ch.size() * sizeof(TmChunk), cudaMemcpyHostToDevice));
    TM_CREATE_CUDA(tm_dev_alloc(&c->d_win_chunk_ptr, (n_win + 1) * sizeof(int)));
    TM_CREATE_CUDA(cudaMemcpy(c->d_win_chunk_ptr, wcp.data(), (n_win + 1) * sizeof(int), cudaMemcpyHostToDevice));
  }
  for (int i = 0; i < 3; ++i) TM_CREATE_CUDA(tm_dev_alloc(&c->d_v[i], c->n * elem_bytes(c)));
  TM_CREATE_CUDA(tm_dev_alloc(&c->d_io, c->n * sizeof(double2)));
  TM_CREATE_CUDA(tm_dev_alloc(&c->d_p, c->n * sizeof(double2)));
  {   // coincident centres are always an error (h_q diverges)
    int* d_flag = nullptr; int* d_wp = nullptr; int h_flag = 0;
    TM_CREATE_CUDA(tm_dev_alloc(&d_flag, sizeof(int)));
    TM_CREATE_CUDA(cudaMemset(d_flag, 0, sizeof(int)));
    TM_CREATE_CUDA(tm_dev_alloc(&d_wp, (n_win + 1) * sizeof(int)));
    TM_CREATE_CUDA(cudaMemcpy(d_wp, wp.data(), (n_win + 1) * sizeof(int), cudaMemcpyHostToDevice));
    k_check_overlap<<<(n_scat + 127) / 128, 128>>>(c->d_pos, c->d_win_of, d_wp, nullptr, nullptr, n_scat, d_flag);
    cudaError_t e = cudaMemcpy(&h_flag, d_flag, sizeof(int), cudaMemcpyDeviceToHost);
    tm_dev_free(d_flag); tm_dev_free(d_wp);
    TM_CREATE_CUDA(e);
    if (h_flag) { g_create_error = "two scatterers of one window share a centre"; tm_destroy(c); return TM_E_INVALID; }
  }
  {
    const int rc = configure_kernel(c);
    if (rc != TM_OK) { g_create_error = c->err; tm_destroy(c); return rc; }
  }
#undef TM_CREATE_CUDA
  *out = c;
  return TM_OK;
}
}  // namespace

extern "C" {

int tm_create(tm_ctx** out, int n_scat, const double* pos_xyz, int n_win, const int* win_ptr, int lmax, double k_b,
              int precision, void* cuda_stream) {
  return create_ctx(out, n_scat, pos_xyz, n_win, win_ptr, lmax, k_b, precision, cuda_stream, TM_MAX_LMAX);
}

int tm_set_kernel(tm_ctx* ctx, int kernel) {
  if (!ctx) return TM_E_INVALID;
  if (kernel < TM_KERNEL_AUTO || kernel > TM_KERNEL_ROT3D) return fail(ctx, TM_E_INVALID, "unknown kernel id");
  const int old = ctx->kernel_req;
  ctx->kernel_req = kernel;
  TM_CUDA(stream_wait(ctx));
  const int rc = configure_kernel(ctx);
  if (rc != TM_OK) { ctx->kernel_req = old; configure_kernel(ctx); }
  return rc;
}

int tm_get_kernel(const tm_ctx* ctx) { return ctx ? ctx->kernel : TM_E_INVALID; }

size_t tm_workspace_bytes(const tm_ctx* ctx, const tm_solve_opts* opts) {
  if (!ctx || !opts || opts->restart < 1) return 0;
  return ws_bytes_for(ctx, opts->restart);
}

int tm_set_workspace(tm_ctx* ctx, void* dev_ptr, size_t bytes) {
  if (!ctx) return TM_E_INVALID;
  if (dev_ptr && (!is_device_ptr(dev_ptr) || (reinterpret_cast<uintptr_t>(dev_ptr) & 255)))
    return fail(ctx, TM_E_INVALID, "workspace must be 256-byte aligned device memory");
  TM_CUDA(stream_wait(ctx));
  if (ctx->ws && ctx->ws_owned) tm_dev_free(ctx->ws);
  ctx->ws = dev_ptr; ctx->ws_bytes = dev_ptr ? bytes : 0; ctx->ws_owned = false;
  return TM_OK;
}

int tm_kernel_time(tm_ctx* ctx, int reset, double* allpairs_ms, long long* allpairs_launches, long long* total_launches) {
  if (!ctx) return TM_E_INVALID;
  TM_CUDA(stream_wait(ctx));
  double ms = 0.0;
  for (size_t i = 0; i + 1 < ctx->ev_used; i += 2) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, ctx->ev[i], ctx->ev[i + 1]) == cudaSuccess) ms += t;
  }
  // scale to all launches if the event pool ran out (stated in DESIGN.md: average over the recorded ones)
  const long long recorded = (long long)(ctx->ev_used / 2);
  if (recorded > 0 && ctx->allpairs_launches > recorded) ms *= (double)ctx->allpairs_launches / (double)recorded;
  if (allpairs_ms) *allpairs_ms = ms;
  if (allpairs_launches) *allpairs_launches = ctx->allpairs_launches;
  if (total_launches) *total_launches = ctx->total_launches;
  if (reset < 0) {                               // leave timing mode: restart cycles run as CUDA graphs again; counters restart
    ctx->time_kernels = false; ctx->ev_used = 0; ctx->allpairs_launches = 0; ctx->total_launches = 0;
  }
  if (reset > 0) {
    if (ctx->ev.empty()) {
      ctx->ev.resize(2 * 4096);
      for (cudaEvent_t& e : ctx->ev) TM_CUDA(cudaEventCreate(&e));
    }
    ctx->ev_used = 0; ctx->allpairs_launches = 0; ctx->total_launches = 0; ctx->time_kernels = true;
  }
  return TM_OK;
}

}  // extern "C"

// ============================================================================================ C ABI, part 2
namespace {

template <typename R>
int set_T_typed(tm_ctx* ctx, size_t count, const tm_c64* T, void* dst) {
  // stage fp64 -> Cx<R>
  double2* tmp = nullptr;
  TM_CUDA(tm_dev_alloc(&tmp, count * sizeof(double2)));
  cudaError_t e = copy_in(tmp, T, count * sizeof(double2), ctx->stream);
  if (e == cudaSuccess) {
    k_from_c64<R><<<grid_for(count, 256), 256, 0, ctx->stream>>>(reinterpret_cast<const double*>(tmp),
                                                                 reinterpret_cast<Cx<R>*>(dst), count);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = stream_wait(ctx);
  tm_dev_free(tmp);
  TM_CUDA(e);
  return TM_OK;
}

template <typename R>
int matvec_typed(tm_ctx* ctx, int transpose, const tm_c64* x, tm_c64* y) {
  TM_CUDA(load_c64<R>(ctx, x, vec<R>(ctx, 0)));
  TM_CUDA(apply_operator<R>(ctx, transpose, vec<R>(ctx, 0), vec<R>(ctx, 1), vec<R>(ctx, 2), nullptr));
  TM_CUDA(store_c64<R>(ctx, vec<R>(ctx, 1), y));
  TM_CUDA(stream_wait(ctx));
  return TM_OK;
}

template <typename RV, typename R>
int solve_typed(tm_ctx* ctx, int adjoint, const tm_c64* w, const tm_solve_opts& o, tm_c64* out, tm_solve_info* info) {
  if (adjoint) {
    TM_CUDA(load_c64<R>(ctx, w, vec<R>(ctx, 1)));                           // b = w
  } else {
    k_from_c64<R><<<grid_for(ctx->n, 256), 256, 0, ctx->stream>>>(reinterpret_cast<const double*>(ctx->d_p), vec<R>(ctx, 2), ctx->n);
    TM_CUDA(cudaGetLastError());
    TM_CUDA(launch_tapply<R>(ctx, 3, vec<R>(ctx, 2), vec<R>(ctx, 1), nullptr));   // b = T p   (Eq. I25)
    ctx->total_launches++;
  }
  if (o.warm_start) TM_CUDA(load_c64<R>(ctx, out, vec<R>(ctx, 0)));        // x0 = caller's guess (read from the output array)
  const int rc = gmres_solve<RV, R>(ctx, adjoint ? 1 : 0, o, info);
  if (rc < 0) return rc;
  TM_CUDA(store_c64<R>(ctx, vec<R>(ctx, 0), out));
  TM_CUDA(stream_wait(ctx));
  return rc;
}

}  // namespace

extern "C" {

int tm_set_tmatrices(tm_ctx* ctx, int n_types, int diag_only, const tm_c64* T, const int* type_of, const double* r_enclosing) {
  if (!ctx) return TM_E_INVALID;
  if (n_types < 1 || !T || !type_of) return fail(ctx, TM_E_INVALID, "need n_types >= 1, T and type_of");
  std::vector<int> ht(ctx->n_scat);
  TM_CUDA(cudaMemcpy(ht.data(), type_of, ht.size() * sizeof(int), is_device_ptr(type_of) ? cudaMemcpyDeviceToHost : cudaMemcpyHostToHost));
  for (int v : ht) if (v < 0 || v >= n_types) return fail(ctx, TM_E_INVALID, "type_of out of range");
  TM_CUDA(stream_wait(ctx));
  if (r_enclosing) {
    for (int t = 0; t < n_types; ++t)
      if (!(r_enclosing[t] >= 0.0)) return fail(ctx, TM_E_INVALID, "negative enclosing radius");
    int *d_flag = nullptr, *d_wp = nullptr, *d_ty = nullptr; double* d_r = nullptr; int h_flag = 0;
    cudaError_t e = tm_dev_alloc(&d_flag, sizeof(int));
    if (e == cudaSuccess) e = cudaMemset(d_flag, 0, sizeof(int));
    if (e == cudaSuccess) e = tm_dev_alloc(&d_wp, (ctx->n_win + 1) * sizeof(int));
    if (e == cudaSuccess) e = cudaMemcpy(d_wp, ctx->win_ptr.data(), (ctx->n_win + 1) * sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = tm_dev_alloc(&d_ty, ht.size() * sizeof(int));
    if (e == cudaSuccess) e = cudaMemcpy(d_ty, ht.data(), ht.size() * sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = tm_dev_alloc(&d_r, n_types * sizeof(double));
    if (e == cudaSuccess) e = cudaMemcpy(d_r, r_enclosing, n_types * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
      k_check_overlap<<<(ctx->n_scat + 127) / 128, 128>>>(ctx->d_pos, ctx->d_win_of, d_wp, d_ty, d_r, ctx->n_scat, d_flag);
      e = cudaMemcpy(&h_flag, d_flag, sizeof(int), cudaMemcpyDeviceToHost);
    }
    tm_dev_free(d_flag); tm_dev_free(d_wp); tm_dev_free(d_ty); tm_dev_free(d_r);
    TM_CUDA(e);
    if (h_flag) return fail(ctx, TM_E_OVERLAP, "enclosing spheres of two scatterers intersect (PAPER.md:275)");
  }
  const size_t count = (size_t)n_types * ctx->L * (diag_only ? 1 : ctx->L);
  void* newT = nullptr;
  TM_CUDA(tm_dev_alloc(&newT, count * elem_bytes(ctx)));
  void* oldT = ctx->d_T;
  ctx->d_T = newT;
  int rc = ctx->precision != TM_FP32 ? set_T_typed<double>(ctx, count, T, newT) : set_T_typed<float>(ctx, count, T, newT);
  if (rc == TM_OK && ctx->precision == TM_MIXED) {            // fp32 copy for the inner Krylov cycles
    void* new32 = nullptr;
    if (tm_dev_alloc(&new32, count * sizeof(Cx<float>)) != cudaSuccess) rc = fail(ctx, TM_E_NOMEM, "tm_dev_alloc(T fp32)");
    else if ((rc = set_T_typed<float>(ctx, count, T, new32)) == TM_OK) { tm_dev_free(ctx->d_T32); ctx->d_T32 = new32; }
    else tm_dev_free(new32);
  }
  if (rc != TM_OK) { tm_dev_free(newT); ctx->d_T = oldT; return rc; }
  tm_dev_free(oldT);
  TM_CUDA(cudaMemcpy(ctx->d_type_of, ht.data(), ht.size() * sizeof(int), cudaMemcpyHostToDevice));
  ctx->n_types = n_types; ctx->diag = diag_only ? 1 : 0; ctx->has_T = true; ctx->T_version++;
  return TM_OK;
}

int tm_set_incident(tm_ctx* ctx, int kind, const void* desc) {
  if (!ctx) return TM_E_INVALID;
  if (!desc) return fail(ctx, TM_E_INVALID, "desc is NULL");
  const int L = ctx->L, lmax = ctx->lmax, LH = L / 2;
  if (kind == TM_INC_COEFFS) {
    const tm_coeffs_desc* d = static_cast<const tm_coeffs_desc*>(desc);
    if (!d->p) return fail(ctx, TM_E_INVALID, "p is NULL");
    TM_CUDA(copy_in(ctx->d_p, d->p, ctx->n * sizeof(double2), ctx->stream));
    TM_CUDA(stream_wait(ctx));
  } else if (kind == TM_INC_PLANE) {
    // Eq. II7 (explicit right-hand forms, reading R9b):
    //   a_{l,m,0} = -4 i^l     e^{-i m alpha} c_l [ i m pibar A_beta + taubar A_alpha ]
    //   a_{l,m,1} = -4 i^{l+1} e^{-i m alpha} c_l [ taubar A_beta - i m pibar A_alpha ]
    const tm_plane_desc* d = static_cast<const tm_plane_desc*>(desc);
    if (!std::isfinite(d->beta) || !std::isfinite(d->alpha)) return fail(ctx, TM_E_INVALID, "non-finite angles");
    double P[TM_MAX_LMAX + 1][TM_MAX_LMAX + 1], PI[TM_MAX_LMAX + 1][TM_MAX_LMAX + 1], TAU[TM_MAX_LMAX + 1][TM_MAX_LMAX + 1];
    ang_functions<TM_MAX_LMAX>(std::cos(d->beta), std::fabs(std::sin(d->beta)), P, PI, TAU);
    // beta in [0, pi] assumed; sin(beta) >= 0
    const cd Ab(d->A_beta.re, d->A_beta.im), Aa(d->A_alpha.re, d->A_alpha.im), I(0.0, 1.0);
    std::vector<cd> a(L);
    for (int l = 1; l <= lmax; ++l) {
      const double cl = 1.0 / std::sqrt(2.0 * l * (l + 1));
      const cd il = std::pow(I, l), il1 = std::pow(I, l + 1);
      for (int m = -l; m <= l; ++m) {
        const int am = std::abs(m);
        const cd e = std::exp(-I * (double)m * d->alpha);
        const double mpi = m * PI[l][am], tau = TAU[l][am];
        const int a0 = l * (l + 1) - 1 + m;
        a[a0] = -4.0 * il * e * cl * (I * mpi * Ab + tau * Aa);
        a[LH + a0] = -4.0 * il1 * e * cl * (tau * Ab - I * mpi * Aa);
      }
    }
    double2* d_a = nullptr;
    TM_CUDA(scratch_get(ctx, 0, L * sizeof(double2), reinterpret_cast<void**>(&d_a)));
    cudaError_t e = cudaMemcpyAsync(d_a, a.data(), L * sizeof(double2), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) {
      const double sb = std::sin(d->beta);
      const double cbt = std::cos(d->beta), ca = std::cos(d->alpha), sa = std::sin(d->alpha);
      ctx->inc_kvec[0] = ctx->k * sb * ca; ctx->inc_kvec[1] = ctx->k * sb * sa; ctx->inc_kvec[2] = ctx->k * cbt;
      // E0 = A_beta beta_hat + A_alpha alpha_hat,  beta_hat = (cb ca, cb sa, -sb), alpha_hat = (-sa, ca, 0)
      const cd ex = Ab * (cbt * ca) - Aa * sa, ey = Ab * (cbt * sa) + Aa * ca, ez = -Ab * sb;
      ctx->inc_e0[0] = make_double2(ex.real(), ex.imag()); ctx->inc_e0[1] = make_double2(ey.real(), ey.imag());
      ctx->inc_e0[2] = make_double2(ez.real(), ez.imag());
      const size_t tot = ctx->n;
      k_incident_plane<<<(unsigned)((tot + 255) / 256), 256, 0, ctx->stream>>>(ctx->d_pos, ctx->n_scat, L, d_a,
          ctx->k * sb * std::cos(d->alpha), ctx->k * sb * std::sin(d->alpha), ctx->k * std::cos(d->beta), ctx->d_p);
      ctx->total_launches++;
      e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = stream_wait(ctx);
    TM_CUDA(e);
  } else if (kind == TM_INC_GAUSS || kind == TM_INC_JINC) {
    // both are angular-spectrum sources (Eqs. II9-II17): per window a list of source centres with transverse amplitudes
    std::vector<double> hsrc;
    std::vector<double2> hamp;
    std::vector<int> hptr(ctx->n_win + 1);
    int nb_req = 0;
    double kw = -1.0, bmax = 0.5 * M_PI;                 // jinc: flat spectrum on [0, pi/2]
    if (kind == TM_INC_GAUSS) {
      const tm_gauss_desc* d = static_cast<const tm_gauss_desc*>(desc);
      if (!d->focus || !(d->w0 > 0.0)) return fail(ctx, TM_E_INVALID, "need focus[n_win][3] and w0 > 0");
      hsrc.assign(d->focus, d->focus + (size_t)ctx->n_win * 3);
      for (int w = 0; w < ctx->n_win; ++w) {
        hamp.push_back(make_double2(d->Ax.re, d->Ax.im)); hamp.push_back(make_double2(d->Ay.re, d->Ay.im));
        hptr[w] = w;
      }
      hptr[ctx->n_win] = ctx->n_win;
      nb_req = d->n_beta;
      // beta in [0, beta_max]: G(beta) < 1e-40 beyond (or pi/2: evanescent part dropped, reading R9)
      kw = ctx->k * d->w0;
      bmax = std::asin(std::min(1.0, 2.0 * std::sqrt(40.0 * std::log(10.0)) / kw));
    } else {
      const tm_jinc_desc* d = static_cast<const tm_jinc_desc*>(desc);
      if (d->n_src < 0 || !d->src_ptr || (d->n_src > 0 && (!d->src_xyz || !d->amp)))
        return fail(ctx, TM_E_INVALID, "need src_xyz, amp and src_ptr");
      hptr.assign(d->src_ptr, d->src_ptr + ctx->n_win + 1);
      if (hptr[0] != 0 || hptr[ctx->n_win] != d->n_src) return fail(ctx, TM_E_INVALID, "src_ptr must start at 0 and end at n_src");
      for (int w = 0; w < ctx->n_win; ++w) if (hptr[w + 1] < hptr[w]) return fail(ctx, TM_E_INVALID, "src_ptr must be monotone");
      hsrc.assign(d->src_xyz, d->src_xyz + (size_t)d->n_src * 3);
      // reading R17: a sample of the band-limited field on the lambda/2 grid is carried by a jinc source of amplitude (pi/2) x sample
      const double nyq = d->amp_is_sample ? 0.5 * M_PI : 1.0;
      for (int sidx = 0; sidx < 2 * d->n_src; ++sidx) hamp.push_back(make_double2(nyq * d->amp[sidx].re, nyq * d->amp[sidx].im));
      nb_req = d->n_beta;
    }
    const size_t nsrc = hsrc.size() / 3;
    // Default node count: 400 (reading R9: part of the definition for the configs), raised when the geometry needs more.
    // The integrand J_n(k rho sin b) e^{i k z cos b} turns by at most k D radians per unit of beta, D = source - scatterer
    // distance, so [0, beta_max] holds k D beta_max / (2 pi) periods; Gauss-Legendre resolves an oscillatory integrand with
    // about pi nodes per period plus a margin:  n >= k D_max beta_max / 2 + 40  (D_max over the pairs of each window).
    int nb = nb_req > 0 ? nb_req : 400;
    if (nb_req <= 0 && nsrc > 0) {
      double dmax2 = 0.0;
      for (int w = 0; w < ctx->n_win; ++w) {
        const int i0 = ctx->win_ptr[w], i1 = ctx->win_ptr[w + 1];
        if (i1 <= i0 || hptr[w + 1] <= hptr[w]) continue;
        double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
        for (int i = i0; i < i1; ++i)
          for (int a = 0; a < 3; ++a) { lo[a] = std::min(lo[a], ctx->h_pos[3 * (size_t)i + a]); hi[a] = std::max(hi[a], ctx->h_pos[3 * (size_t)i + a]); }
        for (int sidx = hptr[w]; sidx < hptr[w + 1]; ++sidx) {
          double d2 = 0.0;
          for (int a = 0; a < 3; ++a) { const double x = hsrc[3 * (size_t)sidx + a]; const double d = std::max(std::fabs(x - lo[a]), std::fabs(x - hi[a])); d2 += d * d; }
          dmax2 = std::max(dmax2, d2);
        }
      }
      const double need = 0.5 * ctx->k * std::sqrt(dmax2) * bmax + 40.0;
      if (need > nb) nb = (int)std::min(65536.0, std::ceil(need / 8.0) * 8.0);
    }
    ctx->inc_src = hsrc; ctx->inc_amp = hamp; ctx->inc_kw = kw; ctx->inc_bmax = bmax; ctx->inc_nb = nb;
    std::vector<double> xg, wg, beta(nb), wq(nb);
    gauss_legendre(nb, xg, wg);
    for (int q = 0; q < nb; ++q) { beta[q] = 0.5 * bmax * (xg[q] + 1.0); wq[q] = 0.5 * bmax * wg[q]; }
    double *d_beta = nullptr, *d_wq = nullptr, *d_src = nullptr; double2* d_amp = nullptr; int* d_ptr = nullptr; void* d_nodes = nullptr;
    const size_t node_bytes = sizeof(GaussNode<TM_MAX_LMAX>);      // upper bound for every lmax
    cudaError_t e = tm_dev_alloc(&d_beta, nb * sizeof(double));
    if (e == cudaSuccess) e = tm_dev_alloc(&d_wq, nb * sizeof(double));
    if (e == cudaSuccess) e = tm_dev_alloc(&d_src, std::max<size_t>(1, nsrc) * 3 * sizeof(double));
    if (e == cudaSuccess) e = tm_dev_alloc(&d_amp, std::max<size_t>(1, nsrc) * 2 * sizeof(double2));
    if (e == cudaSuccess) e = tm_dev_alloc(&d_ptr, (ctx->n_win + 1) * sizeof(int));
    if (e == cudaSuccess) e = tm_dev_alloc(&d_nodes, nb * node_bytes);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_beta, beta.data(), nb * sizeof(double), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_wq, wq.data(), nb * sizeof(double), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess && nsrc) e = cudaMemcpyAsync(d_src, hsrc.data(), nsrc * 3 * sizeof(double), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess && nsrc) e = cudaMemcpyAsync(d_amp, hamp.data(), nsrc * 2 * sizeof(double2), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_ptr, hptr.data(), (ctx->n_win + 1) * sizeof(int), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) {
#define TM_GAUSS(LM)                                                                                                   \
  k_gauss_nodes<LM><<<(nb + 127) / 128, 128, 0, ctx->stream>>>(d_beta, d_wq, nb, kw, static_cast<GaussNode<LM>*>(d_nodes)); \
  k_incident_gauss<LM><<<ctx->n_scat, 128, 0, ctx->stream>>>(ctx->d_pos, ctx->d_win_of, d_src, d_amp, d_ptr,            \
                                                            static_cast<GaussNode<LM>*>(d_nodes), nb, ctx->k, ctx->d_p)
#define TM_GAUSS_MODES(LM)      /* lmax >= 4: warp per scatterer, lane per (l, m >= 0) group, factorised node sums */    \
  k_gauss_nodes<LM><<<(nb + 127) / 128, 128, 0, ctx->stream>>>(d_beta, d_wq, nb, kw, static_cast<GaussNode<LM>*>(d_nodes)); \
  k_incident_modes<LM><<<(ctx->n_scat + 3) / 4, 128, 0, ctx->stream>>>(ctx->d_pos, ctx->d_win_of, d_src, d_amp, d_ptr,  \
                                                            static_cast<GaussNode<LM>*>(d_nodes), nb, ctx->k, ctx->n_scat, ctx->d_p)
      switch (lmax) {
        case 1: TM_GAUSS(1); break;
        case 2: TM_GAUSS(2); break;
        case 3: TM_GAUSS(3); break;
        case 4: TM_GAUSS_MODES(4); break;
        case 5: TM_GAUSS_MODES(5); break;
        default: TM_GAUSS_MODES(6); break;
      }
#undef TM_GAUSS
#undef TM_GAUSS_MODES
      ctx->total_launches += 2;
      e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = stream_wait(ctx);   // the host vectors above must outlive the copies
    tm_dev_free(d_beta); tm_dev_free(d_wq); tm_dev_free(d_src); tm_dev_free(d_amp); tm_dev_free(d_ptr); tm_dev_free(d_nodes);
    TM_CUDA(e);
  } else {
    return fail(ctx, TM_E_INVALID, "unknown incident kind");
  }
  ctx->has_inc = true;
  ctx->inc_kind = kind;
  return TM_OK;
}

int tm_get_incident(tm_ctx* ctx, tm_c64* p_out) {
  if (!ctx) return TM_E_INVALID;
  if (!ctx->has_inc) return fail(ctx, TM_E_STATE, "tm_set_incident has not been called");
  if (!p_out) return fail(ctx, TM_E_INVALID, "p_out is NULL");
  TM_CUDA(copy_out(p_out, ctx->d_p, ctx->n * sizeof(double2), ctx->stream));
  TM_CUDA(stream_wait(ctx));
  return TM_OK;
}

int tm_matvec(tm_ctx* ctx, int transpose, const tm_c64* x, tm_c64* y) {
  if (!ctx) return TM_E_INVALID;
  if (!x || !y || transpose < 0 || transpose > 2) return fail(ctx, TM_E_INVALID, "bad arguments");
  if (transpose != 2 && !ctx->has_T) return fail(ctx, TM_E_STATE, "tm_set_tmatrices has not been called");
  return ctx->precision != TM_FP32 ? matvec_typed<double>(ctx, transpose, x, y) : matvec_typed<float>(ctx, transpose, x, y);
}

int tm_solve(tm_ctx* ctx, const tm_solve_opts* opts, tm_c64* s_out, tm_solve_info* info) {
  if (!ctx) return TM_E_INVALID;
  int rc = check_opts(ctx, opts);
  if (rc != TM_OK) return rc;
  if (!s_out) return fail(ctx, TM_E_INVALID, "s_out is NULL");
  if (!ctx->has_T || !ctx->has_inc) return fail(ctx, TM_E_STATE, "tm_set_tmatrices and tm_set_incident must be called first");
  if ((rc = ensure_workspace(ctx, opts->restart)) != TM_OK) return rc;
  if ((rc = ensure_gmres(ctx, opts->restart)) != TM_OK) return rc;
  if (ctx->precision == TM_MIXED) return solve_typed<float, double>(ctx, 0, nullptr, *opts, s_out, info);
  return ctx->precision == TM_FP64 ? solve_typed<double, double>(ctx, 0, nullptr, *opts, s_out, info)
                                   : solve_typed<float, float>(ctx, 0, nullptr, *opts, s_out, info);
}

int tm_solve_adjoint(tm_ctx* ctx, const tm_c64* w, const tm_solve_opts* opts, tm_c64* lambda_out, tm_solve_info* info) {
  if (!ctx) return TM_E_INVALID;
  int rc = check_opts(ctx, opts);
  if (rc != TM_OK) return rc;
  if (!w || !lambda_out) return fail(ctx, TM_E_INVALID, "w or lambda_out is NULL");
  if (!ctx->has_T) return fail(ctx, TM_E_STATE, "tm_set_tmatrices must be called first");
  if ((rc = ensure_workspace(ctx, opts->restart)) != TM_OK) return rc;
  if ((rc = ensure_gmres(ctx, opts->restart)) != TM_OK) return rc;
  if (ctx->precision == TM_MIXED) return solve_typed<float, double>(ctx, 1, w, *opts, lambda_out, info);
  return ctx->precision == TM_FP64 ? solve_typed<double, double>(ctx, 1, w, *opts, lambda_out, info)
                                   : solve_typed<float, float>(ctx, 1, w, *opts, lambda_out, info);
}

// Several right-hand sides on ONE geometry (both polarisations; many sources): the geometry is
// replicated as one set of windows per right-hand side on an auxiliary context (created at the first call for this n_rhs and
// kept; T is cloned device to device and re-cloned after tm_set_tmatrices), so every right-hand side has its own Krylov scalars
// and convergence mask and all of them share every launch of the batched solver.
int tm_solve_multi(tm_ctx* ctx, int adjoint, int n_rhs, const tm_c64* rhs, const tm_solve_opts* opts, tm_c64* out, tm_solve_info* info) {
  if (!ctx) return TM_E_INVALID;
  int rc = check_opts(ctx, opts);
  if (rc != TM_OK) return rc;
  if (n_rhs < 1 || n_rhs > 64 || !rhs || !out) return fail(ctx, TM_E_INVALID, "need 1 <= n_rhs <= 64, rhs and out");
  if (!ctx->has_T) return fail(ctx, TM_E_STATE, "tm_set_tmatrices must be called first");
  if ((long long)ctx->n * n_rhs > 0x7fffffffLL) return fail(ctx, TM_E_INVALID, "n_rhs * n_scat * L must fit in int32");
  TM_CUDA(stream_wait(ctx));
  if (ctx->multi_aux && ctx->multi_rhs != n_rhs) { tm_destroy(ctx->multi_aux); ctx->multi_aux = nullptr; }
  if (!ctx->multi_aux) {
    const size_t N = ctx->n_scat;
    std::vector<double> pos(3 * N * n_rhs);
    std::vector<int> wp((size_t)ctx->n_win * n_rhs + 1);
    for (int r = 0; r < n_rhs; ++r) {
      std::copy(ctx->h_pos.begin(), ctx->h_pos.end(), pos.begin() + 3 * N * r);
      for (int w = 0; w <= ctx->n_win; ++w) wp[(size_t)r * ctx->n_win + w] = ctx->win_ptr[w] + (int)(N * r);
    }
    rc = create_ctx(&ctx->multi_aux, (int)(N * n_rhs), pos.data(), ctx->n_win * n_rhs, wp.data(), ctx->lmax, ctx->k, ctx->precision,
                    ctx->stream, TM_MAX_LMAX);
    if (rc != TM_OK) return fail(ctx, rc, "auxiliary multi-RHS context: " + g_create_error);
    ctx->multi_rhs = n_rhs; ctx->multi_T_version = -1;
    if (ctx->kernel_req != TM_KERNEL_AUTO) { ctx->multi_aux->kernel_req = ctx->kernel_req; configure_kernel(ctx->multi_aux); }
  }
  tm_ctx* ax = ctx->multi_aux;
  if (ctx->multi_T_version != ctx->T_version) {          // clone T (and its fp32 copy) device to device; replicate type_of
    const size_t count = (size_t)ctx->n_types * ctx->L * (ctx->diag ? 1 : ctx->L);
    tm_dev_free(ax->d_T); tm_dev_free(ax->d_T32); ax->d_T = nullptr; ax->d_T32 = nullptr;
    TM_CUDA(tm_dev_alloc(&ax->d_T, count * elem_bytes(ctx)));
    TM_CUDA(cudaMemcpy(ax->d_T, ctx->d_T, count * elem_bytes(ctx), cudaMemcpyDeviceToDevice));
    if (ctx->d_T32) {
      TM_CUDA(tm_dev_alloc(&ax->d_T32, count * sizeof(Cx<float>)));
      TM_CUDA(cudaMemcpy(ax->d_T32, ctx->d_T32, count * sizeof(Cx<float>), cudaMemcpyDeviceToDevice));
    }
    for (int r = 0; r < n_rhs; ++r)
      TM_CUDA(cudaMemcpy(ax->d_type_of + (size_t)r * ctx->n_scat, ctx->d_type_of, ctx->n_scat * sizeof(int), cudaMemcpyDeviceToDevice));
    ax->n_types = ctx->n_types; ax->diag = ctx->diag; ax->has_T = true; ax->T_version++;
    ctx->multi_T_version = ctx->T_version;
  }
  ax->time_kernels = false;
  if (!adjoint) {                                         // rhs = incident coefficients p of every right-hand side; b = T p
    TM_CUDA(copy_in(ax->d_p, rhs, ax->n * sizeof(double2), ax->stream));
    ax->has_inc = true; ax->inc_kind = TM_INC_COEFFS;
  }
  if ((rc = ensure_workspace(ax, opts->restart)) != TM_OK) return fail(ctx, rc, ax->err);
  if ((rc = ensure_gmres(ax, opts->restart)) != TM_OK) return fail(ctx, rc, ax->err);
  const tm_c64* w = adjoint ? rhs : nullptr;
  if (ctx->precision == TM_MIXED) rc = solve_typed<float, double>(ax, adjoint ? 1 : 0, w, *opts, out, info);
  else rc = ctx->precision == TM_FP64 ? solve_typed<double, double>(ax, adjoint ? 1 : 0, w, *opts, out, info)
                                      : solve_typed<float, float>(ax, adjoint ? 1 : 0, w, *opts, out, info);
  if (rc < 0) return fail(ctx, rc, ax->err);
  ctx->allpairs_launches += ax->allpairs_launches; ctx->total_launches += ax->total_launches;
  ax->allpairs_launches = 0; ax->total_launches = 0;
  return rc;
}

int tm_fields(tm_ctx* ctx, int n_pts, const double* pts, const tm_c64* s, int which, tm_c64* out) {
  if (!ctx) return TM_E_INVALID;
  if (which == TM_FIELD_E_INC) {
    if (n_pts < 1 || !pts || !out) return fail(ctx, TM_E_INVALID, "bad arguments");
    if (!ctx->has_inc || ctx->inc_kind == TM_INC_COEFFS || ctx->inc_kind < 0)
      return fail(ctx, TM_E_STATE, "TM_FIELD_E_INC needs a plane-wave, Gaussian-beam or jinc incident field");
    const size_t nout = (size_t)n_pts * 3;
    double* d_pts = nullptr; double2* d_out = nullptr;
    cudaError_t e = scratch_get(ctx, 1, nout * sizeof(double), reinterpret_cast<void**>(&d_pts));
    if (e == cudaSuccess) e = scratch_get(ctx, 3, nout * sizeof(double2), reinterpret_cast<void**>(&d_out));
    if (e == cudaSuccess) e = copy_in(d_pts, pts, nout * sizeof(double), ctx->stream);
    if (e == cudaSuccess && ctx->inc_kind == TM_INC_PLANE) {
      k_inc_field_plane<<<(n_pts + 127) / 128, 128, 0, ctx->stream>>>(d_pts, n_pts, ctx->inc_kvec[0], ctx->inc_kvec[1], ctx->inc_kvec[2],
                                                                      ctx->inc_e0[0], ctx->inc_e0[1], ctx->inc_e0[2], d_out);
      e = cudaGetLastError();
    } else if (e == cudaSuccess) {
      const int nb = ctx->inc_nb;
      const size_t nsrc = ctx->inc_src.size() / 3;
      std::vector<double> xg, wg, tab(3 * (size_t)nb);          // [w G sin | cos | sin]
      gauss_legendre(nb, xg, wg);
      for (int q = 0; q < nb; ++q) {
        const double b = 0.5 * ctx->inc_bmax * (xg[q] + 1.0), sbq = std::sin(b), kw = ctx->inc_kw;
        tab[q] = 0.5 * ctx->inc_bmax * wg[q] * (kw > 0.0 ? 0.5 * kw * kw * std::exp(-0.25 * kw * kw * sbq * sbq) : 1.0) * sbq;
        tab[nb + q] = std::cos(b); tab[2 * (size_t)nb + q] = sbq;
      }
      double *d_tab = nullptr, *d_src = nullptr; double2* d_amp = nullptr;
      e = scratch_get(ctx, 4, tab.size() * sizeof(double), reinterpret_cast<void**>(&d_tab));
      if (e == cudaSuccess) e = scratch_get(ctx, 5, std::max<size_t>(1, nsrc) * 3 * sizeof(double), reinterpret_cast<void**>(&d_src));
      if (e == cudaSuccess) e = scratch_get(ctx, 6, std::max<size_t>(1, nsrc) * 2 * sizeof(double2), reinterpret_cast<void**>(&d_amp));
      if (e == cudaSuccess) e = cudaMemcpyAsync(d_tab, tab.data(), tab.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream);
      if (e == cudaSuccess && nsrc) e = cudaMemcpyAsync(d_src, ctx->inc_src.data(), nsrc * 3 * sizeof(double), cudaMemcpyHostToDevice, ctx->stream);
      if (e == cudaSuccess && nsrc) e = cudaMemcpyAsync(d_amp, ctx->inc_amp.data(), nsrc * 2 * sizeof(double2), cudaMemcpyHostToDevice, ctx->stream);
      if (e == cudaSuccess) {
        k_inc_field_beams<<<(n_pts + 127) / 128, 128, 0, ctx->stream>>>(d_pts, n_pts, d_src, d_amp, (int)nsrc, d_tab, d_tab + nb,
                                                                        d_tab + 2 * (size_t)nb, nb, ctx->k, d_out);
        e = cudaGetLastError();
      }
      if (e == cudaSuccess) e = stream_wait(ctx);             // tab must outlive the copy
    }
    ctx->total_launches += 1;
    if (e == cudaSuccess) e = copy_out(out, d_out, nout * sizeof(double2), ctx->stream);
    if (e == cudaSuccess) e = stream_wait(ctx);
    TM_CUDA(e);
    return TM_OK;
  }
  if (n_pts < 1 || !pts || !s || !out) return fail(ctx, TM_E_INVALID, "bad arguments");
  if (which != TM_FIELD_E_SCA && which != TM_FIELD_H_SCA) return fail(ctx, TM_E_INVALID, "unknown field id");
  // source chunks: the grid (point blocks x chunks) should fill 148 SMs x 3 resident blocks in whole waves; among the chunk
  // counts that leave >= 32 sources per chunk take the one whose last wave is fullest (ties: fewer chunks)
  int nch = 1;
  {
    const long long pb = (n_pts + 127) / 128, slots = 148LL * 3;
    const int max_ch = std::max(1, std::min(64, ctx->n_scat / 32));
    double best = -1.0;
    for (int c = 1; c <= max_ch; ++c) {
      const double waves = (double)(pb * c) / (double)slots;
      const double eff = waves / std::ceil(waves);
      if (eff > best + 0.02) { best = eff; nch = c; }
    }
  }
  double* d_pts = nullptr; double2 *d_part = nullptr, *d_out = nullptr;
  const size_t nout = (size_t)n_pts * 3;
  cudaError_t e = scratch_get(ctx, 1, nout * sizeof(double), reinterpret_cast<void**>(&d_pts));
  if (e == cudaSuccess) e = scratch_get(ctx, 2, nout * nch * sizeof(double2), reinterpret_cast<void**>(&d_part));
  if (e == cudaSuccess) e = scratch_get(ctx, 3, nout * sizeof(double2), reinterpret_cast<void**>(&d_out));
  if (e == cudaSuccess) e = copy_in(d_pts, pts, nout * sizeof(double), ctx->stream);
  if (e == cudaSuccess) e = copy_in(ctx->d_io, s, ctx->n * sizeof(double2), ctx->stream);
  if (e == cudaSuccess) {
    dim3 grid((n_pts + 127) / 128, nch);
    const int swap = which == TM_FIELD_H_SCA ? 1 : 0;
#define TM_FIELDS(LM) k_fields_sym<LM><<<grid, 128, 0, ctx->stream>>>(ctx->d_pos, ctx->n_scat, ctx->d_io, d_pts, n_pts, ctx->k, 1.0 / ctx->k, swap, d_part)
    switch (ctx->lmax) {
      case 1: TM_FIELDS(1); break;
      case 2: TM_FIELDS(2); break;
      case 3: TM_FIELDS(3); break;
      case 4: TM_FIELDS(4); break;
      case 5: TM_FIELDS(5); break;
      default: TM_FIELDS(6); break;
    }
#undef TM_FIELDS
    k_fields_reduce<<<(unsigned)((nout + 255) / 256), 256, 0, ctx->stream>>>(d_part, nch, nout, d_out);
    ctx->total_launches += 2;
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = copy_out(out, d_out, nout * sizeof(double2), ctx->stream);
  if (e == cudaSuccess) e = stream_wait(ctx);
  TM_CUDA(e);
  return TM_OK;
}

int tm_grad_tmatrix(tm_ctx* ctx, const tm_c64* dT, const tm_c64* lambda, const tm_c64* s, tm_c64* out) {
  if (!ctx) return TM_E_INVALID;
  if (!dT || !lambda || !s || !out) return fail(ctx, TM_E_INVALID, "NULL argument");
  if (!ctx->has_T || !ctx->has_inc) return fail(ctx, TM_E_STATE, "tm_set_tmatrices and tm_set_incident must be called first");
  const size_t count = (size_t)ctx->n_types * ctx->L * (ctx->diag ? 1 : ctx->L);
  void* d_dT = nullptr; double2* d_tmp = nullptr; double2* d_out = nullptr;
  cudaError_t e = tm_dev_alloc(&d_dT, count * elem_bytes(ctx));
  if (e == cudaSuccess) e = tm_dev_alloc(&d_tmp, count * sizeof(double2));
  if (e == cudaSuccess) e = tm_dev_alloc(&d_out, (size_t)ctx->n_scat * sizeof(double2));
  if (e == cudaSuccess) e = copy_in(d_tmp, dT, count * sizeof(double2), ctx->stream);
  const bool f64 = ctx->precision != TM_FP32;
  if (e == cudaSuccess) {
    if (f64) k_from_c64<double><<<grid_for(count, 256), 256, 0, ctx->stream>>>(reinterpret_cast<const double*>(d_tmp), reinterpret_cast<Cx<double>*>(d_dT), count);
    else k_from_c64<float><<<grid_for(count, 256), 256, 0, ctx->stream>>>(reinterpret_cast<const double*>(d_tmp), reinterpret_cast<Cx<float>*>(d_dT), count);
    e = cudaGetLastError();
  }
  // v0 = s ; v1 = A s ; v2 = lambda
  if (e == cudaSuccess) e = f64 ? load_c64<double>(ctx, s, vec<double>(ctx, 0)) : load_c64<float>(ctx, s, vec<float>(ctx, 0));
  if (e == cudaSuccess) e = f64 ? apply_operator<double>(ctx, 2, vec<double>(ctx, 0), vec<double>(ctx, 1), vec<double>(ctx, 2), nullptr)
                                : apply_operator<float>(ctx, 2, vec<float>(ctx, 0), vec<float>(ctx, 1), vec<float>(ctx, 2), nullptr);
  if (e == cudaSuccess) e = f64 ? load_c64<double>(ctx, lambda, vec<double>(ctx, 2)) : load_c64<float>(ctx, lambda, vec<float>(ctx, 2));
  if (e == cudaSuccess) {
    const int grid = (ctx->n_scat + 3) / 4;
    if (f64) k_grad_tmatrix<double><<<grid, 128, 0, ctx->stream>>>(ctx->L, ctx->n_scat, vec<double>(ctx, 1), ctx->d_p, vec<double>(ctx, 2),
                                                                  reinterpret_cast<Cx<double>*>(d_dT), ctx->diag, ctx->d_type_of, d_out);
    else k_grad_tmatrix<float><<<grid, 128, 0, ctx->stream>>>(ctx->L, ctx->n_scat, vec<float>(ctx, 1), ctx->d_p, vec<float>(ctx, 2),
                                                              reinterpret_cast<Cx<float>*>(d_dT), ctx->diag, ctx->d_type_of, d_out);
    ctx->total_launches += 2;
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = copy_out(out, d_out, (size_t)ctx->n_scat * sizeof(double2), ctx->stream);
  if (e == cudaSuccess) e = stream_wait(ctx);
  tm_dev_free(d_dT); tm_dev_free(d_tmp); tm_dev_free(d_out);
  TM_CUDA(e);
  return TM_OK;
}

}  // extern "C"

namespace {

// Analytic position gradient (PAPER.md:517-546 Eqs. IV2-IV6; :560 "can be computed analytically").  With
// dA/dd_alpha = k D^alpha A^ext (gen_tables.py: gradient_entries) the two products with the derivative of the translation
// operator become two ORDINARY all-pairs products at lmax + 1 on the auxiliary context `ax` (same positions and windows),
// each followed by the constant sparse contraction k_grad_contract for the three directions at once.
template <typename R>
int grad_positions_typed(tm_ctx* ctx, tm_ctx* ax, const tm_c64* lambda, const tm_c64* s, const tm_c64* dp, tm_c64* out) {
  const size_t n = ctx->n, vb = n * sizeof(Cx<R>);
  const int L = ctx->L, Le = ax->L, N = ctx->n_scat;
  Cx<R>*S = vec<R>(ctx, 0), *LAM = vec<R>(ctx, 2);
  Cx<R>*XP = vec<R>(ax, 0), *V = vec<R>(ax, 1);
  Cx<R>* PMU = nullptr; double2 *d_out = nullptr, *d_dp = nullptr;
  auto cleanup = [&]() { tm_dev_free(PMU); tm_dev_free(d_out); tm_dev_free(d_dp); };
#define TM_G(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { cleanup(); return fail(ctx, TM_E_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); } } while (0)
  TM_G(tm_dev_alloc(&PMU, vb)); TM_G(tm_dev_alloc(&d_out, (size_t)N * 3 * sizeof(double2)));
  TM_G(cudaMemsetAsync(d_out, 0, (size_t)N * 3 * sizeof(double2), ctx->stream));
  TM_G(load_c64<R>(ctx, s, S));
  TM_G(load_c64<R>(ctx, lambda, LAM));
  TM_G(launch_tapply<R>(ctx, 4, LAM, PMU, nullptr));                 // P mu = P T^T lambda
  const int gb = (N + 3) / 4;
  for (int which = 0; which < 2; ++which) {
    const Cx<R>* vecx = which == 0 ? S : PMU;                         // dA s   /   dA (P mu)
    const Cx<R>* left = which == 0 ? PMU : S;                         // mu = P(P mu)  /   P s   (k_grad_contract applies P)
    TM_G(cudaMemsetAsync(XP, 0, ax->n * sizeof(Cx<R>), ctx->stream));
    k_pad_modes<R><<<grid_for(n, 256), 256, 0, ctx->stream>>>(vecx, XP, L, Le, n);
    TM_G(launch_allpairs<R>(ax, XP, nullptr));                        // A^ext (padded vector): rows l' <= lmax + 1
    TM_G(launch_tapply<R>(ax, 2, XP, V, nullptr));
    k_grad_contract<R><<<gb, 128, 0, ctx->stream>>>(L, Le, N, left, V, ctx->d_const, ctx->grad_tab, ctx->k, d_out);
    ctx->total_launches += 4; ctx->allpairs_launches++;
    TM_G(cudaGetLastError());
  }
  if (dp) {                                                          // incident part: mu_j^T dp_j[alpha]
    TM_G(tm_dev_alloc(&d_dp, n * 3 * sizeof(double2)));
    TM_G(copy_in(d_dp, dp, n * 3 * sizeof(double2), ctx->stream));
    for (int alpha = 0; alpha < 3; ++alpha)
      k_bilinear_rows<R, double><<<gb, 128, 0, ctx->stream>>>(L, N, PMU, reinterpret_cast<const Cx<double>*>(d_dp) + (size_t)alpha * L,
                                                             (size_t)3 * L, ctx->d_const, d_out + alpha, 3);
    TM_G(cudaGetLastError());
  }
  TM_G(copy_out(out, d_out, (size_t)N * 3 * sizeof(double2), ctx->stream));
  TM_G(stream_wait(ctx));
#undef TM_G
  cleanup();
  return TM_OK;
}

}  // namespace

extern "C" {

int tm_grad_positions(tm_ctx* ctx, const tm_c64* lambda, const tm_c64* s, const tm_c64* dp, tm_c64* out) {
  if (!ctx) return TM_E_INVALID;
  if (!lambda || !s || !out) return fail(ctx, TM_E_INVALID, "NULL argument");
  if (!ctx->has_T) return fail(ctx, TM_E_STATE, "tm_set_tmatrices must be called first");
  TM_CUDA(stream_wait(ctx));
  if (!ctx->grad_aux) {            // the same layout at lmax + 1 (kept for later calls of an optimisation loop)
    const int rc = create_ctx(&ctx->grad_aux, ctx->n_scat, ctx->d_pos, ctx->n_win, ctx->win_ptr.data(), ctx->lmax + 1, ctx->k,
                              ctx->precision == TM_FP32 ? TM_FP32 : TM_FP64, ctx->stream, TM_INT_LMAX);
    if (rc != TM_OK) return fail(ctx, rc, "auxiliary lmax + 1 context: " + g_create_error);
  }
  if (!ctx->d_grad_tab) {          // D^alpha entries of this lmax
    const TmGradTable& t = tm_grad_tables[ctx->lmax - 1];
    const size_t nn = (size_t)t.n, off_re = (3 * nn + 255) / 256 * 256, bytes = off_re + 2 * nn * sizeof(double);
    std::vector<unsigned char> h(bytes, 0);
    std::memcpy(h.data(), t.alpha, nn); std::memcpy(h.data() + nn, t.row, nn); std::memcpy(h.data() + 2 * nn, t.col, nn);
    std::memcpy(h.data() + off_re, t.re, nn * sizeof(double)); std::memcpy(h.data() + off_re + nn * sizeof(double), t.im, nn * sizeof(double));
    TM_CUDA(tm_dev_alloc(&ctx->d_grad_tab, bytes));
    TM_CUDA(cudaMemcpy(ctx->d_grad_tab, h.data(), bytes, cudaMemcpyHostToDevice));
    const unsigned char* b = static_cast<const unsigned char*>(ctx->d_grad_tab);
    ctx->grad_tab = TmGradDev{t.n, b, b + nn, b + 2 * nn, reinterpret_cast<const double*>(b + off_re),
                              reinterpret_cast<const double*>(b + off_re) + nn};
  }
  return ctx->precision != TM_FP32 ? grad_positions_typed<double>(ctx, ctx->grad_aux, lambda, s, dp, out)
                                   : grad_positions_typed<float>(ctx, ctx->grad_aux, lambda, s, dp, out);
}

int tm_mie_tmatrix(int lmax, double k_b, double radius, tm_c64 eps_r, tm_c64* out);

int tm_mie_tmatrix_dR(int lmax, double k_b, double radius, tm_c64 eps_r, tm_c64* out) {
  if (lmax < 1 || lmax > TM_MAX_LMAX || !(k_b > 0.0) || !(radius > 0.0) || !out) return TM_E_INVALID;
  const int L = tm_num_modes(lmax);
  const double h = 1e-3 * radius;            // relative step: the accuracy does not depend on the caller's length unit
  std::vector<tm_c64> a(L), b(L), c(L), d(L);
  tm_mie_tmatrix(lmax, k_b, radius + h, eps_r, a.data());
  tm_mie_tmatrix(lmax, k_b, radius - h, eps_r, b.data());
  tm_mie_tmatrix(lmax, k_b, radius + 0.5 * h, eps_r, c.data());
  tm_mie_tmatrix(lmax, k_b, radius - 0.5 * h, eps_r, d.data());
  for (int i = 0; i < L; ++i) {          // Richardson: (4 D(h/2) - D(h)) / 3
    const double d1r = (a[i].re - b[i].re) / (2 * h), d1i = (a[i].im - b[i].im) / (2 * h);
    const double d2r = (c[i].re - d[i].re) / h, d2i = (c[i].im - d[i].im) / h;
    out[i].re = (4.0 * d2r - d1r) / 3.0; out[i].im = (4.0 * d2i - d1i) / 3.0;
  }
  return TM_OK;
}

// Lorenz-Mie coefficients (reading R11), x = k_b R, m_r = sqrt(eps_r), psi_l(z) = z j_l(z), xi_l(z) = z h_l^(1)(z):
//   a_l = [m psi_l(mx) psi_l'(x) - psi_l(x) psi_l'(mx)] / [m psi_l(mx) xi_l'(x) - xi_l(x) psi_l'(mx)]
//   b_l = [psi_l(mx) psi_l'(x) - m psi_l(x) psi_l'(mx)] / [psi_l(mx) xi_l'(x) - m xi_l(x) psi_l'(mx)]
//   psi_l'(z) = z j_{l-1}(z) - l j_l(z)   (same for xi_l with h_l)
int tm_mie_tmatrix(int lmax, double k_b, double radius, tm_c64 eps_r, tm_c64* out) {
  if (lmax < 1 || lmax > TM_MAX_LMAX || !(k_b > 0.0) || !(radius > 0.0) || !out) return TM_E_INVALID;
  const double x = k_b * radius;
  const cd mr = std::sqrt(cd(eps_r.re, eps_r.im));
  std::vector<cd> jx, jm;
  std::vector<double> yx;
  sph_jn_complex(lmax, cd(x, 0.0), jx);
  sph_jn_complex(lmax, mr * x, jm);
  sph_yn_real(lmax, x, yx);
  const int LH = lmax * (lmax + 2);
  for (int l = 1; l <= lmax; ++l) {
    const cd z = mr * x;
    const cd psx = x * jx[l], dpsx = x * jx[l - 1] - (double)l * jx[l];
    const cd psm = z * jm[l], dpsm = z * jm[l - 1] - (double)l * jm[l];
    const cd hx = jx[l] + cd(0, 1) * yx[l], hx1 = jx[l - 1] + cd(0, 1) * yx[l - 1];
    const cd xix = x * hx, dxix = x * hx1 - (double)l * hx;
    const cd a = (mr * psm * dpsx - psx * dpsm) / (mr * psm * dxix - xix * dpsm);
    const cd b = (psm * dpsx - mr * psx * dpsm) / (psm * dxix - mr * xix * dpsm);
    for (int m = -l; m <= l; ++m) {
      const int a0 = l * (l + 1) - 1 + m;
      out[a0].re = -b.real(); out[a0].im = -b.imag();              // p = 0 (M-type, magnetic multipoles)
      out[LH + a0].re = -a.real(); out[LH + a0].im = -a.imag();    // p = 1 (N-type, electric multipoles)
    }
  }
  return TM_OK;
}

}  // extern "C"

// ============================================================================================ measurement helpers
namespace {

template <typename R>
__global__ void __launch_bounds__(256) k_fma_peak(R* out, int iters, R a, R b) {
  R x0 = R(threadIdx.x) * R(1e-3), x1 = x0 + R(1), x2 = x0 + R(2), x3 = x0 + R(3), x4 = x0 + R(4), x5 = x0 + R(5),
    x6 = x0 + R(6), x7 = x0 + R(7);
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 16; ++u) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  const R s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
  if (s == R(123.456)) out[0] = s;                      // never true; keeps the chains alive
}

// FP64 tensor-core (DMMA m8n8k4) chains: the number the multi-RHS dense-block route would be bounded by.
__global__ void __launch_bounds__(256) k_dmma_peak(double* out, int iters, double a, double b) {
  double c[8][2];
#pragma unroll
  for (int u = 0; u < 8; ++u) { c[u][0] = threadIdx.x * 1e-3 + u; c[u][1] = threadIdx.x * 2e-3 - u; }
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
      for (int u = 0; u < 8; ++u)
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                     : "+d"(c[u][0]), "+d"(c[u][1]) : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int u = 0; u < 8; ++u) s += c[u][0] + c[u][1];
  if (s == 123.456) out[0] = s;
}

int dmma_peak(double* tflops, cudaStream_t st) {
  double* d = nullptr;
  if (tm_dev_alloc(&d, sizeof(double)) != cudaSuccess) return TM_E_CUDA;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int blocks = 148 * 8, iters = 2048;
  double best = 0.0;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, st);
    k_dmma_peak<<<blocks, 256, 0, st>>>(d, iters, 0.999999, 1e-7);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { tm_dev_free(d); return TM_E_CUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double fl = 2.0 * 8 * 8 * 4 * 8.0 * 4.0 * (double)iters * (256.0 / 32.0) * blocks;   // m8n8k4 = 256 FMA per warp instruction
    if (rep > 0) best = std::max(best, fl / (ms * 1e-3) * 1e-12);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); tm_dev_free(d);
  *tflops = best;
  return TM_OK;
}

template <typename R>
int fma_peak_typed(double* tflops, cudaStream_t st) {
  R* d = nullptr;
  if (tm_dev_alloc(&d, sizeof(R)) != cudaSuccess) return TM_E_CUDA;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int blocks = 148 * 8, iters = 4096;
  double best = 0.0;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, st);
    k_fma_peak<R><<<blocks, 256, 0, st>>>(d, iters, R(0.999999), R(1e-7));
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { tm_dev_free(d); return TM_E_CUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double fl = 2.0 * 8 * 16 * (double)iters * 256.0 * blocks;
    if (rep > 0) best = std::max(best, fl / (ms * 1e-3) * 1e-12);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); tm_dev_free(d);
  *tflops = best;
  return TM_OK;
}

}  // namespace

extern "C" {

int tm_pair_cost(const tm_ctx* ctx, double* fp_instructions, double* flop) {
  if (!ctx) return TM_E_INVALID;
  double inst = 0.0, fl = 0.0;
  if (ctx->kernel == TM_KERNEL_COPLANAR) tm_cost_coplanar(ctx->lmax, &inst, &fl);
  else if (ctx->kernel == TM_KERNEL_ROT3D && tm_rot3d_ws(ctx->lmax)) tm_cost_rot3d_ws(ctx->lmax, &inst, &fl);
  else if (ctx->kernel == TM_KERNEL_ROT3D) tm_cost_rot3d(ctx->lmax, &inst, &fl);
  else if (ctx->kernel == TM_KERNEL_SYM3D) tm_cost_sym3d(ctx->lmax, &inst, &fl);
  else {   // general kernel: per (term, source): 2 MUL + 4 FMA
    const double nt = tm_term_tables[ctx->lmax - 1].n_terms;
    inst = 6.0 * nt; fl = 10.0 * nt;
  }
  if (fp_instructions) *fp_instructions = inst;
  if (flop) *flop = fl;
  return TM_OK;
}

long long tm_debug_guards(int enable, long long* n_blocks) {
  if (cudaDeviceSynchronize() != cudaSuccess) { cudaGetLastError(); return TM_E_CUDA; }
  GuardRegistry& g = guards();
  std::lock_guard<std::mutex> lock(g.mu);
  if (enable >= 0) g.on = enable != 0;
  long long bad = g.violations;
  for (const auto& kv : g.live) bad += guard_damage(kv.first, kv.second);
  if (n_blocks) *n_blocks = g.blocks;
  return bad;
}

int tm_release_cached_memory(void) {
  int dev = 0;
  cudaMemPool_t pool;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetDefaultMemPool(&pool, dev) != cudaSuccess) return TM_E_CUDA;
  if (cudaDeviceSynchronize() != cudaSuccess) return TM_E_CUDA;
  return cudaMemPoolTrimTo(pool, 0) == cudaSuccess ? TM_OK : TM_E_CUDA;
}

}  // extern "C"

namespace {
// Richardson-extrapolated central difference of four T-matrices per shape: T(+h), T(-h), T(+h/2), T(-h/2)
__global__ void k_nullfield_richardson(const double2* __restrict__ T4, double2* __restrict__ dT, size_t LL, size_t total, double inv_h) {
  const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (i >= total) return;
  const size_t shape = i / LL, e = i % LL;
  const double2* t = T4 + shape * 4 * LL + e;
  const double2 a = t[0], b = t[LL], c = t[2 * LL], d = t[3 * LL];
  // (4 D(h/2) - D(h)) / 3,  D(h) = (T(+h) - T(-h)) / 2h
  dT[i] = make_double2((4.0 * (c.x - d.x) - 0.5 * (a.x - b.x)) * inv_h / 3.0, (4.0 * (c.y - d.y) - 0.5 * (a.y - b.y)) * inv_h / 3.0);
}

int nullfield_run(int lmax, int l_int, double k_b, tm_c64 eps_r, int n_shapes, int n_nodes, const double* theta, const double* r,
                  const double* dr_dtheta, const double* weight, tm_c64* out, cudaStream_t st, double richardson_h) {
  const bool deriv = richardson_h > 0.0;
  const int n_gen = deriv ? 4 * n_shapes : n_shapes;
  const size_t nn = (size_t)n_gen * n_nodes, L = (size_t)tm_num_modes(lmax), LL = L * L;
  {   // the surface must be star-shaped about the origin with finite nodes: r > 0, 0 < theta < pi
    std::vector<double> hr(nn), ht(nn);
    if (cudaMemcpy(hr.data(), r, nn * sizeof(double), is_device_ptr(r) ? cudaMemcpyDeviceToHost : cudaMemcpyHostToHost) != cudaSuccess ||
        cudaMemcpy(ht.data(), theta, nn * sizeof(double), is_device_ptr(theta) ? cudaMemcpyDeviceToHost : cudaMemcpyHostToHost) != cudaSuccess) {
      cudaGetLastError(); return TM_E_CUDA;
    }
    for (size_t i = 0; i < nn; ++i)
      if (!(hr[i] > 0.0) || !std::isfinite(hr[i]) || !(ht[i] > 0.0) || !(ht[i] < 3.14159265358979324)) return TM_E_INVALID;
  }
  double* d_in = nullptr; double2* d_T = nullptr; double2* d_dT = nullptr;
  if (tm_dev_alloc(&d_in, 4 * nn * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return TM_E_NOMEM; }
  if (tm_dev_alloc(&d_T, n_gen * LL * sizeof(double2)) != cudaSuccess) { cudaGetLastError(); tm_dev_free(d_in); return TM_E_NOMEM; }
  if (deriv && tm_dev_alloc(&d_dT, n_shapes * LL * sizeof(double2)) != cudaSuccess) {
    cudaGetLastError(); tm_dev_free(d_in); tm_dev_free(d_T); return TM_E_NOMEM;
  }
  const double* src[4] = {theta, r, dr_dtheta, weight};
  cudaError_t e = cudaSuccess;
  for (int i = 0; i < 4 && e == cudaSuccess; ++i) e = copy_in(d_in + i * nn, src[i], nn * sizeof(double), st);
  if (e == cudaSuccess) e = cudaMemsetAsync(d_T, 0, n_gen * LL * sizeof(double2), st);
  if (e == cudaSuccess) {
    const cd ks = k_b * std::sqrt(cd(eps_r.re, eps_r.im));              // principal root: Im k_s >= 0 for a lossy medium
    nullfield::k_nullfield<<<dim3(n_gen, 2 * lmax + 1), nullfield::NT, 0, st>>>(lmax, l_int, k_b, cx<double>(ks.real(), ks.imag()), n_nodes, d_in, d_in + nn,
                                                                      d_in + 2 * nn, d_in + 3 * nn, d_T);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess && deriv) {
    const size_t total = n_shapes * LL;
    k_nullfield_richardson<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(d_T, d_dT, LL, total, 1.0 / richardson_h);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = copy_out(out, deriv ? d_dT : d_T, n_shapes * LL * sizeof(double2), st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  tm_dev_free(d_in); tm_dev_free(d_T); tm_dev_free(d_dT);
  if (e != cudaSuccess) { cudaGetLastError(); return TM_E_CUDA; }
  return TM_OK;
}
}  // namespace

extern "C" {

int tm_nullfield_tmatrix(int lmax, int lmax_internal, double k_b, tm_c64 eps_r, int n_shapes, int n_nodes, const double* theta, const double* r,
                         const double* dr_dtheta, const double* weight, tm_c64* T_out, void* cuda_stream) {
  if (lmax < 1 || lmax > TM_MAX_LMAX || (lmax_internal != 0 && (lmax_internal < lmax || lmax_internal > nullfield::NF_MAX_L)) ||
      !(k_b > 0.0) || !std::isfinite(eps_r.re) || !std::isfinite(eps_r.im) || (eps_r.re == 0.0 && eps_r.im == 0.0) || eps_r.im < 0.0 ||
      (eps_r.im == 0.0 && eps_r.re < 0.0) || n_shapes < 1 || n_nodes < 1 ||
      !theta || !r || !dr_dtheta || !weight || !T_out)
    return TM_E_INVALID;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return TM_E_CUDA; }
  return nullfield_run(lmax, lmax_internal > 0 ? lmax_internal : lmax, k_b, eps_r, n_shapes, n_nodes, theta, r, dr_dtheta, weight, T_out,
                       reinterpret_cast<cudaStream_t>(cuda_stream), 0.0);
}

int tm_nullfield_dtmatrix(int lmax, int lmax_internal, double k_b, tm_c64 eps_r, int n_shapes, int n_nodes, const double* theta, const double* r,
                          const double* dr_dtheta, const double* weight, double h, tm_c64* dT_out, void* cuda_stream) {
  if (lmax < 1 || lmax > TM_MAX_LMAX || (lmax_internal != 0 && (lmax_internal < lmax || lmax_internal > nullfield::NF_MAX_L)) ||
      !(k_b > 0.0) || !std::isfinite(eps_r.re) || !std::isfinite(eps_r.im) || (eps_r.re == 0.0 && eps_r.im == 0.0) || eps_r.im < 0.0 ||
      (eps_r.im == 0.0 && eps_r.re < 0.0) || n_shapes < 1 || n_nodes < 1 ||
      !theta || !r || !dr_dtheta || !weight || !dT_out || !(h > 0.0) || !std::isfinite(h))
    return TM_E_INVALID;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return TM_E_CUDA; }
  return nullfield_run(lmax, lmax_internal > 0 ? lmax_internal : lmax, k_b, eps_r, n_shapes, n_nodes, theta, r, dr_dtheta, weight, dT_out,
                       reinterpret_cast<cudaStream_t>(cuda_stream), h);
}

int tm_ttable_interp(int n_tab, const double* p_tab, long long n_entry, const tm_c64* T_tab, int n_out, const double* p, tm_c64* T_out,
                     tm_c64* dT_out, void* cuda_stream) {
  if (n_tab < 4 || !p_tab || n_entry < 1 || n_entry > 0x7fffffffLL || !T_tab || n_out < 1 || !p || !T_out) return TM_E_INVALID;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return TM_E_CUDA; }
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  {   // nodes: finite and strictly increasing
    std::vector<double> h(n_tab);
    if (cudaMemcpy(h.data(), p_tab, n_tab * sizeof(double), is_device_ptr(p_tab) ? cudaMemcpyDeviceToHost : cudaMemcpyHostToHost) != cudaSuccess) {
      cudaGetLastError(); return TM_E_CUDA;
    }
    for (int i = 0; i < n_tab; ++i)
      if (!std::isfinite(h[i]) || (i > 0 && !(h[i] > h[i - 1]))) return TM_E_INVALID;
  }
  const size_t tab_elems = (size_t)n_tab * n_entry, total = (size_t)n_out * n_entry;
  // host arrays are staged on the device, device arrays are used where they are
  double *s_ptab = nullptr, *s_p = nullptr, *d_w = nullptr;
  double2 *s_tab = nullptr, *s_T = nullptr, *s_dT = nullptr;
  int *d_i0 = nullptr;                                     // [n_out] stencil starts, then the out-of-table flag
  cudaError_t e = cudaSuccess;
  auto release = [&]() {
    tm_dev_free(s_ptab); tm_dev_free(s_p); tm_dev_free(d_w); tm_dev_free(s_tab); tm_dev_free(s_T); tm_dev_free(s_dT); tm_dev_free(d_i0);
  };
  auto nomem = [&]() { cudaGetLastError(); release(); return TM_E_NOMEM; };
  if (tm_dev_alloc(&d_w, (size_t)ttable::TT_NW * n_out * sizeof(double)) != cudaSuccess) return nomem();
  if (tm_dev_alloc(&d_i0, ((size_t)n_out + 1) * sizeof(int)) != cudaSuccess) return nomem();
  const double* d_ptab = p_tab; const double* d_p = p; const double2* d_tab = reinterpret_cast<const double2*>(T_tab);
  double2* d_T = reinterpret_cast<double2*>(T_out); double2* d_dT = reinterpret_cast<double2*>(dT_out);
  if (!is_device_ptr(p_tab)) { if (tm_dev_alloc(&s_ptab, n_tab * sizeof(double)) != cudaSuccess) return nomem(); d_ptab = s_ptab; }
  if (!is_device_ptr(p)) { if (tm_dev_alloc(&s_p, n_out * sizeof(double)) != cudaSuccess) return nomem(); d_p = s_p; }
  if (!is_device_ptr(T_tab)) { if (tm_dev_alloc(&s_tab, tab_elems * sizeof(double2)) != cudaSuccess) return nomem(); d_tab = s_tab; }
  if (!is_device_ptr(T_out)) { if (tm_dev_alloc(&s_T, total * sizeof(double2)) != cudaSuccess) return nomem(); d_T = s_T; }
  if (dT_out && !is_device_ptr(dT_out)) { if (tm_dev_alloc(&s_dT, total * sizeof(double2)) != cudaSuccess) return nomem(); d_dT = s_dT; }
  if (s_ptab) e = cudaMemcpyAsync(s_ptab, p_tab, n_tab * sizeof(double), cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess && s_p) e = cudaMemcpyAsync(s_p, p, n_out * sizeof(double), cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess && s_tab) e = cudaMemcpyAsync(s_tab, T_tab, tab_elems * sizeof(double2), cudaMemcpyHostToDevice, st);
  int* d_bad = d_i0 + n_out;
  if (e == cudaSuccess) e = cudaMemsetAsync(d_bad, 0, sizeof(int), st);
  if (e == cudaSuccess) {
    ttable::k_ttable_weights<<<(n_out + 127) / 128, 128, 0, st>>>(d_ptab, n_tab, d_p, n_out, d_i0, d_w, d_bad);
    const unsigned ne = (unsigned)n_entry;
    if (ne > 256) {
      const unsigned grid = (unsigned)std::min<size_t>((size_t)n_out, (size_t)148 * 8);
      if (d_dT) ttable::k_ttable_apply_wide<true><<<grid, 256, 0, st>>>(d_tab, ne, d_i0, d_w, n_out, d_T, d_dT);
      else ttable::k_ttable_apply_wide<false><<<grid, 256, 0, st>>>(d_tab, ne, d_i0, d_w, n_out, d_T, nullptr);
    } else {
      const size_t per_block = 256 / ne;
      const unsigned grid = (unsigned)std::min<size_t>(((size_t)n_out + per_block - 1) / per_block, (size_t)148 * 8 * 4);
      if (d_dT) ttable::k_ttable_apply_narrow<true><<<grid, 256, 0, st>>>(d_tab, ne, d_i0, d_w, n_out, d_T, d_dT);
      else ttable::k_ttable_apply_narrow<false><<<grid, 256, 0, st>>>(d_tab, ne, d_i0, d_w, n_out, d_T, nullptr);
    }
    e = cudaGetLastError();
  }
  int bad = 0;
  if (e == cudaSuccess) e = cudaMemcpyAsync(&bad, d_bad, sizeof(int), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && s_T) e = cudaMemcpyAsync(T_out, s_T, total * sizeof(double2), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && s_dT) e = cudaMemcpyAsync(dT_out, s_dT, total * sizeof(double2), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  release();
  if (e != cudaSuccess) { cudaGetLastError(); return TM_E_CUDA; }
  return bad ? TM_E_INVALID : TM_OK;
}

int tm_measure_fma_peak(int precision, double* tflops, void* cuda_stream) {
  if (!tflops) return TM_E_INVALID;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return TM_E_CUDA; }
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  if (precision == TM_PEAK_FP64_TENSOR) return dmma_peak(tflops, st);
  return precision == TM_FP32 ? fma_peak_typed<float>(tflops, st) : fma_peak_typed<double>(tflops, st);
}

}  // extern "C"

#ifdef TM_ARN_STAMPS
extern "C" int tm_debug_arn_stamps(unsigned long long* out32) {
  return cudaMemcpyFromSymbol(out32, g_arn_stamps, 32 * sizeof(unsigned long long)) == cudaSuccess ? 0 : -1;
}
extern "C" int tm_debug_fine_stamps(unsigned long long* out64) {
  return cudaMemcpyFromSymbol(out64, g_fine, 64 * sizeof(unsigned long long)) == cudaSuccess ? 0 : -1;
}
#endif
