// tm_fields_static: scattered-field evaluation (Eqs. I13/I24) through an entry point that ALLOCATES NOTHING -
// for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
//
// Same kernels as tm_fields (k_fields_sym: thread per detector point x source chunk; k_fields_reduce: fixed-order sum of the
// chunk partials), but the per-chunk partial sums - the scratch tm_fields takes from the context's cached device buffers - live
// in a file-scope static device array of a fixed, modest size.  Every GPU that loads libtm.so holds that array until the
// process exits.  Consequences, all part of the contract (include/tm.h):
//   * sizes beyond the array are REJECTED (TM_E_INVALID), never served by a hidden allocation;
//   * every call on a device shares the one array: calls that overlap on the GPU (two streams, two host threads, two
//     captured graphs replayed concurrently) race on it - serialise them;
//   * the array keeps the last call's contents.  Nothing has to start at zero here: every partial sum the reduction reads is
//     written by k_fields_sym of the SAME call first (all n_chunk x n_pts x 3 entries, also for an empty source chunk).
// In host code the array's name is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, taken once per device with that device current (static_scratch() below).
#include "../../include/tm.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <mutex>
#include <string>
#include <type_traits>

#include "tm_common.cuh"
#include "tm_special.cuh"
namespace {                      // internal linkage: tm_api.cu instantiates the same kernels
#include "tm_fields.cuh"
}  // namespace

namespace {

constexpr size_t STATIC_SCRATCH_ELEMS = (size_t)1 << 19;      // double2 entries = 8 MiB per GPU
constexpr int STATIC_MAX_PTS = 65536;                         // stated maximum of n_pts (3 * 65536 * 2 chunks fit)
static_assert((size_t)3 * STATIC_MAX_PTS <= STATIC_SCRATCH_ELEMS, "one chunk of the largest point set must fit");

static __device__ __align__(256) double2 g_fields_scratch[STATIC_SCRATCH_ELEMS];

constexpr int MAX_DEV = 64;
std::mutex g_mu;
double2* g_scratch_ptr[MAX_DEV] = {};                         // device address of g_fields_scratch on device i (nullptr: not set up)
thread_local std::string g_err;

int fail_static(int code, const std::string& msg) { g_err = msg; return code; }

// Device address of the scratch array on the CURRENT device; cudaGetSymbolAddress once per device.
int static_scratch(double2** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { cudaGetLastError(); return fail_static(TM_E_CUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e)); }
  if (dev < 0 || dev >= MAX_DEV) return fail_static(TM_E_INVALID, "device ordinal out of range");
  std::lock_guard<std::mutex> lock(g_mu);
  if (g_scratch_ptr[dev] == nullptr) {
    double2* p = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_fields_scratch);
    if (e != cudaSuccess || p == nullptr) {
      cudaGetLastError();
      return fail_static(TM_E_CUDA, std::string("cudaGetSymbolAddress(g_fields_scratch): ") + cudaGetErrorString(e));
    }
    g_scratch_ptr[dev] = p;
  }
  *out = g_scratch_ptr[dev];
  return TM_OK;
}

bool on_device(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" {

const char* tm_fields_static_error(void) { return g_err.c_str(); }

int tm_fields_static_setup(void) {
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return fail_static(TM_E_CUDA, "no CUDA device: libtm has no CPU fallback");
  }
  double2* p = nullptr;
  return static_scratch(&p);
}

int tm_fields_static(int lmax, double k_b, int n_scat, const double* pos_dev, const tm_c64* s_dev, int n_pts,
                     const double* pts_dev, int which, tm_c64* out_dev, void* cuda_stream) {
  if (lmax < 1 || lmax > TM_MAX_LMAX) return fail_static(TM_E_INVALID, "lmax must be in 1..6");
  if (!(k_b > 0.0)) return fail_static(TM_E_INVALID, "k_b must be positive");
  if (n_scat < 1 || n_pts < 1 || !pos_dev || !s_dev || !pts_dev || !out_dev) return fail_static(TM_E_INVALID, "bad sizes or NULL pointer");
  if (which != TM_FIELD_E_SCA && which != TM_FIELD_H_SCA) return fail_static(TM_E_INVALID, "which must be TM_FIELD_E_SCA or TM_FIELD_H_SCA");
  if (n_pts > STATIC_MAX_PTS)
    return fail_static(TM_E_INVALID, "tm_fields_static: n_pts = " + std::to_string(n_pts) + " exceeds the static scratch (maximum " +
                                         std::to_string(STATIC_MAX_PTS) + " points per call): split the point set or use tm_fields");
  if (!on_device(pos_dev) || !on_device(s_dev) || !on_device(pts_dev) || !on_device(out_dev))
    return fail_static(TM_E_INVALID, "tm_fields_static takes DEVICE pointers only (it copies nothing)");
  double2* scratch = nullptr;
  const int rc = static_scratch(&scratch);
  if (rc != TM_OK) return rc;
  // source chunks as in tm_fields, capped by what the static array holds
  const int want = std::max(1, std::min(64, (int)(148LL * 8 * 128 / n_pts)));
  int nch = std::min(want, std::max(1, n_scat / 32));
  nch = std::max(1, std::min<int>(nch, (int)(STATIC_SCRATCH_ELEMS / ((size_t)3 * n_pts))));
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const size_t nout = (size_t)n_pts * 3;
  const dim3 grid((n_pts + 127) / 128, nch);
  const int swap = which == TM_FIELD_H_SCA ? 1 : 0;
  const double2* s2 = reinterpret_cast<const double2*>(s_dev);
#define TM_FIELDS_S(LM) k_fields_sym<LM><<<grid, 128, 0, st>>>(pos_dev, n_scat, s2, pts_dev, n_pts, k_b, 1.0 / k_b, swap, scratch)
  switch (lmax) {
    case 1: TM_FIELDS_S(1); break;
    case 2: TM_FIELDS_S(2); break;
    case 3: TM_FIELDS_S(3); break;
    case 4: TM_FIELDS_S(4); break;
    case 5: TM_FIELDS_S(5); break;
    default: TM_FIELDS_S(6); break;
  }
#undef TM_FIELDS_S
  k_fields_reduce<<<(unsigned)((nout + 255) / 256), 256, 0, st>>>(scratch, nch, nout, reinterpret_cast<double2*>(out_dev));
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail_static(TM_E_CUDA, std::string("tm_fields_static launch: ") + cudaGetErrorString(e));
  return TM_OK;
}

}  // extern "C"
