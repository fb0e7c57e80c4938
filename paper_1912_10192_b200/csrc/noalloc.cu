// noalloc.cu — ONE entry point that allocates nothing: hamr_divb_noalloc (include/hamr.h).
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
// it).  It is the div B diagnostic of misc.cu (k_divb; C-11; "divergence-free evolution of the
// magnetic field") on caller-supplied dense face arrays, with the scratch memory of its two-pass reduction in a
// file-scope device array of fixed size instead of a grid's arena.  No grid object, no cudaMalloc / cudaFree, no
// allocating library routine; the existing paths are untouched.
//
// The scratch array is shared by every call on a device and keeps the last call's contents.  No slot is accumulated
// into: every slot a call reads, that call has written first (per-block partial maxima [0, nblk), then the reduced
// denominator maximum), so nothing has to start at zero and stale contents are never seen.  Two calls that OVERLAP on
// the GPU (different streams without ordering between them, two host threads) race on it: serialise them.
#include <atomic>
#include <cstdio>
#include "../../include/hamr.h"
#include "hamr_dev.cuh"

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_MAXB = HAMR_NOALLOC_MAX_ZONES / NA_THREADS;   // 65536 blocks of 256 zones
constexpr int NA_DENMAX = 2 * NA_MAXB;                          // slot of the reduced denominator maximum
// [0, MAXB): per-block max denominators; [MAXB, 2 MAXB): per-block max |div| / den; then the denominator maximum.
// 1 MB + 256 B, held by every GPU that loads the library until the process exits.
static __device__ __align__(256) double na_scratch[2 * NA_MAXB + 32];

static_assert(HAMR_NOALLOC_MAX_ZONES % NA_THREADS == 0, "whole blocks");

__device__ __forceinline__ double block_max(double v) {
  __shared__ double wm[NA_THREADS / 32];
  v = hamr::warp_max(v);
  if ((threadIdx.x & 31) == 0) wm[threadIdx.x >> 5] = v;
  __syncthreads();
  double r = 0.0;
  if (threadIdx.x < 32) {
    r = threadIdx.x < NA_THREADS / 32 ? wm[threadIdx.x] : 0.0;
    r = hamr::warp_max(r);
  }
  return r;   // valid in thread 0
}

// dense arrays, x3 fastest: bf0 (n0 + 1, n1, n2), bf1 (n0, n1 + 1, n2), bf2 (n0, n1, n2 + 1).  One thread per zone;
// the arithmetic is that of k_divb (misc.cu), expression for expression.
// PASS 0: per-block maximum of the denominators; PASS 1: of |div| / den over zones with den > 1e-12 max den
template <int PASS>
__global__ void __launch_bounds__(NA_THREADS) k_na_part(double* __restrict__ scr, const double* __restrict__ bf0,
                                                        const double* __restrict__ bf1, const double* __restrict__ bf2,
                                                        int n0, int n1, int n2, double dx0, double dx1, double dx2) {
  const long long tot = (long long)n0 * n1 * n2;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  double val = 0.0;
  if (t < tot) {
    const int k = (int)(t % n2), j = (int)((t / n2) % n1), i = (int)(t / ((long long)n2 * n1));
    const double* a[3] = {bf0 + ((long long)i * n1 + j) * n2 + k, bf1 + ((long long)i * (n1 + 1) + j) * n2 + k,
                          bf2 + ((long long)i * n1 + j) * (n2 + 1) + k};
    const long long S[3] = {(long long)n1 * n2, n2, 1};
    const double dx[3] = {dx0, dx1, dx2};
    double div = 0.0, den = 0.0;
    for (int d = 0; d < 3; d++) {
      const double lo = a[d][0], hi = a[d][S[d]];
      div += (hi - lo) / dx[d];
      den += (fabs(hi) + fabs(lo)) / (2.0 * dx[d]);
    }
    if (PASS == 0) val = den;
    else if (den > 1e-12 * scr[NA_DENMAX]) val = fabs(div) / den;
  }
  val = block_max(val);
  if (threadIdx.x == 0) scr[PASS * NA_MAXB + blockIdx.x] = val;
}

// one block: maximum of the nblk partials of a pass; pass 0 -> the denominator slot, pass 1 -> the caller's output
__global__ void __launch_bounds__(NA_THREADS) k_na_reduce(double* __restrict__ scr, int pass, int nblk,
                                                          double* __restrict__ out) {
  double v = 0.0;
  for (int b = threadIdx.x; b < nblk; b += NA_THREADS) v = hamr::dmax(v, scr[pass * NA_MAXB + b]);
  v = block_max(v);
  if (threadIdx.x == 0) {
    if (pass == 0) scr[NA_DENMAX] = v;
    else *out = v;
  }
}

// device address of the scratch array, per device.  In host code `na_scratch` is a host-side stand-in, not a device
// address: the address comes from cudaGetSymbolAddress, once per device, with that device current.
constexpr int NA_MAXDEV = 64;
std::atomic<double*> na_addr[NA_MAXDEV];
thread_local char na_err[256] = "";

int na_fail(int code, const char* what, cudaError_t e = cudaSuccess) {
  if (e != cudaSuccess) std::snprintf(na_err, sizeof(na_err), "%s: %s", what, cudaGetErrorString(e));
  else std::snprintf(na_err, sizeof(na_err), "%s", what);
  return code;
}

int na_scratch_ptr(double** ptr) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return na_fail(HAMR_ECUDA, "cudaGetDevice", e);
  if (dev >= 0 && dev < NA_MAXDEV) {
    double* p = na_addr[dev].load(std::memory_order_acquire);
    if (p) { *ptr = p; return HAMR_OK; }
  }
  double* p = nullptr;
  e = cudaGetSymbolAddress((void**)&p, na_scratch);
  if (e != cudaSuccess || !p) return na_fail(HAMR_ECUDA, "cudaGetSymbolAddress(na_scratch)", e);
  if (dev >= 0 && dev < NA_MAXDEV) na_addr[dev].store(p, std::memory_order_release);
  *ptr = p;
  return HAMR_OK;
}

}  // namespace

extern "C" {

int hamr_noalloc_setup(void) {
  double* p = nullptr;
  return na_scratch_ptr(&p);
}

const char* hamr_noalloc_last_error(void) { return na_err; }

int hamr_divb_noalloc(const int n[3], const double dx[3], const double* const bface_dev[3], double* out_dev,
                      void* cuda_stream) {
  if (!n || !dx || !bface_dev || !out_dev) return na_fail(HAMR_EINVAL, "hamr_divb_noalloc: null argument");
  if (n[0] < 1 || n[1] < 1 || n[2] < 1) return na_fail(HAMR_EINVAL, "hamr_divb_noalloc: n must be positive");
  if (!(dx[0] > 0.0) || !(dx[1] > 0.0) || !(dx[2] > 0.0)) return na_fail(HAMR_EINVAL, "hamr_divb_noalloc: dx must be positive");
  const long long tot = (long long)n[0] * n[1] * n[2];
  if (tot > (long long)HAMR_NOALLOC_MAX_ZONES) {
    std::snprintf(na_err, sizeof(na_err),
                  "hamr_divb_noalloc: %lld zones exceed HAMR_NOALLOC_MAX_ZONES = %d (the fixed scratch array holds one "
                  "partial result per 256 zones); use hamr_divb on a grid",
                  tot, (int)HAMR_NOALLOC_MAX_ZONES);
    return HAMR_EINVAL;
  }
  if (!bface_dev[0] || !bface_dev[1] || !bface_dev[2]) return na_fail(HAMR_EINVAL, "hamr_divb_noalloc: null face array");
  double* scr = nullptr;
  const int rc = na_scratch_ptr(&scr);
  if (rc != HAMR_OK) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int nblk = (int)((tot + NA_THREADS - 1) / NA_THREADS);
  k_na_part<0><<<nblk, NA_THREADS, 0, st>>>(scr, bface_dev[0], bface_dev[1], bface_dev[2], n[0], n[1], n[2], dx[0], dx[1], dx[2]);
  k_na_reduce<<<1, NA_THREADS, 0, st>>>(scr, 0, nblk, out_dev);
  k_na_part<1><<<nblk, NA_THREADS, 0, st>>>(scr, bface_dev[0], bface_dev[1], bface_dev[2], n[0], n[1], n[2], dx[0], dx[1], dx[2]);
  k_na_reduce<<<1, NA_THREADS, 0, st>>>(scr, 1, nblk, out_dev);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return na_fail(HAMR_ECUDA, "hamr_divb_noalloc: launch", e);
  na_err[0] = 0;
  return HAMR_OK;
}

}  // extern "C"
