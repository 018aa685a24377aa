// sc_ivr_fourier_static (include/sc_ivr.h): the direct-sum Fourier stage of Eq. 11 for callers that
// cannot allocate device memory.
//
// Who that is.  sc_ivr_fourier wants a workspace, and somebody has to cudaMalloc it.  Some callers have nobody who can:
//   - a host program that handed all of HBM to its own pool at start-up (a framework's caching allocator, a simulation
//     code's arena) -- a later cudaMalloc from a plug-in simply fails there, and the plug-in has no handle on the pool;
//   - a step inside a latency-bound loop (instrument control, an online analysis between two acquisitions): cudaMalloc and
//     cudaFree take the driver's allocation lock and synchronise the device, so their cost is neither small nor bounded;
//   - a process that runs under a fixed device-memory budget (MPS client limit, a partitioned job) that is already spent.
// For them the scratch of this one stage (the zero-padded copy of z that the tiled kernel reads, and the twiddle table
// W[c][i] = e^{i E_i c dt}) lives in a file-scope __device__ array of SC_IVR_STATIC_SCRATCH_BYTES.  It is part of the
// library's device image: a GPU holds these bytes from the moment the CUDA runtime loads this part of the library on it (at
// the latest the first call here; with eager module loading, as soon as the library is used on that GPU at all) until the
// process exits.  Nothing here calls cudaMalloc, cudaFree, cudaMemcpy or any routine that allocates; the caller passes the
// input z, the energies and the output, all in device memory.
//
// The array's name in HOST code is only a handle for the runtime: it is not a device address (a kernel handed
// `g_fourier_scratch` from the host would fault, or quietly scribble over host memory on systems where the GPU can reach
// it).  The device address comes from cudaGetSymbolAddress, asked once per device with that device current, below.
//
// The kernels are the ones sc_ivr_fourier launches (spectrum.cu: k_twiddle, k_fourier), so the numbers are the same.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>

#include <mutex>

#include "common.cuh"

namespace {

static __device__ __align__(256) unsigned char g_fourier_scratch[SC_IVR_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_addr_mutex;
unsigned char *g_scratch_addr[kMaxDevices];  // device address of g_fourier_scratch on device d; nullptr = not asked yet

thread_local char g_static_err[384] = "";

sc_ivr_status fail_static(sc_ivr_status st, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_static_err, sizeof(g_static_err), fmt, ap);
  va_end(ap);
  return st;
}

inline size_t up256(size_t x) { return (x + 255) / 256 * 256; }
inline long long up_ll(long long x, long long a) { return (x + a - 1) / a * a; }

// Set-up, once per device: the address of the array in the CURRENT device's copy of the library image.
cudaError_t scratch_of_current_device(unsigned char **out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_addr_mutex);
  if (g_scratch_addr[dev] == nullptr) {
    unsigned char *p = nullptr;
    e = cudaGetSymbolAddress((void **)&p, g_fourier_scratch);
    if (e != cudaSuccess) return e;
    if (p == nullptr) return cudaErrorInvalidSymbol;
    g_scratch_addr[dev] = p;
  }
  *out = g_scratch_addr[dev];
  return cudaSuccess;
}

// Padded copy of the caller's z[c][j] (rows x n) into zp[c][j] (zrows x ncp).  EVERY element of the padded block is written,
// so whatever the previous call left in the array is gone: the padding rows and columns, which the tiled kernel sums over,
// are zero, and nothing else of the array is read before it is written (the twiddle kernel fills all of W).
__global__ void __launch_bounds__(256) k_stage_z(const double2 *__restrict__ z, long long n, int rows, double2 *__restrict__ zp,
                                                 long long ncp, int zrows) {
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= (long long)zrows * ncp) return;
  const long long c = e / ncp, j = e - c * ncp;
  zp[e] = (c < rows && j < n) ? z[c * n + j] : make_double2(0.0, 0.0);
}

// bytes of the array a call needs; 0 = arguments out of range or the products overflow what the array could hold anyway
size_t scratch_need(long long n, int nsteps, int k, long long *ncp_out, int *zrows_out, int *kp_out) {
  const long long cap = (long long)SC_IVR_STATIC_SCRATCH_BYTES / (long long)sizeof(double2);  // elements
  if (n < 1 || k < 1 || nsteps < 0 || n > cap || k > cap || nsteps >= cap) return 0;
  const long long ncp = up_ll(n, SCI_TJ), kp = up_ll(k, SCI_TI), zrows = up_ll((long long)nsteps + 1, SCI_KC);
  if (ncp_out) *ncp_out = ncp;
  if (zrows_out) *zrows_out = (int)zrows;
  if (kp_out) *kp_out = (int)kp;
  return up256(sizeof(double2) * (size_t)zrows * (size_t)ncp) + up256(sizeof(double2) * (size_t)zrows * (size_t)kp);
}

}  // namespace

extern "C" {

const char *sc_ivr_fourier_static_last_error(void) { return g_static_err; }

size_t sc_ivr_fourier_static_scratch_bytes(long long n, int nsteps, int k) { return scratch_need(n, nsteps, k, nullptr, nullptr, nullptr); }

sc_ivr_status sc_ivr_fourier_static(const double *z, long long n, int nsteps, double dt, const double *E, int k, double *A_out,
                                    void *cuda_stream) {
  if (!z || !E || !A_out) return fail_static(SC_IVR_EINVAL, "NULL argument");
  if (n < 1 || k < 1 || nsteps < 0) return fail_static(SC_IVR_EINVAL, "need n >= 1, k >= 1, nsteps >= 0");
  if (!isfinite(dt)) return fail_static(SC_IVR_EINVAL, "dt is not finite");
  long long ncp = 0;
  int zrows = 0, kp = 0;
  const size_t need = scratch_need(n, nsteps, k, &ncp, &zrows, &kp);
  if (need == 0 || need > (size_t)SC_IVR_STATIC_SCRATCH_BYTES)
    return fail_static(SC_IVR_EINVAL,
                       "n = %lld, nsteps = %d, k = %d need %zu bytes of scratch; the static array holds %zu "
                       "(16 (ceil16(nsteps+1)) (ceil128(n) + ceil64(k)) must fit): split the call or use sc_ivr_fourier with a workspace",
                       n, nsteps, k, need, (size_t)SC_IVR_STATIC_SCRATCH_BYTES);
  unsigned char *base = nullptr;
  cudaError_t e = scratch_of_current_device(&base);
  if (e != cudaSuccess) return fail_static(SC_IVR_ECUDA, "cudaGetSymbolAddress(static scratch): %s", cudaGetErrorString(e));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  double2 *zp = (double2 *)base;
  double2 *W = (double2 *)(base + up256(sizeof(double2) * (size_t)zrows * (size_t)ncp));
  const long long nel = (long long)zrows * ncp;
  k_stage_z<<<(unsigned)((nel + 255) / 256), 256, 0, st>>>((const double2 *)z, n, nsteps + 1, zp, ncp, zrows);
  if ((e = cudaGetLastError()) != cudaSuccess) return fail_static(SC_IVR_ECUDA, "k_stage_z: %s", cudaGetErrorString(e));
  if ((e = sci_launch_twiddle(E, k, kp, zrows, dt, W, st)) != cudaSuccess)
    return fail_static(SC_IVR_ECUDA, "twiddle kernel: %s", cudaGetErrorString(e));
  if ((e = sci_launch_fourier(zp, ncp, ncp, zrows, W, kp, n, nullptr, nullptr, (double2 *)A_out, k, st)) != cudaSuccess)
    return fail_static(SC_IVR_ECUDA, "Fourier kernel: %s", cudaGetErrorString(e));
  return SC_IVR_OK;
}

}  // extern "C"
