// Spectrum stage: z assembly (a5 phase branch + a6 + a8 input), twiddle table, Fourier contraction with
// fused |.|^2 and per-tile trajectory reduction (a8, a9), and the fixed-order final reduction (a9).
#include "common.cuh"

namespace {

// ---- z assembly: one thread per trajectory walks its time series ---------------------------------------
// record (ln|<chi|pq>|, S + arg<chi|pq>, Re D, Im D), D = det 2K.  Steps ii and iv of DESIGN.md "Algorithm":
//   u^ = principal sqrt(D/|D|);  if Re(u^ conj(u_prev)) < 0 then u^ = -u^   (continuous branch, R6)
//   z_c = exp(a) * e^{i(S + b)} * u                                            (Eq. 11)
// Also (debug) the unwrapped angle theta = sum wrap(arg D_c - arg D_{c-1}).
__global__ void __launch_bounds__(128) k_zassemble(const double4 *__restrict__ raw, long long raw_stride, long long nb,
                                                   int nsteps, double2 *__restrict__ z, long long zstride, long long zcols,
                                                   int zrows, double *__restrict__ theta_out) {
  const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= zcols) return;
  if (j >= nb) {  // padding columns of the z matrix
    if (z != nullptr)
      for (int c = 0; c < zrows; c++) z[(long long)c * zstride + j] = make_double2(0.0, 0.0);
    return;
  }
  double upr = 1.0, upi = 0.0;
  double theta = 0.0, arg_prev = 0.0;
  const double PI = 3.14159265358979323846;
  for (int c = 0; c <= nsteps; c++) {
    double4 r = raw[(long long)c * raw_stride + j];
    const double inv = unit_scale(r.z, r.w);
    const double x = r.z * inv, y = r.w * inv;
    double ur, ui;
    if (x >= 0.0) {
      ur = sqrt(0.5 * (1.0 + x));
      ui = 0.5 * y / ur;
    } else {
      ui = copysign(sqrt(0.5 * (1.0 - x)), y);
      ur = 0.5 * y / ui;
    }
    if (ur * upr + ui * upi < 0.0) {
      ur = -ur;
      ui = -ui;
    }
    upr = ur;
    upi = ui;
    if (z != nullptr) {
      const double ea = exp(r.x);
      double s, co;
      sincos(r.y, &s, &co);
      z[(long long)c * zstride + j] = make_double2(ea * (co * ur - s * ui), ea * (co * ui + s * ur));
    }
    if (theta_out != nullptr) {
      const double arg = atan2(r.w, r.z);
      double d = arg - arg_prev;
      if (d > PI) d -= 2.0 * PI;
      if (d <= -PI) d += 2.0 * PI;
      theta += d;
      arg_prev = arg;
    }
  }
  if (z != nullptr)
    for (int c = nsteps + 1; c < zrows; c++) z[(long long)c * zstride + j] = make_double2(0.0, 0.0);
  if (theta_out != nullptr) theta_out[j] = theta;
}

// ---- twiddle table W[c][i] = exp(i E_i (c dt)), trajectory independent (Eq. 11) ----------------------------
__global__ void k_twiddle(const double *__restrict__ E, int k, int kp, int rows, double dt, double2 *__restrict__ W) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int c = blockIdx.y;
  if (i >= kp || c >= rows) return;
  double s = 0.0, co = 0.0;
  if (i < k) sincos(E[i] * ((double)c * dt), &s, &co);
  W[(long long)c * kp + i] = make_double2(co, s);
}

// ---- Fourier contraction A[j][i] = sum_c z[c][j] W[c][i], fused |A|^2 * w_j, summed over the tile's trajectories -----
// CTA tile 128 trajectories x 64 energies, 256 threads, thread tile 8 x 4 complex accumulators in registers.
// Warp = 4 (trajectory) x 8 (energy) threads so that every LDS.128 of a fragment is one wavefront.
constexpr int TJ = SCI_TJ, TI = SCI_TI, KC = SCI_KC;
constexpr int FTHREADS = 256;
constexpr int STAGES = 3;

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }

__global__ void __launch_bounds__(FTHREADS, 1) k_fourier(const double2 *__restrict__ z, long long zstride, int zrows,
                                                         const double2 *__restrict__ W, int kp, long long nb,
                                                         const double *__restrict__ wg, double *__restrict__ partial,
                                                         double2 *__restrict__ A_out, int k) {
  extern __shared__ double2 sm2[];
  double2 *zs = sm2;                       // [STAGES][KC][TJ]
  double2 *wsm = sm2 + STAGES * KC * TJ;   // [STAGES][KC][TI]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tx = lane & 7, ty = lane >> 3;  // 8 energy x 4 trajectory threads per warp
  const int wx = warp & 1, wy = warp >> 1;  // 2 x 4 warps
  const int i0 = blockIdx.x * TI;
  const long long j0 = (long long)blockIdx.y * TJ;
  const int nchunks = zrows / KC;

  auto load_stage = [&](int chunk, int stage) {
    const int c0 = chunk * KC;
    double2 *zd = zs + stage * KC * TJ;
    double2 *wd = wsm + stage * KC * TI;
#pragma unroll
    for (int t = 0; t < KC * TJ / FTHREADS; t++) {
      const int e = tid + t * FTHREADS;
      const int r = e / TJ, col = e % TJ;
      cp_async16(zd + e, z + (long long)(c0 + r) * zstride + j0 + col);
    }
#pragma unroll
    for (int t = 0; t < KC * TI / FTHREADS; t++) {
      const int e = tid + t * FTHREADS;
      const int r = e / TI, col = e % TI;
      cp_async16(wd + e, W + (long long)(c0 + r) * kp + i0 + col);
    }
  };

  double are[8][4], aim[8][4];
#pragma unroll
  for (int r = 0; r < 8; r++)
#pragma unroll
    for (int s = 0; s < 4; s++) are[r][s] = aim[r][s] = 0.0;

#pragma unroll
  for (int s = 0; s < STAGES - 1; s++) {
    if (s < nchunks) load_stage(s, s);
    cp_async_commit();
  }
  for (int ch = 0; ch < nchunks; ch++) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    {
      const int nx = ch + STAGES - 1;
      if (nx < nchunks) load_stage(nx, nx % STAGES);
      cp_async_commit();
    }
    const double2 *zc = zs + (ch % STAGES) * KC * TJ + wy * 32 + ty;
    const double2 *wc = wsm + (ch % STAGES) * KC * TI + wx * 32 + tx;
#pragma unroll
    for (int kk = 0; kk < KC; kk++) {
      double2 zf[8], wf[4];
#pragma unroll
      for (int r = 0; r < 8; r++) zf[r] = zc[kk * TJ + 4 * r];
#pragma unroll
      for (int s = 0; s < 4; s++) wf[s] = wc[kk * TI + 8 * s];
#pragma unroll
      for (int r = 0; r < 8; r++)
#pragma unroll
        for (int s = 0; s < 4; s++) {
          are[r][s] = fma(zf[r].x, wf[s].x, are[r][s]);
          are[r][s] = fma(-zf[r].y, wf[s].y, are[r][s]);
          aim[r][s] = fma(zf[r].x, wf[s].y, aim[r][s]);
          aim[r][s] = fma(zf[r].y, wf[s].x, aim[r][s]);
        }
    }
  }
  cp_async_wait<0>();
  __syncthreads();

  // epilogue: |A|^2 w_j, fixed-order sum over the tile's 128 trajectories (no atomics)
  if (A_out != nullptr) {
#pragma unroll
    for (int r = 0; r < 8; r++) {
      const long long j = j0 + wy * 32 + ty + 4 * r;
#pragma unroll
      for (int s = 0; s < 4; s++) {
        const int i = i0 + wx * 32 + tx + 8 * s;
        if (j < nb && i < k) A_out[j * k + i] = make_double2(are[r][s], aim[r][s]);
      }
    }
  }
  if (partial == nullptr) return;
  double ps[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
  for (int r = 0; r < 8; r++) {
    const long long j = j0 + wy * 32 + ty + 4 * r;
    const double w = (j < nb) ? wg[j] : 0.0;
#pragma unroll
    for (int s = 0; s < 4; s++) {
      const double m = fma(are[r][s], are[r][s], aim[r][s] * aim[r][s]);
      ps[s] += (w != 0.0) ? w * m : 0.0;  // a rejected trajectory may carry NaN: select, never multiply
    }
  }
#pragma unroll
  for (int s = 0; s < 4; s++) {
    ps[s] += __shfl_xor_sync(0xffffffffu, ps[s], 8);
    ps[s] += __shfl_xor_sync(0xffffffffu, ps[s], 16);
  }
  double *redbuf = reinterpret_cast<double *>(sm2);  // [4 wy][64]
  if (ty == 0) {
#pragma unroll
    for (int s = 0; s < 4; s++) redbuf[wy * TI + wx * 32 + tx + 8 * s] = ps[s];
  }
  __syncthreads();
  if (tid < TI) {
    const double v = ((redbuf[tid] + redbuf[TI + tid]) + redbuf[2 * TI + tid]) + redbuf[3 * TI + tid];
    partial[(long long)blockIdx.y * kp + i0 + tid] = v;
  }
}

__global__ void k_weights(const double *__restrict__ w, const unsigned char *__restrict__ good, long long n,
                          double *__restrict__ wg) {
  const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (j < n) wg[j] = good[j] ? (w ? w[j] : 1.0) : 0.0;
}

// single block: integer count, order irrelevant
__global__ void k_count_good(const unsigned char *__restrict__ good, long long n, long long *ngood, int accumulate) {
  __shared__ long long sh[256];
  long long s = 0;
  for (long long j = threadIdx.x; j < n; j += blockDim.x) s += good[j] ? 1 : 0;
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) *ngood = (accumulate ? *ngood : 0) + sh[0];
}

// I[i] = norm / n_good * sum over tiles in index order (a9; deterministic)
__global__ void k_final(const double *__restrict__ partial, long long ntiles, int kp, int k,
                        const long long *__restrict__ ngood, double norm, double *__restrict__ I_out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= k) return;
  double s = 0.0;
  for (long long t = 0; t < ntiles; t++) s += partial[t * kp + i];
  const long long ng = *ngood;
  I_out[i] = ng > 0 ? s * (norm / (double)ng) : 0.0;
}

// ---- FP64 probes (measurement only) ------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_probe_dfma(int iters, double *out) {
  double a[16];
  const double x = 1.0 + 1e-9 * threadIdx.x, y = 1e-9;
#pragma unroll
  for (int i = 0; i < 16; i++) a[i] = (double)i;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 16; i++) a[i] = fma(a[i], x, y);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; i++) s += a[i];
  if (s == 12345.678) out[0] = s;
}

__global__ void __launch_bounds__(256) k_probe_dmma(int iters, double *out) {
  double c[8][2];
  const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * (threadIdx.x + 1);
#pragma unroll
  for (int i = 0; i < 8; i++) c[i][0] = c[i][1] = (double)i;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 8; i++)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                   : "+d"(c[i][0]), "+d"(c[i][1])
                   : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
  if (s == 12345.678) out[0] = s;
}

// Issue-budget probes (kernel A "what bounds it"): the DFMA loop of k_probe_dfma with ONE other instruction after every
// NF DFMAs, so that the time per DFMA says whether that instruction issues in the shadow of the FP64 pipe or takes a slot of its own.
//   MIX 2: a 64-bit warp shuffle (two SHFL.IDX) every 4 DFMAs     MIX 3: an LDS.64 every 4 DFMAs (its value is the next addend)
//   MIX 4: one integer LOP3 / IADD3 pair after EVERY DFMA
// Only the DFMAs are counted as flop.
template <int MIX>
__global__ void __launch_bounds__(256) k_probe_mix(int iters, double *out) {
  __shared__ double tab[512];
  tab[threadIdx.x] = 1e-9 * (threadIdx.x + 1);
  tab[256 + threadIdx.x] = 2e-9 * (threadIdx.x + 1);
  __syncthreads();
  // nothing but the DFMA chains themselves is a dependent chain: a loaded value is first used a whole iteration (16 DFMAs)
  // later, the 16 integer counters are independent of one another, a shuffled accumulator is next touched 13 DFMAs later
  double a[16], yv[4];
  unsigned k[16];
  const double x = 1.0 + 1e-9 * threadIdx.x;
#pragma unroll
  for (int i = 0; i < 16; i++) {
    a[i] = (double)i;
    k[i] = threadIdx.x + i;
  }
#pragma unroll
  for (int i = 0; i < 4; i++) yv[i] = 1e-9;
  for (int it = 0; it < iters; it++) {
    double yn[4] = {yv[0], yv[1], yv[2], yv[3]};
    const double *tp = tab + ((threadIdx.x + it) & 255);
#pragma unroll
    for (int i = 0; i < 16; i++) {
      a[i] = fma(a[i], x, yv[i >> 2]);
      if (MIX == 2 && (i & 3) == 3) a[i - 3] = __shfl_xor_sync(0xffffffffu, a[i - 3], 1);
      if (MIX == 3 && (i & 3) == 3) yn[i >> 2] = tp[i];
      if (MIX == 4) k[i] = (k[i] ^ (unsigned)it) + (unsigned)i;
    }
#pragma unroll
    for (int i = 0; i < 4; i++) yv[i] = yn[i];
  }
  double s = yv[0] + yv[1] + yv[2] + yv[3];
#pragma unroll
  for (int i = 0; i < 16; i++) s += a[i] + (double)(k[i] & 1u);
  if (s == 12345.678) out[0] = s;
}

}  // namespace

cudaError_t sci_launch_zassemble(const double4 *raw, long long raw_stride, long long nb, int nsteps, double2 *z,
                                 long long zstride, long long zcols, int zrows, double *theta_out, cudaStream_t st) {
  const long long n = z ? zcols : nb;
  k_zassemble<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(raw, raw_stride, nb, nsteps, z, zstride, n, zrows, theta_out);
  return cudaGetLastError();
}

cudaError_t sci_launch_twiddle(const double *E_dev, int k, int kp, int rows, double dt, double2 *W, cudaStream_t st) {
  dim3 grid((kp + 255) / 256, rows);
  k_twiddle<<<grid, 256, 0, st>>>(E_dev, k, kp, rows, dt, W);
  return cudaGetLastError();
}

cudaError_t sci_launch_fourier(const double2 *z, long long zstride, long long zcols, int zrows, const double2 *W, int kp,
                               long long nb, const double *wg, double *partial, double2 *A_out, int k, cudaStream_t st) {
  const size_t smem = sizeof(double2) * STAGES * KC * (TJ + TI);
  {  // per device, cheap: set on every launch
    cudaError_t e = cudaFuncSetAttribute(k_fourier, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  dim3 grid(kp / TI, (unsigned)(zcols / TJ));
  k_fourier<<<grid, FTHREADS, smem, st>>>(z, zstride, zrows, W, kp, nb, wg, partial, A_out, k);
  return cudaGetLastError();
}

cudaError_t sci_launch_weights(const double *w, const unsigned char *good, long long n, double *wg, cudaStream_t st) {
  k_weights<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(w, good, n, wg);
  return cudaGetLastError();
}

cudaError_t sci_launch_count_good(const unsigned char *good, long long n, long long *ngood, int accumulate, cudaStream_t st) {
  k_count_good<<<1, 256, 0, st>>>(good, n, ngood, accumulate);
  return cudaGetLastError();
}

cudaError_t sci_launch_final(const double *partial, long long ntiles, int kp, int k, const long long *ngood, double norm,
                             double *I_out, cudaStream_t st) {
  k_final<<<(k + 127) / 128, 128, 0, st>>>(partial, ntiles, kp, k, ngood, norm, I_out);
  return cudaGetLastError();
}

cudaError_t sci_fp64_probe(int mode, int iters, double *flops, double *ms_out) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return e;
  double *d = nullptr;
  e = cudaMalloc(&d, 8);
  if (e != cudaSuccess) return e;
  cudaEvent_t a, b;
  cudaEventCreate(&a);
  cudaEventCreate(&b);
  // mode = kind + 10 * wps.  kind: 0 DFMA, 1 DMMA, 2 DFMA + SHFL, 3 DFMA + LDS, 4 DFMA + integer.  wps: 0 = 16 warps per scheduler
  // (8 CTAs of 256 threads per SM), 1 or 2 = that many warps per scheduler (one CTA of 128 or 256 threads per SM)
  const int kind = mode % 10, wps = mode / 10;
  if (kind > 4 || wps > 2 || mode < 0) {
    cudaFree(d);
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    return cudaErrorInvalidValue;
  }
  const int blocks = wps == 0 ? sms * 8 : sms, threads = wps == 1 ? 128 : 256;
  for (int rep = 0; rep < 2; rep++) {  // first pass is the warm-up
    cudaEventRecord(a);
    if (kind == 0) k_probe_dfma<<<blocks, threads>>>(iters, d);
    else if (kind == 1) k_probe_dmma<<<blocks, threads>>>(iters, d);
    else if (kind == 2) k_probe_mix<2><<<blocks, threads>>>(iters, d);
    else if (kind == 3) k_probe_mix<3><<<blocks, threads>>>(iters, d);
    else k_probe_mix<4><<<blocks, threads>>>(iters, d);
    cudaEventRecord(b);
    e = cudaEventSynchronize(b);
    if (e != cudaSuccess) break;
  }
  float ms = 0.f;
  cudaEventElapsedTime(&ms, a, b);
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  cudaFree(d);
  if (e != cudaSuccess) return e;
  const double fl = kind != 1 ? 2.0 * 16.0 * (double)iters * blocks * threads
                              : 2.0 * 8.0 * 8 * 8 * 4 * (double)iters * blocks * (threads / 32);
  *flops = fl / (ms * 1e-3);
  *ms_out = ms;
  return cudaGetLastError();
}
