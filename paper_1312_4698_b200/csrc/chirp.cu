// Fourier stage for an equally spaced energy grid ("E_1 = E_min ... E_k = E_max" equally spaced):
// the sum of Eq. 11
//     A_j(E_i) = sum_{c=0}^{n} z_{j,c} exp(i E_i c dt),     E_i = E_0 + i dE,
// is a chirp-z transform.  With theta = dE dt and  i c = (i^2 + c^2 - (i - c)^2) / 2,
//     A_i = exp(i theta i^2 / 2) * sum_c [ z_c exp(i (E_0 dt c + theta c^2 / 2)) ] * exp(-i theta (i - c)^2 / 2)
//         = exp(i theta i^2 / 2) * (x * h)_i,      x_c = z_c pc_c,   h_m = exp(-i theta m^2 / 2),  m = -n .. k-1,
// a linear convolution, evaluated exactly (to rounding) as a circular one of length L = 8192 with two FFTs per block of
// B = L - k + 1 time samples (one block when n + k <= L; longer series are split, block b using the filter shifted by
// its offset, h^(b)_m = h_(m - b B), and the blocks' outputs y^(b) are added before the modulus is taken).  Only |A_i|^2 = |(x * h)_i|^2 enters I(E) (Eq. 11), so the outer chirp is never applied.
// Cost per trajectory-step: ~ 2 * 5 L log2 L / (n + 1) = 270 flop instead of 8 k = 32000 for the direct sum.
//
// One CTA transforms one trajectory at a time out of shared memory (L complex doubles = 128 KB + padding) and loops
// over its trajectories (persistent, fixed assignment => fixed summation order, no atomics):
//   forward  DIF passes of radix 16, 16, 32 (natural order in, digit-reversed out; pass 1 reads x from HBM),
//   pointwise product with the filter spectrum Hp (stored in the same digit-reversed order, 1/L folded in),
//   inverse  DIT passes of radix 32, 16, 16 (digit-reversed in, natural out), |y_i|^2 w_j accumulated in shared memory.
// The radix-32 forward pass, the product and the radix-32 inverse pass run on registers without touching memory.
#include "common.cuh"

namespace {

constexpr int CL = SCI_CHIRP_L;       // 8192
constexpr int CT = 256;               // threads per CTA
constexpr int CPAD = CL + CL / 32;    // one element of padding per 32: conflict-free radix-32 pass
__device__ __forceinline__ int phys(int i) { return i + (i >> 5); }

// cos(2 pi k / 32), k = 0..8 (k = 8 is exactly 0); a switch so that unrolled callers fold it to an immediate
__host__ __device__ constexpr double cos32(int k) {
  switch (k) {
    case 0: return 1.0;
    case 1: return 0.9807852804032304491261822;
    case 2: return 0.9238795325112867561281832;
    case 3: return 0.8314696123025452370787884;
    case 4: return 0.7071067811865475244008444;
    case 5: return 0.5555702330196022247428308;
    case 6: return 0.38268343236508977172846;
    case 7: return 0.1950903220161282678482849;
    default: return 0.0;
  }
}
// W_32^k = exp(-2 pi i k / 32) for k = 0..15 from the quarter table
__host__ __device__ constexpr double w32_re(int k) { return k <= 8 ? cos32(k) : -cos32(16 - k); }
__host__ __device__ constexpr double w32_im(int k) { return k <= 8 ? -cos32(8 - k) : -cos32(k - 8); }

template <int R>
__host__ __device__ constexpr int brev(int i) {
  int r = 0;
  for (int b = 1; b < R; b <<= 1) {
    r = (r << 1) | (i & 1);
    i >>= 1;
  }
  return r;
}

// In-register DFT of size R (8, 16 or 32), radix-2 decimation in frequency, all indices compile-time.
// INV = false: v[brev(f)] <- sum_n v[n] exp(-2 pi i f n / R);  INV = true: the conjugate transform.
template <int R, bool INV>
__device__ __forceinline__ void dft_reg(double2 (&v)[R]) {
#pragma unroll
  for (int half = R / 2; half >= 1; half >>= 1) {
    const int step = 16 / half;  // twiddle exponent step in units of W_32 (W_{2 half}^p = W_32^{p * 16 / half})
#pragma unroll
    for (int base = 0; base < R; base += 2 * half) {
#pragma unroll
      for (int p = 0; p < half; p++) {
        const int i = base + p, j = i + half;
        const double2 a = v[i], b = v[j];
        v[i] = make_double2(a.x + b.x, a.y + b.y);
        const double dx = a.x - b.x, dy = a.y - b.y;
        const int e = p * step;  // 0 <= e < 16
        if (e == 0) {
          v[j] = make_double2(dx, dy);
        } else if (e == 8) {  // W = -i (forward), +i (inverse)
          v[j] = INV ? make_double2(-dy, dx) : make_double2(dy, -dx);
        } else {
          const double wr = w32_re(e), wi = INV ? -w32_im(e) : w32_im(e);
          v[j] = make_double2(fma(dx, wr, -dy * wi), fma(dx, wi, dy * wr));
        }
      }
    }
  }
}

// The same transform by decimation in time: input in bit-reversed order (v[brev(f)] = X_f), output in natural order.
template <int R, bool INV>
__device__ __forceinline__ void dft_reg_dit(double2 (&v)[R]) {
#pragma unroll
  for (int half = 1; half < R; half <<= 1) {
    const int step = 16 / half;
#pragma unroll
    for (int base = 0; base < R; base += 2 * half) {
#pragma unroll
      for (int p = 0; p < half; p++) {
        const int i = base + p, j = i + half;
        const double2 a = v[i], b = v[j];
        const int e = p * step;
        double tx, ty;
        if (e == 0) {
          tx = b.x;
          ty = b.y;
        } else if (e == 8) {
          tx = INV ? -b.y : b.y;
          ty = INV ? b.x : -b.x;
        } else {
          const double wr = w32_re(e), wi = INV ? -w32_im(e) : w32_im(e);
          tx = fma(b.x, wr, -b.y * wi);
          ty = fma(b.x, wi, b.y * wr);
        }
        v[i] = make_double2(a.x + tx, a.y + ty);
        v[j] = make_double2(a.x - tx, a.y - ty);
      }
    }
  }
}

__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
  return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ double2 cmulc(double2 a, double2 b) {  // a * conj(b)
  return make_double2(fma(a.x, b.x, a.y * b.y), fma(a.y, b.x, -a.x * b.y));
}

// w^1 .. w^15 from w (products of depth <= 4: a few ulp), tw[0] unused
__device__ __forceinline__ void powers16(double2 w, double2 (&tw)[16]) {
  tw[1] = w;
  tw[2] = cmul(w, w);
  tw[3] = cmul(tw[2], w);
  tw[4] = cmul(tw[2], tw[2]);
  tw[5] = cmul(tw[4], w);
  tw[6] = cmul(tw[3], tw[3]);
  tw[7] = cmul(tw[4], tw[3]);
  tw[8] = cmul(tw[4], tw[4]);
  tw[9] = cmul(tw[8], w);
  tw[10] = cmul(tw[5], tw[5]);
  tw[11] = cmul(tw[8], tw[3]);
  tw[12] = cmul(tw[6], tw[6]);
  tw[13] = cmul(tw[8], tw[5]);
  tw[14] = cmul(tw[7], tw[7]);
  tw[15] = cmul(tw[8], tw[7]);
}

// MODE 0: production.  CTA b transforms rows b, b + gridDim.x, ... of x, accumulates w_j |y_i|^2 (i < k) in registers
//         and writes its partial spectrum to partial[b * kp + i].
// MODE 1: spectrum of one row (the filter): HpT[s * 256 + t] = forward transform / L in the register layout of pass 3.
// MODE 2: parity entry: power[row * k + i] = |y_i|^2 per row.
template <int MODE>
__global__ void __launch_bounds__(CT, 1) k_chirp_fft(const double2 *__restrict__ x, long long xstride, int n1, long long nrows,
                                                     const double2 *__restrict__ HpT, const double *__restrict__ wg, int k,
                                                     int kp, double *__restrict__ out, double2 *__restrict__ spec_out,
                                                     int nblocks, int bsz, double2 *__restrict__ yscr) {
  extern __shared__ double2 S[];
  const int t = threadIdx.x;
  // per-thread base twiddles (fixed for the whole launch): W_L^t, W_L^(t+256), W_512^(t & 31)
  double2 w1[2], w2;
  {
    double s, c;
    sincospi(-2.0 * (double)t / (double)CL, &s, &c);
    w1[0] = make_double2(c, s);
    sincospi(-2.0 * (double)(t + 256) / (double)CL, &s, &c);
    w1[1] = make_double2(c, s);
    sincospi(-2.0 * (double)(t & 31) / 512.0, &s, &c);
    w2 = make_double2(c, s);
  }
  // power accumulators of this CTA, one per output i < kp, behind the FFT buffer in shared memory (thread t owns
  // i = t + 256 b + 512 j: no two threads share an entry, consecutive threads hit consecutive banks)
  double *accs = reinterpret_cast<double *>(S + CPAD);
  if (MODE == 0)
    for (int i = t; i < CL; i += CT) accs[i] = 0.0;

  double2 *ys = (nblocks > 1) ? yscr + (long long)blockIdx.x * CL : nullptr;  // this CTA's running sum of block outputs
  for (long long row = blockIdx.x; row < nrows; row += gridDim.x)
  for (int blk = 0; blk < nblocks; blk++) {
    const double2 *xr = x + row * xstride + (long long)blk * bsz;
    const int n1b = min(bsz, n1 - blk * bsz);
    const double2 *Hb = HpT + (long long)blk * CL;
    // ---- forward pass 1: radix 16 over stride 512, input from HBM (zero beyond n1), twiddle W_L^(n' k1)
#pragma unroll
    for (int b = 0; b < 2; b++) {
      const int np = t + 256 * b;
      double2 v[16];
#pragma unroll
      for (int j = 0; j < 16; j++) {
        const int idx = np + 512 * j;
        v[j] = (idx < n1b) ? xr[idx] : make_double2(0.0, 0.0);
      }
      dft_reg<16, false>(v);
      double2 tw[16];
      powers16(w1[b], tw);
#pragma unroll
      for (int s = 0; s < 16; s++) {
        const int k1 = brev<16>(s);
        S[phys(k1 * 512 + np)] = (k1 == 0) ? v[s] : cmul(v[s], tw[k1]);
      }
    }
    __syncthreads();
    // ---- forward pass 2: radix 16 over stride 32 inside each block of 512, twiddle W_512^(n'' k2)
    {
      double2 tw[16];
      powers16(w2, tw);
#pragma unroll
      for (int b = 0; b < 2; b++) {
        const int q = t + 256 * b, base = (q >> 5) * 512 + (q & 31);
        double2 v[16];
#pragma unroll
        for (int j = 0; j < 16; j++) v[j] = S[phys(base + 32 * j)];
        dft_reg<16, false>(v);
#pragma unroll
        for (int s = 0; s < 16; s++) {
          const int k2 = brev<16>(s);
          S[phys(base + 32 * k2)] = (k2 == 0) ? v[s] : cmul(v[s], tw[k2]);
        }
      }
    }
    __syncthreads();
    // ---- forward pass 3 (radix 32, contiguous), product with the filter spectrum, inverse pass 3: all in registers
    {
      double2 v[32];
#pragma unroll
      for (int j = 0; j < 32; j++) v[j] = S[phys(t * 32 + j)];
      dft_reg<32, false>(v);  // slot s holds f'' = brev32(s)
      if (MODE == 1) {
        const double sc = 1.0 / (double)CL;
#pragma unroll
        for (int s = 0; s < 32; s++) spec_out[s * CT + t] = make_double2(v[s].x * sc, v[s].y * sc);
      } else {
#pragma unroll
        for (int s = 0; s < 32; s++) v[s] = cmul(v[s], Hb[s * CT + t]);
        dft_reg_dit<32, true>(v);  // bit-reversed spectrum in, natural n'' out
#pragma unroll
        for (int j = 0; j < 32; j++) S[phys(t * 32 + j)] = v[j];
      }
    }
    if (MODE == 1) break;
    __syncthreads();
    // ---- inverse pass 2: conj twiddle, radix 16 over k2 (stride 32)
    {
      double2 tw[16];
      powers16(w2, tw);
#pragma unroll
      for (int b = 0; b < 2; b++) {
        const int q = t + 256 * b, base = (q >> 5) * 512 + (q & 31);
        double2 v[16];
#pragma unroll
        for (int k2 = 0; k2 < 16; k2++) {
          const double2 a = S[phys(base + 32 * k2)];
          v[k2] = (k2 == 0) ? a : cmulc(a, tw[k2]);
        }
        dft_reg<16, true>(v);
#pragma unroll
        for (int s = 0; s < 16; s++) S[phys(base + 32 * brev<16>(s))] = v[s];
      }
    }
    __syncthreads();
    // ---- inverse pass 1: conj twiddle, radix 16 over k1 (stride 512); y_i, i = n' + 512 j, stays in registers
    const double w = (MODE == 0 && wg != nullptr) ? wg[row] : 1.0;
#pragma unroll
    for (int b = 0; b < 2; b++) {
      const int np = t + 256 * b;
      double2 tw[16];
      powers16(w1[b], tw);
      double2 v[16];
#pragma unroll
      for (int k1 = 0; k1 < 16; k1++) {
        const double2 a = S[phys(k1 * 512 + np)];
        v[k1] = (k1 == 0) ? a : cmulc(a, tw[k1]);
      }
      dft_reg<16, true>(v);
#pragma unroll
      for (int s = 0; s < 16; s++) {
        const int i = np + 512 * brev<16>(s);
        if (nblocks > 1) {  // y = sum of the blocks' outputs, kept in this CTA's global scratch row between blocks
          if (i < kp) {
            if (blk > 0) {
              const double2 p = ys[i];
              v[s].x += p.x;
              v[s].y += p.y;
            }
            if (blk < nblocks - 1) ys[i] = v[s];
          }
          if (blk < nblocks - 1) continue;
        }
        const double m = fma(v[s].x, v[s].x, v[s].y * v[s].y);
        if (MODE == 0) {
          if (i < kp && w != 0.0) accs[i] = fma(w, m, accs[i]);  // a rejected trajectory may carry NaN: skip, never multiply
        } else if (i < k) {
          out[row * (long long)k + i] = m;
        }
      }
    }
    __syncthreads();
  }
  if (MODE == 0) {
#pragma unroll
    for (int b = 0; b < 2; b++)
#pragma unroll
      for (int s = 0; s < 16; s++) {
        const int i = t + 256 * b + 512 * brev<16>(s);
        if (i < kp) out[(long long)blockIdx.x * kp + i] = accs[i];
      }
  }
}

// pc[c] = exp(i (E_0 dt c + theta c^2 / 2)), c = 0..n1-1, and for each block b (offset c0 = b bsz) the filter row
// hrow[b][(m + L) % L] = exp(-i theta (m - c0)^2 / 2), m = -(bsz-1) .. k-1 (zero elsewhere).  c^2 and (m - c0)^2 are exact
// in double; the phase carries one rounding.
__global__ void k_chirp_tables(double e0dt, double theta, int n1, int k, int nblocks, int bsz, double2 *__restrict__ pc,
                               double2 *__restrict__ hrow) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n1) {
    const double c = (double)i;
    double s, co;
    sincos(fma(0.5 * theta, c * c, e0dt * c), &s, &co);
    pc[i] = make_double2(co, s);
  }
  if (i < CL) {
    int m = i;
    bool in = (m <= k - 1);
    if (!in && i >= CL - (bsz - 1)) {
      m = i - CL;
      in = true;
    }
    for (int b = 0; b < nblocks; b++) {
      double2 v = make_double2(0.0, 0.0);
      if (in) {
        const double mm = (double)(m - b * bsz);
        double s, co;
        sincos(-0.5 * theta * (mm * mm), &s, &co);
        v = make_double2(co, s);
      }
      hrow[(long long)b * CL + i] = v;
    }
  }
}

// z assembly for the chirp path: same arithmetic as k_zassemble (steps ii and iv of DESIGN.md "Algorithm"), times the
// inner chirp pc[c]; output x[j][c] with the time series of a trajectory contiguous.  One warp = 32 trajectories; the
// records are read time-major (coalesced over trajectories), transposed through a padded shared tile and written as
// 512-byte row segments.
#ifndef SCI_ZU
#define SCI_ZU 4
#endif
#ifndef SCI_ZREG
#define SCI_ZREG 128
#endif
__global__ void __maxnreg__(SCI_ZREG) k_zassemble_rows(const double4 *__restrict__ raw, long long raw_stride, long long nb, int nsteps,
                                                        const double2 *__restrict__ pc, double2 *__restrict__ xrows, long long xstride) {
  __shared__ double2 tile[2][32][33];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long j0 = ((long long)blockIdx.x * 2 + warp) * 32;
  if (j0 >= nb) return;
  const long long j = j0 + lane;
  const bool valid = j < nb;
  const long long jr = valid ? j : nb - 1;
  double upr = 1.0, upi = 0.0;
  const int n1 = nsteps + 1;
  for (int c0 = 0; c0 < n1; c0 += 32) {
    const int cn = min(32, n1 - c0);
    for (int cb = 0; cb < cn; cb += SCI_ZU) {
      // SCI_ZU independent record loads in flight before the (sequential) branch rule consumes them
      double4 rec[SCI_ZU];
#pragma unroll
      for (int u = 0; u < SCI_ZU; u++) {
        const int c = min(c0 + cb + u, nsteps);
        rec[u] = raw[(long long)c * raw_stride + jr];
      }
#pragma unroll
      for (int u = 0; u < SCI_ZU; u++) {
        const int cc = cb + u, c = c0 + cc;
        if (cc >= cn) break;
        double4 r = rec[u];
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
        const double ea = exp(r.x);
        double s, co;
        sincos(r.y, &s, &co);
        const double2 z = make_double2(ea * (co * ur - s * ui), ea * (co * ui + s * ur));
        tile[warp][lane][cc] = cmul(z, pc[c]);
      }
    }
    __syncwarp();
    for (int rr = 0; rr < 32; rr++) {
      if (j0 + rr < nb && lane < cn) xrows[(j0 + rr) * xstride + c0 + lane] = tile[warp][rr][lane];
    }
    __syncwarp();
  }
}

// z assembly for reference states that are combinations of coherent states (row f4), in two stages so
// that the (P, Q) stream is read once per batch, not once per reference state:
//   stage 1 (k_overlap_phase, one thread per trajectory, sequential in c for the branch rule R6):
//       ph[c][j]    = e^{i S} u pc[c]                       from the plain records (0, S, Re D, Im D)
//       ov[c][m][j] = exp(a_m + i b_m) = <p_m q_m|p q>      (Eq. 3, reduced coordinates) for every coherent state m
//   stage 2 (k_combine_rows, per reference state n, fully parallel):
//       x_n[j][c]   = ph[c][j] * sum_m conj(eps_nm) ov[c][m][j],   transposed to trajectory-major rows for the chirp-z stage
__global__ void __maxnreg__(128) k_overlap_phase(const double4 *__restrict__ raw, const double2 *__restrict__ pqs, long long raw_stride,
                                                 long long nb, int nsteps, int F, const double *__restrict__ chis, int ncs,
                                                 const double2 *__restrict__ pc, double2 *__restrict__ ovph) {
  const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= nb) return;
  double upr = 1.0, upi = 0.0;
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
    double s, co;
    sincos(r.y, &s, &co);
    double2 *o = ovph + (long long)c * (ncs + 1) * raw_stride + j;
    o[0] = cmul(make_double2(co * ur - s * ui, co * ui + s * ur), pc[c]);
    for (int m = 0; m < ncs; m++) {
      double am = 0.0, bm = 0.0;
      for (int a = 0; a < F; a++) {
        const double2 pq = pqs[((long long)c * F + a) * raw_stride + j];
        const double dq = chis[(2 * m + 1) * F + a] - pq.y, dp = chis[2 * m * F + a] - pq.x;
        am = fma(-0.25, fma(dq, dq, dp * dp), am);
        bm = fma(0.5 * (chis[2 * m * F + a] + pq.x), dq, bm);
      }
      const double ea = exp(am);
      sincos(bm, &s, &co);
      o[(long long)(m + 1) * raw_stride] = make_double2(ea * co, ea * s);
    }
  }
}

__global__ void __launch_bounds__(64) k_combine_rows(const double2 *__restrict__ ovph, long long raw_stride, long long nb, int nsteps,
                                                     const double *__restrict__ eps, int ncs, double2 *__restrict__ xrows,
                                                     long long xstride) {
  __shared__ double2 tile[2][32][33];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long j0 = ((long long)blockIdx.x * 2 + warp) * 32;
  const int c0 = blockIdx.y * 32;
  if (j0 >= nb) return;
  const long long j = (j0 + lane < nb) ? j0 + lane : nb - 1;
  const int cn = min(32, nsteps + 1 - c0);
  for (int cc = 0; cc < cn; cc++) {
    const double2 *o = ovph + (long long)(c0 + cc) * (ncs + 1) * raw_stride + j;
    double wr = 0.0, wi = 0.0;
    for (int m = 0; m < ncs; m++) {
      const double2 v = o[(long long)(m + 1) * raw_stride];
      const double er = eps[2 * m], ei = -eps[2 * m + 1];  // conj(eps_m)
      wr += er * v.x - ei * v.y;
      wi += er * v.y + ei * v.x;
    }
    tile[warp][lane][cc] = cmul(make_double2(wr, wi), o[0]);
  }
  __syncwarp();
  for (int rr = 0; rr < 32; rr++)
    if (j0 + rr < nb && lane < cn) xrows[(j0 + rr) * xstride + c0 + lane] = tile[warp][rr][lane];
}

// parity entry only: x[j][c] = z[c][j] pc[c] from a time-major z series
__global__ void k_rows_from_z(const double2 *__restrict__ z, long long n, int n1, const double2 *__restrict__ pc,
                              double2 *__restrict__ xrows, long long xstride) {
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n * n1) return;
  const long long j = e / n1;
  const int c = (int)(e - j * n1);
  xrows[j * xstride + c] = cmul(z[(long long)c * n + j], pc[c]);
}

}  // namespace

size_t sci_chirp_smem_bytes() { return sizeof(double2) * CPAD + sizeof(double) * CL; }
int sci_chirp_threads() { return CT; }

cudaError_t sci_launch_chirp_tables(double e0dt, double theta, int n1, int k, int nblocks, int bsz, double2 *pc, double2 *hrow,
                                    cudaStream_t st) {
  const int n = n1 > CL ? n1 : CL;
  k_chirp_tables<<<(n + 255) / 256, 256, 0, st>>>(e0dt, theta, n1, k, nblocks, bsz, pc, hrow);
  return cudaGetLastError();
}

cudaError_t sci_launch_zassemble_rows(const double4 *raw, long long raw_stride, long long nb, int nsteps, const double2 *pc,
                                      double2 *xrows, long long xstride, cudaStream_t st) {
  const long long warps = (nb + 31) / 32;
  k_zassemble_rows<<<(unsigned)((warps + 1) / 2), 64, 0, st>>>(raw, raw_stride, nb, nsteps, pc, xrows, xstride);
  return cudaGetLastError();
}

// mode 0: partial spectra (out = partial [grid][kp]); mode 1: filter spectra of the nblocks rows of x (spec_out [nblocks][8192]);
// mode 2: per-row power (out [nrows][k]).  yscr: [grid][8192] complex scratch, needed when nblocks > 1.
cudaError_t sci_launch_chirp_fft(int mode, const double2 *x, long long xstride, int n1, long long nrows, const double2 *HpT,
                                 const double *wg, int k, int kp, double *out, double2 *spec_out, int nblocks, int bsz,
                                 double2 *yscr, int grid, cudaStream_t st) {
  const size_t smem = sci_chirp_smem_bytes();
  {  // the attribute is per device and the call is cheap: set it on every launch (no process-wide flag)
    cudaError_t e = cudaSuccess;
    if (mode == 0) e = cudaFuncSetAttribute(k_chirp_fft<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    else if (mode == 1) e = cudaFuncSetAttribute(k_chirp_fft<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    else e = cudaFuncSetAttribute(k_chirp_fft<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  if (mode == 0) {
    k_chirp_fft<0><<<grid, CT, smem, st>>>(x, xstride, n1, nrows, HpT, wg, k, kp, out, spec_out, nblocks, bsz, yscr);
  } else if (mode == 1) {
    for (int b = 0; b < nblocks; b++)  // one full-length row per block
      k_chirp_fft<1><<<1, CT, smem, st>>>(x + (long long)b * CL, CL, CL, 1, HpT, wg, k, kp, out, spec_out + (long long)b * CL, 1,
                                          CL, nullptr);
  } else {
    k_chirp_fft<2><<<grid, CT, smem, st>>>(x, xstride, n1, nrows, HpT, wg, k, kp, out, spec_out, nblocks, bsz, yscr);
  }
  return cudaGetLastError();
}

cudaError_t sci_launch_rows_from_z(const double2 *z, long long n, int n1, const double2 *pc, double2 *xrows, long long xstride,
                                   cudaStream_t st) {
  const long long tot = n * n1;
  k_rows_from_z<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(z, n, n1, pc, xrows, xstride);
  return cudaGetLastError();
}

cudaError_t sci_launch_overlap_phase(const double4 *raw, const double2 *pq_steps, long long raw_stride, long long nb, int nsteps, int F,
                                     const double *chis_reduced, int ncs, const double2 *pc, double2 *ovph, cudaStream_t st) {
  k_overlap_phase<<<(unsigned)((nb + 127) / 128), 128, 0, st>>>(raw, pq_steps, raw_stride, nb, nsteps, F, chis_reduced, ncs, pc, ovph);
  return cudaGetLastError();
}

cudaError_t sci_launch_combine_rows(const double2 *ovph, long long raw_stride, long long nb, int nsteps, const double *eps, int ncs,
                                    double2 *xrows, long long xstride, cudaStream_t st) {
  const long long warps = (nb + 31) / 32;
  dim3 grid((unsigned)((warps + 1) / 2), (unsigned)((nsteps + 1 + 31) / 32));
  k_combine_rows<<<grid, 64, 0, st>>>(ovph, raw_stride, nb, nsteps, eps, ncs, xrows, xstride);
  return cudaGetLastError();
}
