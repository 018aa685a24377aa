// Kernel A for small systems (F <= 3): ONE THREAD PER TRAJECTORY.
// The whole state (2F + 4F^2 + 1 doubles = 43 at F = 3), H dQ and the working copies of both eliminations fit the
// register file of one thread, so nothing is exchanged between lanes: no shared memory, no shuffles.  The reduced PES
// constants are kernel parameters, i.e. warp-uniform constant-bank operands of the FMAs (no load instructions).
// Same arithmetic as the lane-distributed kernels (propagate_cml.cu): reduced coordinates, generic kick/drift stages,
// fixed-order eliminations with a monitored multiplier growth and a pivoted fallback (here a plain loop over local
// arrays, executed by the rare thread that needs it).
#include "common.cuh"

namespace {

constexpr int kTptThreads = 128;

__device__ __forceinline__ double rcp_nr(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  return r;
}

// dense reduced constants: QFF: phi3[F][F][F], P[F][F], w2[F];  Morse: D[F], a~[F], Qe[F]
template <int F>
struct TC {
  static constexpr int PHI = 0, PP = F * F * F, W2 = PP + F * F, N_QFF = W2 + F, N_MORSE = 3 * F;
};

// a1: V, g[F], H[F][F] (symmetric, full) at Q
template <int F, int KIND>
__device__ __forceinline__ void pes_tpt(const double *__restrict__ c, const double (&Q)[F], double &V, double (&g)[F],
                                        double (&H)[F][F]) {
  using T = TC<F>;
  if (KIND == SC_IVR_PES_QFF) {
    double u[F], q2[F];
#pragma unroll
    for (int j = 0; j < F; j++) q2[j] = Q[j] * Q[j];
    V = 0.0;
#pragma unroll
    for (int a = 0; a < F; a++) {
      double ua = 0.0;
#pragma unroll
      for (int j = 0; j < F; j++) ua = fma(c[T::PP + a * F + j], q2[j], ua);
      u[a] = ua;
    }
#pragma unroll
    for (int a = 0; a < F; a++) {
      double s3 = 0.0;
#pragma unroll
      for (int b = 0; b < F; b++) {
        double h3 = 0.0;
#pragma unroll
        for (int k = 0; k < F; k++) h3 = fma(c[T::PHI + (a * F + b) * F + k], Q[k], h3);
        s3 = fma(h3, Q[b], s3);
        H[a][b] = (a == b) ? c[T::W2 + a] + h3 + 0.5 * u[a] : fma(c[T::PP + a * F + b] * Q[a], Q[b], h3);
      }
      const double w2 = c[T::W2 + a], paa = c[T::PP + a * F + a];
      const double g3 = 0.5 * s3;
      const double g4 = Q[a] * (0.5 * u[a] - (1.0 / 3.0) * paa * q2[a]);
      g[a] = fma(w2, Q[a], g3 + g4);
      V += Q[a] * (0.5 * w2 * Q[a] + (1.0 / 3.0) * g3 + 0.25 * g4);
    }
  } else {
    V = 0.0;
#pragma unroll
    for (int a = 0; a < F; a++) {
      const double D = c[a], at = c[F + a], Qe = c[2 * F + a];
      const double y = exp(-at * (Q[a] - Qe));
      V += D * (1.0 - y) * (1.0 - y);
      g[a] = 2.0 * D * at * y * (1.0 - y);
#pragma unroll
      for (int b = 0; b < F; b++) H[a][b] = (a == b) ? 2.0 * D * at * at * y * (2.0 * y - 1.0) : 0.0;
    }
  }
}

// fixed-order elimination of an N x N real matrix A[row][col]; returns det, grow = largest |multiplier| high word
template <int N>
__device__ __forceinline__ double det_static_real(double (&A)[N][N], unsigned &grow) {
  double det = 1.0;
  unsigned gm = 0u;
#pragma unroll
  for (int k = 0; k < N; k++) {
    det *= A[k][k];
    if (k == N - 1) break;
    const double r = rcp_nr(A[k][k]);
#pragma unroll
    for (int j = k + 1; j < N; j++) {
      const double m = A[k][j] * r;
      gm = max(gm, (unsigned)__double2hiint(m) & 0x7fffffffu);
#pragma unroll
      for (int i = k + 1; i < N; i++) A[i][j] = fma(-m, A[i][k], A[i][j]);
    }
  }
  grow = gm;
  return det;
}

template <int N>
__device__ __forceinline__ void det_static_complex(double (&Ar)[N][N], double (&Ai)[N][N], double &Dre, double &Dim, unsigned &grow) {
  double dr = 1.0, di = 0.0;
  unsigned gk = 0u;
#pragma unroll
  for (int k = 0; k < N; k++) {
    const double t = dr * Ar[k][k] - di * Ai[k][k];
    di = fma(dr, Ai[k][k], di * Ar[k][k]);
    dr = t;
    if (k == N - 1) break;
    const double rn = rcp_nr(fma(Ar[k][k], Ar[k][k], Ai[k][k] * Ai[k][k]));
    const double rx = Ar[k][k] * rn, ry = -Ai[k][k] * rn;
#pragma unroll
    for (int j = k + 1; j < N; j++) {
      const double mr = Ar[k][j] * rx - Ai[k][j] * ry;
      const double mi = fma(Ar[k][j], ry, Ai[k][j] * rx);
      gk = max(gk, max((unsigned)__double2hiint(mr) & 0x7fffffffu, (unsigned)__double2hiint(mi) & 0x7fffffffu));
#pragma unroll
      for (int i = k + 1; i < N; i++) {
        const double pr = Ar[i][k], pi = Ai[i][k];
        Ar[i][j] = fma(-mr, pr, fma(mi, pi, Ar[i][j]));
        Ai[i][j] = fma(-mr, pi, fma(-mi, pr, Ai[i][j]));
      }
    }
  }
  Dre = dr;
  Dim = di;
  grow = gk;
}

// rare path: partial-pivoting eliminations on local arrays (dynamic indexing); A row-major
template <int N>
__device__ __noinline__ double det_pivoted_real(const double *A0) {
  double A[N * N];
  for (int i = 0; i < N * N; i++) A[i] = A0[i];
  double det = 1.0;
  for (int k = 0; k < N; k++) {
    int p = k;
    double best = fabs(A[k * N + k]);
    for (int i = k + 1; i < N; i++)
      if (fabs(A[i * N + k]) > best) {
        best = fabs(A[i * N + k]);
        p = i;
      }
    if (p != k) {
      for (int j = 0; j < N; j++) {
        const double t = A[k * N + j];
        A[k * N + j] = A[p * N + j];
        A[p * N + j] = t;
      }
      det = -det;
    }
    det *= A[k * N + k];
    const double r = 1.0 / A[k * N + k];
    for (int i = k + 1; i < N; i++) {
      const double m = A[i * N + k] * r;
      for (int j = k + 1; j < N; j++) A[i * N + j] = fma(-m, A[k * N + j], A[i * N + j]);
    }
  }
  return det;
}

template <int N>
__device__ __noinline__ void det_pivoted_complex(const double *Ar0, const double *Ai0, double *out) {
  double Ar[N * N], Ai[N * N];
  for (int i = 0; i < N * N; i++) {
    Ar[i] = Ar0[i];
    Ai[i] = Ai0[i];
  }
  double dr = 1.0, di = 0.0;
  for (int k = 0; k < N; k++) {
    int p = k;
    double best = fma(Ar[k * N + k], Ar[k * N + k], Ai[k * N + k] * Ai[k * N + k]);
    for (int i = k + 1; i < N; i++) {
      const double m = fma(Ar[i * N + k], Ar[i * N + k], Ai[i * N + k] * Ai[i * N + k]);
      if (m > best) {
        best = m;
        p = i;
      }
    }
    if (p != k) {
      for (int j = 0; j < N; j++) {
        double t = Ar[k * N + j];
        Ar[k * N + j] = Ar[p * N + j];
        Ar[p * N + j] = t;
        t = Ai[k * N + j];
        Ai[k * N + j] = Ai[p * N + j];
        Ai[p * N + j] = t;
      }
      dr = -dr;
      di = -di;
    }
    const double pr = Ar[k * N + k], pi = Ai[k * N + k];
    const double t = dr * pr - di * pi;
    di = fma(dr, pi, di * pr);
    dr = t;
    const double rn = 1.0 / fma(pr, pr, pi * pi);
    const double rx = pr * rn, ry = -pi * rn;
    for (int i = k + 1; i < N; i++) {
      const double mr = Ar[i * N + k] * rx - Ai[i * N + k] * ry;
      const double mi = fma(Ar[i * N + k], ry, Ai[i * N + k] * rx);
      for (int j = k + 1; j < N; j++) {
        const double ur = Ar[k * N + j], ui = Ai[k * N + j];
        Ar[i * N + j] = fma(-mr, ur, fma(mi, ui, Ar[i * N + j]));
        Ai[i * N + j] = fma(-mr, ui, fma(-mi, ur, Ai[i * N + j]));
      }
    }
  }
  out[0] = dr;
  out[1] = di;
}

template <int F>
__device__ __forceinline__ void matmul_h(const double (&H)[F][F], const double (&A)[F][F], double (&R)[F][F]) {
#pragma unroll
  for (int i = 0; i < F; i++)
#pragma unroll
    for (int b = 0; b < F; b++) {
      double s = H[i][0] * A[0][b];
#pragma unroll
      for (int l = 1; l < F; l++) s = fma(H[i][l], A[l][b], s);
      R[i][b] = s;
    }
}

template <int F, int KIND>
__global__ void __launch_bounds__(kTptThreads) k_propagate_tpt(const __grid_constant__ TptParams TP) {
  const PropParams &P = TP.P;
  const double *c = TP.coef;
  const long long jj = (long long)blockIdx.x * kTptThreads + threadIdx.x;
  const bool valid = jj < P.nb;
  const long long jg = P.j0 + (valid ? jj : P.nb - 1);
  double Pm[F], Q[F], S = 0.0;
  double Mpp[F][F], Mpq[F][F], Mqp[F][F], Mqq[F][F], HMp[F][F], HMq[F][F], H[F][F], g[F], V;
#pragma unroll
  for (int a = 0; a < F; a++) {
    Pm[a] = P.p0q0[(long long)a * P.stride + jg] * P.isg[a];
    Q[a] = P.p0q0[(long long)(F + a) * P.stride + jg] * P.sg[a];
#pragma unroll
    for (int b = 0; b < F; b++) {
      Mpp[a][b] = Mqq[a][b] = (a == b) ? 1.0 : 0.0;
      Mpq[a][b] = Mqp[a][b] = 0.0;
    }
  }
  pes_tpt<F, KIND>(c, Q, V, g, H);
  matmul_h<F>(H, Mqp, HMp);
  matmul_h<F>(H, Mqq, HMq);
  bool good = true, dirty = false;
  int det_count = 0;
  const int nsteps = P.nsteps;
#pragma unroll 1
  for (int cstep = 0;; cstep++) {
    const bool last = (cstep == nsteps);
    const bool check = (det_count == 0) || last;
    // a6: overlap exponent and phase (Eq. 3)
    double oa = 0.0, ob = S;
#pragma unroll
    for (int a = 0; a < F; a++) {
      const double dq = P.Qeq[a] - Q[a], dp = P.Peq[a] - Pm[a];
      oa = fma(-0.25, fma(dq, dq, dp * dp), oa);
      ob = fma(0.5 * (P.Peq[a] + Pm[a]), dq, ob);
      if (P.pq_steps != nullptr && valid) P.pq_steps[((long long)cstep * F + a) * P.raw_stride + jj] = make_double2(Pm[a], Q[a]);
    }
    if (P.raw_plain) {  // several reference states: the record carries S alone
      oa = 0.0;
      ob = S;
    }
    // a5: det 2K (Eq. 5, R2)
    double Dre, Dim;
    unsigned growK;
    {
      double Ar[F][F], Ai[F][F];
#pragma unroll
      for (int i = 0; i < F; i++)
#pragma unroll
        for (int b = 0; b < F; b++) {
          Ar[i][b] = Mqq[i][b] + Mpp[i][b];
          Ai[i][b] = Mpq[i][b] - Mqp[i][b];
        }
      det_static_complex<F>(Ar, Ai, Dre, Dim, growK);
    }
    if (growK >= P.grow_k_max) {
      double br[F * F], bi[F * F], o[2];
#pragma unroll
      for (int i = 0; i < F; i++)
#pragma unroll
        for (int b = 0; b < F; b++) {
          br[i * F + b] = Mqq[i][b] + Mpp[i][b];
          bi[i * F + b] = Mpq[i][b] - Mqp[i][b];
        }
      det_pivoted_complex<F>(br, bi, o);
      Dre = o[0];
      Dim = o[1];
      if (P.fb_count != nullptr && valid) atomicAdd(P.fb_count, 1ULL);  // statistics only
    }
    if (valid && P.raw != nullptr) P.raw[(long long)cstep * P.raw_stride + jj] = make_double4(oa, ob, Dre, Dim);
    // a7: |det M - 1| <= tol and finite
    if (check) {
      double A[2 * F][2 * F];
#pragma unroll
      for (int i = 0; i < F; i++)
#pragma unroll
        for (int b = 0; b < F; b++) {
          A[i][b] = Mpp[i][b];
          A[i][F + b] = Mpq[i][b];
          A[F + i][b] = Mqp[i][b];
          A[F + i][F + b] = Mqq[i][b];
        }
      unsigned growM;
      double dM = det_static_real<2 * F>(A, growM);
      // a rejection by the fixed-order elimination is confirmed by the pivoted one before it sticks (see propagate_cml.cu)
      if (growM >= P.grow_m_max || (good && !(fabs(dM - 1.0) <= P.det_tol))) {
        double buf[4 * F * F];
#pragma unroll
        for (int i = 0; i < F; i++)
#pragma unroll
          for (int b = 0; b < F; b++) {
            buf[i * 2 * F + b] = Mpp[i][b];
            buf[i * 2 * F + F + b] = Mpq[i][b];
            buf[(F + i) * 2 * F + b] = Mqp[i][b];
            buf[(F + i) * 2 * F + F + b] = Mqq[i][b];
          }
        dM = det_pivoted_real<2 * F>(buf);
        if (P.fb_count != nullptr && valid && growK < P.grow_k_max) atomicAdd(P.fb_count, 1ULL);  // not counted twice
      }
      bool fin = isfinite(S);
#pragma unroll
      for (int a = 0; a < F; a++) fin = fin && isfinite(Pm[a]) && isfinite(Q[a]);
      good = good && fin && (fabs(dM - 1.0) <= P.det_tol);
      det_count = P.det_stride;
    }
    det_count--;
    if (last) break;
#pragma unroll 1
    for (int st = 0; st < P.nstages; st++) {
      if (dirty) {
        pes_tpt<F, KIND>(c, Q, V, g, H);
        matmul_h<F>(H, Mqp, HMp);
        matmul_h<F>(H, Mqq, HMq);
        dirty = false;
      }
      const double bdt = P.kick[st];
      S = fma(-bdt, V, S);
#pragma unroll
      for (int i = 0; i < F; i++) {
        Pm[i] = fma(-bdt, g[i], Pm[i]);
#pragma unroll
        for (int b = 0; b < F; b++) {
          Mpp[i][b] = fma(-bdt, HMp[i][b], Mpp[i][b]);
          Mpq[i][b] = fma(-bdt, HMq[i][b], Mpq[i][b]);
        }
      }
      const double adt = P.drift[st];
      if (adt != 0.0) {
#pragma unroll
        for (int i = 0; i < F; i++) {
          const double am = adt * P.mu[i];
          S = fma(0.5 * am, Pm[i] * Pm[i], S);
          Q[i] = fma(am, Pm[i], Q[i]);
#pragma unroll
          for (int b = 0; b < F; b++) {
            Mqp[i][b] = fma(am, Mpp[i][b], Mqp[i][b]);
            Mqq[i][b] = fma(am, Mpq[i][b], Mqq[i][b]);
          }
        }
        dirty = true;
      }
    }
  }
  if (!valid) return;
  if (P.good != nullptr) P.good[jj] = good ? 1 : 0;
  if (P.S_out != nullptr) P.S_out[jg] = S;
#pragma unroll
  for (int a = 0; a < F; a++) {
    if (P.pq_out != nullptr) {
      P.pq_out[(long long)a * P.stride + jg] = Pm[a] * P.sg[a];
      P.pq_out[(long long)(F + a) * P.stride + jg] = Q[a] * P.isg[a];
    }
    if (P.M_out != nullptr) {
#pragma unroll
      for (int i = 0; i < F; i++) {
        const double si = P.sg[i], ii = P.isg[i], sa = P.sg[a], ia = P.isg[a];
        const long long e = ((long long)i * F + a) * P.stride + jg;
        const long long blk = (long long)F * F * P.stride;
        P.M_out[0 * blk + e] = Mpp[i][a] * si * ia;
        P.M_out[1 * blk + e] = Mpq[i][a] * si * sa;
        P.M_out[2 * blk + e] = Mqp[i][a] * ii * ia;
        P.M_out[3 * blk + e] = Mqq[i][a] * ii * sa;
      }
    }
  }
}

// debug kernel for a1 (sc_ivr_eval_pes): same pes_tpt, caller's units out
template <int F, int KIND>
__global__ void __launch_bounds__(kTptThreads) k_eval_pes_tpt(const __grid_constant__ TptParams TP, const double *__restrict__ q,
                                                              long long n, double *Vo, double *go, double *Ho) {
  const long long j = (long long)blockIdx.x * kTptThreads + threadIdx.x;
  if (j >= n) return;
  const PropParams &P = TP.P;
  double Q[F], g[F], H[F][F], V;
#pragma unroll
  for (int a = 0; a < F; a++) Q[a] = q[(long long)a * n + j] * P.sg[a];
  pes_tpt<F, KIND>(TP.coef, Q, V, g, H);
  Vo[j] = V;
#pragma unroll
  for (int a = 0; a < F; a++) {
    go[(long long)a * n + j] = g[a] * P.sg[a];
#pragma unroll
    for (int b = 0; b < F; b++) Ho[((long long)a * F + b) * n + j] = H[a][b] * P.sg[a] * P.sg[b];
  }
}

template <int F, int KIND>
int tpt_occupancy() {
  int nb = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_propagate_tpt<F, KIND>, kTptThreads, 0) != cudaSuccess) nb = 1;
  return nb < 1 ? 1 : nb;
}

}  // namespace

int sci_tpt_traj_per_block() { return kTptThreads; }

int sci_tpt_blocks_per_sm(int F, int kind) {
  const bool qff = kind == SC_IVR_PES_QFF;
  switch (F) {
    case 1: return qff ? tpt_occupancy<1, SC_IVR_PES_QFF>() : tpt_occupancy<1, SC_IVR_PES_MORSE_UNCOUPLED>();
    case 2: return qff ? tpt_occupancy<2, SC_IVR_PES_QFF>() : tpt_occupancy<2, SC_IVR_PES_MORSE_UNCOUPLED>();
    case 3: return qff ? tpt_occupancy<3, SC_IVR_PES_QFF>() : tpt_occupancy<3, SC_IVR_PES_MORSE_UNCOUPLED>();
  }
  return 1;
}

cudaError_t sci_tpt_launch_propagate(int F, int kind, const TptParams &TP, cudaStream_t st) {
  const bool qff = kind == SC_IVR_PES_QFF;
  const unsigned blocks = (unsigned)((TP.P.nb + kTptThreads - 1) / kTptThreads);
  switch (F) {
    case 1:
      if (qff) k_propagate_tpt<1, SC_IVR_PES_QFF><<<blocks, kTptThreads, 0, st>>>(TP);
      else k_propagate_tpt<1, SC_IVR_PES_MORSE_UNCOUPLED><<<blocks, kTptThreads, 0, st>>>(TP);
      break;
    case 2:
      if (qff) k_propagate_tpt<2, SC_IVR_PES_QFF><<<blocks, kTptThreads, 0, st>>>(TP);
      else k_propagate_tpt<2, SC_IVR_PES_MORSE_UNCOUPLED><<<blocks, kTptThreads, 0, st>>>(TP);
      break;
    case 3:
      if (qff) k_propagate_tpt<3, SC_IVR_PES_QFF><<<blocks, kTptThreads, 0, st>>>(TP);
      else k_propagate_tpt<3, SC_IVR_PES_MORSE_UNCOUPLED><<<blocks, kTptThreads, 0, st>>>(TP);
      break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

cudaError_t sci_tpt_launch_eval_pes(int F, int kind, const TptParams &TP, const double *q, long long n, double *V, double *g,
                                    double *H, cudaStream_t st) {
  const bool qff = kind == SC_IVR_PES_QFF;
  const unsigned blocks = (unsigned)((n + kTptThreads - 1) / kTptThreads);
  switch (F) {
    case 1:
      if (qff) k_eval_pes_tpt<1, SC_IVR_PES_QFF><<<blocks, kTptThreads, 0, st>>>(TP, q, n, V, g, H);
      else k_eval_pes_tpt<1, SC_IVR_PES_MORSE_UNCOUPLED><<<blocks, kTptThreads, 0, st>>>(TP, q, n, V, g, H);
      break;
    case 2:
      if (qff) k_eval_pes_tpt<2, SC_IVR_PES_QFF><<<blocks, kTptThreads, 0, st>>>(TP, q, n, V, g, H);
      else k_eval_pes_tpt<2, SC_IVR_PES_MORSE_UNCOUPLED><<<blocks, kTptThreads, 0, st>>>(TP, q, n, V, g, H);
      break;
    case 3:
      if (qff) k_eval_pes_tpt<3, SC_IVR_PES_QFF><<<blocks, kTptThreads, 0, st>>>(TP, q, n, V, g, H);
      else k_eval_pes_tpt<3, SC_IVR_PES_MORSE_UNCOUPLED><<<blocks, kTptThreads, 0, st>>>(TP, q, n, V, g, H);
      break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

// Host: dense reduced constants for the thread-per-trajectory kernels (layout TC<F>).
//   Phi~_ijk = Phi_ijk / sqrt(g_i g_j g_k),  P~_ij = Phi_iijj / (g_i g_j),  w~_a^2 = w_a^2 / g_a   (QFF)
//   a~ = a / sqrt(g),  Q_e = sqrt(g) q_e                                                           (Morse)
int sci_tpt_pack_coeffs(int F, int kind, const double *c, const double *gamma, double *out) {
  if (kind != SC_IVR_PES_QFF) {
    for (int a = 0; a < F; a++) {
      const double sg = sqrt(gamma[a]);
      out[a] = c[4 * a];
      out[F + a] = c[4 * a + 1] / sg;
      out[2 * F + a] = c[4 * a + 2] * sg;
    }
    return 3 * F;
  }
  const int PP = F * F * F, W2 = PP + F * F;
  const double *cub = c + F;
  int m = 0;
  for (int i = 0; i < F; i++)
    for (int j = i; j < F; j++)
      for (int k = j; k < F; k++) {
        const double v = cub[m++] / sqrt(gamma[i] * gamma[j] * gamma[k]);
        const int p[6][3] = {{i, j, k}, {i, k, j}, {j, i, k}, {j, k, i}, {k, i, j}, {k, j, i}};
        for (auto &t : p) out[(t[0] * F + t[1]) * F + t[2]] = v;
      }
  const double *qua = cub + m;
  m = 0;
  for (int i = 0; i < F; i++)
    for (int j = i; j < F; j++) {
      const double v = qua[m++] / (gamma[i] * gamma[j]);
      out[PP + i * F + j] = out[PP + j * F + i] = v;
    }
  for (int a = 0; a < F; a++) out[W2 + a] = c[a] * c[a] / gamma[a];
  return W2 + F;
}
