// Kernel A, "C modes per lane" mapping with the monodromy state in tensor memory (rows a1-a7 of DESIGN.md).
//
// Mapping.  L lanes per trajectory, G = floor(32 / L) trajectories per warp, lane = l * G + g (l = lane class,
// g = trajectory of the warp).  Lane l owns the modes a = l + s L, s = 0 .. C-1 (C = ceil(F / L)): their (P_a, Q_a), its
// share of the action, and the 2 C tangent vectors d(P,Q)/dP0_a (slot s) and d(P,Q)/dQ0_a (slot C + s), i.e. 2 C
// columns of the 2F x 2F monodromy matrix M.  The columns of M evolve independently given the
// Hessian, so nothing but the Hessian and the pivot columns of the two eliminations crosses lanes.
//
// Where the state lives (per SM: one CTA of 8 warps):
//   tensor memory   the lane's 2 C columns of M (4 C F doubles), exactly the matrix M(c) of the last integer time c:
//                   TMEM is used as lane-private scratch through tcgen05.ld / tcgen05.st (32x32b), two warps per
//                   32-lane quadrant, 128 doubles per lane each; layout [dP rows | dQ rows][column][F]
//   registers       the working copies of the two eliminations (a5: det 2K, complex F x F; a7: det M, real 2F x 2F, in two
//                   row halves) and of the pass
//   shared memory   per trajectory: Q exchange, Hessian entries, cubic gradient terms of the PES; per lane: H dQ of the
//                   last evaluation point (used twice: closing kick before the snapshot, opening kick after it)
//   warp shuffles   the pivot columns of the eliminations (owner lane -> the L lanes of the trajectory): no shared memory,
//                   no barrier in the snapshot
//
// Per time step (velocity-Verlet; the general "kick b_s, drift a_s" composition is a table of evaluation points):
//   snapshot  M-LU and K-LU from the TMEM state (static pivot order with look-ahead, monitored multipliers, pivoted
//             fallback, which also confirms every rejection), record (ln|<chi|pq>|, S + arg<chi|pq>, det 2K), flag
//             |det M - 1| <= tol
//   pass      scalars kick/drift; PES at the new Q (gradient, Hessian -> shared memory); per column: opening kick with
//             the parked H dQ, drift, new H dQ, closing kick, store to TMEM, park H dQ
//
// Everything runs in reduced coordinates Q = sqrt(gamma) q, P = p / sqrt(gamma): 2K = (M_qq + M_pp) + i (M_pq - M_qp).
//
// This file is compiled once per row (F, L) of cml_table.h (-DSCI_CML_INST_F, -DSCI_CML_INST_L: the kernels) and once without
// them (the dispatcher at the end).  Measurements, the instruction mix and the variants that were tried and dropped:
// profiles/r02_kernelA_ncu_config4.md; design: DESIGN.md section 3.
#include "common.cuh"
#include "tmem_ldst.cuh"

#include "cml_table.h"

#ifndef SCI_CML_WARPS
#define SCI_CML_WARPS 8
#endif
constexpr int kWarpsC = SCI_CML_WARPS;
constexpr int kThreadsC = kWarpsC * 32;

#ifdef SCI_CML_INST_F
// ======== one (F, L) instantiation per translation unit (build.py compiles this file once per row of cml_table.h) ========
namespace {


__device__ __forceinline__ double rcp_nr2(double x) {
  // MUFU.RCP64H seed (2^-23 relative) + two Newton steps: ~1 ulp for normal x, no slow path.  One step (2^-46) is not
  // enough: det M of a strongly stretched trajectory is a difference of large terms, and multipliers that are off by
  // 1e-14 move |det M - 1| across the 1e-6 threshold where the oracle's exact multipliers do not (152 of 131072
  // trajectories of config 4 change their flag).
#ifndef SCI_CML_RCP_NR
#define SCI_CML_RCP_NR 3
#endif
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
#if SCI_CML_RCP_NR == 3
  // cubic step: r (1 + e + e^2), e = 1 - x r = 2^-23  ->  2^-69 before rounding, three dependent FMAs instead of four
  const double e = fma(-x, r, 1.0);
  const double t = fma(e, e, e);
  r = fma(r, t, r);
#else
#pragma unroll
  for (int it = 0; it < SCI_CML_RCP_NR; it++) {
    const double e = fma(-x, r, 1.0);
    r = fma(r, e, r);
  }
#endif
  return r;
}

__device__ __forceinline__ unsigned abs_hi(double x) { return (unsigned)__double2hiint(x) & 0x7fffffffu; }

// shared memory through 32-bit addresses (one base register, the offsets are immediates)
__device__ __forceinline__ double lds(uint32_t a) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ void sts(uint32_t a, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory"); }
__device__ __forceinline__ void lds2(uint32_t a, double &x, double &y) {
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(x), "=d"(y) : "r"(a) : "memory");
}
__device__ __forceinline__ void sts2(uint32_t a, double x, double y) {
  asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(x), "d"(y) : "memory");
}
// value of v on lane src (every lane of the warp executes this).  One 64-bit broadcast costs two SHFL = one cycle of
// the SM's shared-memory data pipe, against 2 (LDS.64) + 1.3 (owner's STS.64) + a warp barrier through shared memory
// (ncu: l1tex__data_pipe_lsu_wavefronts_mem_shared, profiles/r02b)
template <int L>
__device__ __forceinline__ double bcast(double v, int src) {
  if (L == 1) return v;  // one lane per trajectory: the owner is the lane itself
  return __shfl_sync(0xffffffffu, v, src);
}

// Optional barriers that keep the warps of a CTA in step (SCI_CML_SYNC = 1: one CTA barrier per time step; 6: the warps 4..
// run half a time step behind the warps 0..3; 7: both).  Measured on config 4 (profiles/r02): none of them pays once the
// launch is balanced (219 cycles per trajectory-step per SM without, 232 / 222 / 240 with), so the default is 0.
#ifndef SCI_CML_SYNC
#define SCI_CML_SYNC 0
#endif
__device__ __forceinline__ void cta_sync(int nthreads) { asm volatile("bar.sync 0, %0;" ::"r"(nthreads) : "memory"); }

template <int F, int L>
struct Cml {
  static constexpr int C = (F + L - 1) / L;   // modes per lane
  static constexpr int G = 32 / L;            // trajectories per warp
  static constexpr int ACT = G * L;           // lanes that own a trajectory share; the rest clone lane 0 (same numbers, same
                                              // shared-memory stores) and write nothing to global memory
  static constexpr int N = 2 * F;             // rows of M: dP_0..dP_{F-1}, dQ_0..dQ_{F-1}
  static constexpr int NS = 2 * C;            // columns (slots) of M per lane
  static constexpr int ND = F / 2 + 1;        // Hessian entries (a, (a+d)%F), d = 0..ND-1, computed by the owner of mode a
  static constexpr int NR = (F - 1) / 2;      // cubic-gradient terms received from the owners of modes a-d
  static constexpr int NH = ND * F;
  // tensor memory, per lane, in doubles: [row half: dP rows, dQ rows][slot][F]
  static constexpr int TH = NS * F;           // doubles per row half
  static constexpr int TCOLS = 2 * TH * 2;    // 32-bit TMEM columns per lane
  static_assert(TCOLS <= 256, "state does not fit the half quadrant of tensor memory a warp owns");
  static constexpr bool EXACT = (F % L) == 0; // no phantom modes
  // packed coefficients.  QFF: per lane class l and slot s a list of LAP doubles, pair t of the list of (l, s) at
  // double2 index (s * LAP/2 + t) * L + l.  Positions within a list:
  static constexpr int L_C3 = 0;               // [ND][F]  (d, k) -> Phi~[a][(a+d)%F][k]
  static constexpr int L_C4U = L_C3 + ND * F;  // [F]      j      -> P~[a][j]
  static constexpr int L_C4D = L_C4U + F;      // [ND]     d      -> P~[a][(a+d)%F]
  static constexpr int L_W2 = L_C4D + ND;      //                    omega_a^2 / gamma_a
  static constexpr int LA = L_W2 + 1;
  static constexpr int LAP = (LA + 1) & ~1;
  static constexpr int NCOEF_QFF = C * LAP * L;
  static constexpr int NCOEF_MORSE = 3 * C * L;  // (D, a~, Qe) of slot s, lane class l at ((s * 3 + j) * L + l)
  static constexpr int NCOEF = NCOEF_QFF > NCOEF_MORSE ? NCOEF_QFF : NCOEF_MORSE;
  static constexpr int NCOEFP = (NCOEF + 1) & ~1;
  // per-warp shared memory, in doubles.  Group arrays are [element][G] (the L lanes of trajectory g read the same word,
  // the G trajectories adjacent words); the parked H dQ is lane-private, in pairs: element e of the lane at byte
  // 512 (e / 2) + 16 lane + 8 (e % 2).
  __host__ __device__ static constexpr int ev(int x) { return (x + 1) & ~1; }
  static constexpr int O_QS = 0;                      // [F]
  static constexpr int O_HS = O_QS + F;               // [NH]
  static constexpr int O_G3 = O_HS + NH;              // [NR][F]
  static constexpr int O_RED = O_G3 + NR * F;         // [L][2]
  static constexpr int O_DUMP = O_RED + 2 * L;        // [1]: stores of phantom modes (F % L != 0)
  static constexpr int WSG = ev((O_DUMP + 1) * G);    // doubles of group arrays per warp
  static constexpr int HMH = ev(C * F);               // parked H dQ: elements per half
  static constexpr int WS = WSG + 2 * HMH * 32;
  static constexpr size_t SMEM = sizeof(double) * (NCOEFP + (size_t)kWarpsC * WS) + 16;
  // Dynamic shared memory the propagation kernel is LAUNCHED with.  Every CTA takes all 512 columns of the SM's tensor memory,
  // so a second CTA on the same SM would sit in tcgen05.alloc, holding its slot, until the first one ends, and the launch
  // shape ("whole rounds of one CTA per SM") would no longer describe what runs.  __launch_bounds__(.., 1) does not cap
  // residency; shared memory does: two CTAs of more than (228 KB - 2 x 1 KB reserved) / 2 = 113 KB cannot share an SM.  The
  // small-F rows (F = 4: 113 KB would fit twice) are padded up to that.
  static constexpr size_t SMEM_ONE_CTA = 115 * 1024;
  static constexpr size_t SMEM_LAUNCH = SMEM > SMEM_ONE_CTA ? SMEM : SMEM_ONE_CTA;
  __host__ __device__ static constexpr int hm(int e) { return 512 * (e / 2) + 8 * (e % 2); }

  // column (l, s) of M: mode a = l + (s % C) L, half h = s / C (0: d/dP0_a, 1: d/dQ0_a), global index h F + a.
  // Elimination step k uses the diagonal pivot of the column with global index k.
  __host__ __device__ static constexpr int step_lane(int k) { return (k % F) % L; }
  __host__ __device__ static constexpr int step_slot(int k) { return (k % F) / L + (k / F) * C; }
  // is slot s (d/dP0 columns: s < C) still live on SOME lane class after the first k + 1 pivots?
  __host__ __device__ static constexpr bool slot_live(int s, int k) {
    return s >= C || ((s * L + L - 1 < F - 1 ? s * L + L - 1 : F - 1) > k);
  }
};

// store in chunks of at most WMAX 32-bit columns: a tcgen05.st needs its source in consecutive registers, and gathering
// 54 of them costs a register move each; short chunks take the values where they are
#ifndef SCI_CML_ST_W
#define SCI_CML_ST_W 128
#endif
template <int ND, int WMAX, bool WAIT = true>
__device__ __forceinline__ void tmem_st_f64_w(uint32_t taddr, const double (&d)[ND]) {
  uint32_t v[2 * ND];
#pragma unroll
  for (int i = 0; i < ND; i++) {
    v[2 * i] = (uint32_t)__double2loint(d[i]);
    v[2 * i + 1] = (uint32_t)__double2hiint(d[i]);
  }
  tmem_st_issue<2 * ND, 0, WMAX>(taddr, v);
  if (WAIT) asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

// one column of M from / to the lane's tensor memory: rows 0..F-1 (dP) and F..2F-1 (dQ) live in different halves
template <int F, int L>
__device__ __forceinline__ void tmem_ld_col(uint32_t tm, int s, double (&col)[2 * F]) {
  double a[F], b[F];
  tmem_ld_f64<F>(tm + s * F * 2, a);
  tmem_ld_f64<F>(tm + (Cml<F, L>::TH + s * F) * 2, b);
#pragma unroll
  for (int i = 0; i < F; i++) {
    col[i] = a[i];
    col[F + i] = b[i];
  }
}
template <int F, int L>
__device__ __forceinline__ void tmem_st_col(uint32_t tm, int s, const double (&col)[2 * F]) {
  double a[F], b[F];
#pragma unroll
  for (int i = 0; i < F; i++) {
    a[i] = col[i];
    b[i] = col[F + i];
  }
  tmem_st_f64<F>(tm + s * F * 2, a);
  tmem_st_f64<F>(tm + (Cml<F, L>::TH + s * F) * 2, b);
}

// shared-memory addresses of one lane
struct LaneAddr {
  uint32_t g;   // element 0 of the trajectory's group arrays: element e at g + 8 G e
  uint32_t hm;  // the lane's parked H dQ
  int g0;       // lane of class 0 of this trajectory: class c sits on lane g0 + c G
};

// ---- a1: potential share, gradient components and Hessian entries of the lane's modes (reduced coordinates) ----------
// QFF (BASELINE.json configs 2-5, stand-in for the fitted surfaces of PAPER.md:157):
//   H3_ab = sum_k Phi_abk Q_k,  g3_a = 1/2 sum_b H3_ab Q_b,  u_a = sum_j P_aj Q_j^2,
//   g4_a = Q_a (u_a/2 - P_aa Q_a^2/3),  H4_aa = u_a/2,  H4_ab = P_ab Q_a Q_b,
//   V = sum_a Q_a (w_a^2 Q_a/2 + g3_a/3 + g4_a/4)   (Euler's theorem on the homogeneous parts).
// Morse: y = exp(-a (Q - Q_e)), V = D (1-y)^2, g = 2 D a y (1-y), H = 2 D a^2 y (2y-1).
// The owner of mode a computes the entries (a, (a+d)%F), d < ND, and stores them at HS[d F + a]; the cubic gradient
// terms that belong to the modes a+d travel through G3.  Two warp barriers inside; the caller needs one more before
// it reads HS.  Stores of phantom modes (F % L != 0) go to the dump word.
template <int F, int L, int KIND>
__device__ __forceinline__ void pes_cml(const double *__restrict__ cs, const LaneAddr &A, int l, const double (&Q)[Cml<F, L>::C],
                                        double (&gq)[Cml<F, L>::C], double &Va) {
  using X = Cml<F, L>;
  constexpr int C = X::C, G = X::G;
  const uint32_t gsa = A.g;
  const uint32_t dump = gsa + 8 * X::O_DUMP * G;
  Va = 0.0;
  if (KIND == SC_IVR_PES_QFF) {
#pragma unroll
    for (int s = 0; s < C; s++) {
      const int a = l + s * L;
      sts((X::EXACT || a < F) ? gsa + 8 * (X::O_QS + a) * G : dump, Q[s]);
    }
    __syncwarp();
    double q[F], q2[F];
#pragma unroll
    for (int i = 0; i < F; i++) {
      q[i] = lds(gsa + 8 * (X::O_QS + i) * G);
      q2[i] = q[i] * q[i];
    }
    double s3[C], u[C], w2[C], paa[C];
    const double2 *c2 = reinterpret_cast<const double2 *>(cs);
#pragma unroll
    for (int s = 0; s < C; s++) {
      const int a = l + s * L;
      const bool real = X::EXACT || a < F;
      const int ae = real ? a : 0;
      double cf[X::LAP];
#pragma unroll
      for (int t = 0; t < X::LAP / 2; t++) {
        const double2 v = c2[(s * (X::LAP / 2) + t) * L + l];
        cf[2 * t] = v.x;
        cf[2 * t + 1] = v.y;
      }
      double qd[X::ND];
      qd[0] = Q[s];
#pragma unroll
      for (int d = 1; d < X::ND; d++) {
        int b = ae + d;
        b = b >= F ? b - F : b;
        qd[d] = lds(gsa + 8 * (X::O_QS + b) * G);
      }
      double uu = 0.0;
#pragma unroll
      for (int j = 0; j < F; j++) uu = fma(cf[X::L_C4U + j], q2[j], uu);
      double h3[X::ND];
#pragma unroll
      for (int d = 0; d < X::ND; d++) {
        double t = 0.0;
#pragma unroll
        for (int k = 0; k < F; k++) t = fma(cf[X::L_C3 + d * F + k], q[k], t);
        h3[d] = t;
      }
      double t3 = 0.0;
#pragma unroll
      for (int d = 0; d < X::ND; d++) t3 = fma(h3[d], qd[d], t3);
      s3[s] = t3;
      u[s] = uu;
      w2[s] = cf[X::L_W2];
      paa[s] = cf[X::L_C4D];
      sts(real ? gsa + 8 * (X::O_HS + ae) * G : dump, w2[s] + h3[0] + 0.5 * uu);
#pragma unroll
      for (int d = 1; d < X::ND; d++) {
        int b = ae + d;
        b = b >= F ? b - F : b;
        sts(real ? gsa + 8 * (X::O_HS + d * F + ae) * G : dump, fma(cf[X::L_C4D + d] * Q[s], qd[d], h3[d]));
        if (d <= X::NR) sts(real ? gsa + 8 * (X::O_G3 + (d - 1) * F + b) * G : dump, h3[d] * Q[s]);
      }
    }
    __syncwarp();
#pragma unroll
    for (int s = 0; s < C; s++) {
      const int a = l + s * L;
      const bool real = X::EXACT || a < F;
      const int ae = real ? a : 0;
      double t3 = s3[s];
#pragma unroll
      for (int d = 1; d <= X::NR; d++) t3 += lds(gsa + 8 * (X::O_G3 + (d - 1) * F + ae) * G);
      const double g3 = 0.5 * t3;
      const double g4 = Q[s] * (0.5 * u[s] - (1.0 / 3.0) * paa[s] * Q[s] * Q[s]);
      const double gg = fma(w2[s], Q[s], g3 + g4);
      const double vv = Q[s] * (0.5 * w2[s] * Q[s] + (1.0 / 3.0) * g3 + 0.25 * g4);
      gq[s] = real ? gg : 0.0;
      Va += real ? vv : 0.0;
    }
  } else {
#pragma unroll
    for (int s = 0; s < C; s++) {
      const int a = l + s * L;
      const bool real = X::EXACT || a < F;
      const double D = cs[(s * 3 + 0) * L + l], at = cs[(s * 3 + 1) * L + l], Qe = cs[(s * 3 + 2) * L + l];
      const double y = exp(-at * (Q[s] - Qe));
      const double vv = D * (1.0 - y) * (1.0 - y);
      gq[s] = real ? 2.0 * D * at * y * (1.0 - y) : 0.0;
      Va += real ? vv : 0.0;
      sts(real ? gsa + 8 * (X::O_HS + a) * G : dump, 2.0 * D * at * at * y * (2.0 * y - 1.0));
    }
  }
}

// ---- a3 helper: HM = H dQ for NB columns at once, H from the trajectory's shared slot (entries (i, (i+d)%F) at HS[d F + i])
template <int F, int L, int KIND, int NB>
__device__ __forceinline__ void hessian_times(uint32_t gsa, const double (&dQ)[NB][F], double (&HM)[NB][F]) {
  using X = Cml<F, L>;
  constexpr int G = X::G;
#pragma unroll
  for (int i = 0; i < F; i++) {
    const double h = lds(gsa + 8 * (X::O_HS + i) * G);
#pragma unroll
    for (int c = 0; c < NB; c++) HM[c][i] = h * dQ[c][i];
  }
  if (KIND == SC_IVR_PES_QFF) {
#pragma unroll
    for (int d = 1; d < X::ND; d++) {
#pragma unroll
      for (int i = 0; i < F; i++) {
        if (F % 2 == 0 && d == F / 2 && i >= F / 2) continue;  // pair (i, i+F/2) is also stored by the owner of i+F/2
        const int j = (i + d) % F;
        const double h = lds(gsa + 8 * (X::O_HS + d * F + i) * G);
#pragma unroll
        for (int c = 0; c < NB; c++) {
          HM[c][i] = fma(h, dQ[c][j], HM[c][i]);
          HM[c][j] = fma(h, dQ[c][i], HM[c][j]);
        }
      }
    }
  }
}

// ---- one pass over the lane's columns at a new evaluation point (a2, a3) ----------------------------------------------
//   dP -= post * HMprev (opening kick of the point just left, H dQ parked there);  dQ += adt mu dP (drift);
//   HM = H(Q_new) dQ;  dP -= pre * HM (kick at the new point up to the snapshot);  state -> TMEM;  HM parked.
// Columns are handled C at a time (the slots of one half h).
template <int F, int L, int KIND>
__device__ __forceinline__ void pass_cml(uint32_t tm, const LaneAddr &A, const PropParams &P, double post, double adt, double pre) {
  using X = Cml<F, L>;
  constexpr int C = X::C;
  // a real loop: the second half runs from the instruction-cache lines the first one fetched
#pragma unroll 1
  for (int h = 0; h < 2; h++) {
    const uint32_t tmh = tm + h * C * F * 2;
    const uint32_t hmh = A.hm + h * (X::HMH * 256);
    double sp[C * F], sq[C * F];
    tmem_ld_f64<C * F>(tmh, sp);
    tmem_ld_f64<C * F>(tmh + X::TH * 2, sq);
    double hp[X::HMH];
#pragma unroll
    for (int e = 0; e < C * F; e += 2) lds2(hmh + X::hm(e), hp[e], hp[e + 1]);
    double dP[C][F], dQ[C][F], HM[C][F];
#pragma unroll
    for (int c = 0; c < C; c++)
#pragma unroll
      for (int i = 0; i < F; i++) {
        dP[c][i] = fma(-post, hp[c * F + i], sp[c * F + i]);
        dQ[c][i] = fma(adt * P.mu[i], dP[c][i], sq[c * F + i]);
      }
    hessian_times<F, L, KIND, C>(A.g, dQ, HM);
#pragma unroll
    for (int c = 0; c < C; c++)
#pragma unroll
      for (int i = 0; i < F; i++) {
        sp[c * F + i] = fma(-pre, HM[c][i], dP[c][i]);
        sq[c * F + i] = dQ[c][i];
      }
#pragma unroll
    for (int e = 0; e < C * F; e += 2)
      sts2(hmh + X::hm(e), HM[e / F][e % F], (e + 1 < C * F) ? HM[(e + 1) / F][(e + 1) % F] : 0.0);
    tmem_st_f64_w<C * F, SCI_CML_ST_W, false>(tmh + X::TH * 2, sq);
    tmem_st_f64_w<C * F, SCI_CML_ST_W>(tmh, sp);
  }
}

// ---- a5: the F-1 steps of the complex elimination of 2K, one at a time (called from both snapshot variants) -------------
// (rr, ri): reciprocal pivot of step j; (pr, pi)[i], i > j: the pivot column.  sn: slot that holds the next pivot (-1:
// none); on return (nr, ni)[i], i >= j + 1 hold the next pivot column as broadcast by its owner, row j + 1 the pivot.
template <int F, int L>
struct KStep {
  using X = Cml<F, L>;
  static constexpr int C = X::C, G = X::G;
  // update slot s with step j
  static __device__ __forceinline__ void upd(int j, int s, int l, double (&Kr)[C][F], double (&Ki)[C][F], double rr, double ri,
                                             const double (&pr)[F], const double (&pi)[F], unsigned &gk) {
    const bool live = s * L + l > j && (X::EXACT || s * L + l < F);
    const double mr = Kr[s][j] * rr - Ki[s][j] * ri;
    const double mi = fma(Kr[s][j], ri, Ki[s][j] * rr);
    if (live) gk = max(gk, max(abs_hi(mr), abs_hi(mi)));
#pragma unroll
    for (int i = j + 1; i < F; i++) {
      Kr[s][i] = fma(-mr, pr[i], fma(mi, pi[i], Kr[s][i]));
      Ki[s][i] = fma(-mr, pi[i], fma(-mi, pr[i], Ki[s][i]));
    }
  }
  // broadcast column `s` (rows j..F-1) from lane class c; row j is replaced by the reciprocal of the pivot
  static __device__ __forceinline__ void cast(int j, int s, int src, const double (&Kr)[C][F], const double (&Ki)[C][F], double &rr,
                                              double &ri, double (&pr)[F], double (&pi)[F]) {
#pragma unroll
    for (int i = j; i < F; i++) {
      pr[i] = bcast<L>(Kr[s][i], src);
      pi[i] = bcast<L>(Ki[s][i], src);
    }
    const double rn = rcp_nr2(fma(pr[j], pr[j], pi[j] * pi[j]));
    rr = pr[j] * rn;
    ri = -pi[j] * rn;
  }
};

// ---- a7 + a5: det M by LU in a STATIC pivot order with look-ahead, in two ROW halves; det 2K alongside --------------------
// The lane holds NS = 2C columns of M (slot s < C: d/dP0 of its mode s, slot C + s: d/dQ0).  Step k eliminates row k with
// the diagonal pivot of the column with global index k: every lane receives that column from its owner by warp shuffles
// (no shared memory, no barrier), scales its row-k elements by the reciprocal pivot (multiplier m[s][k]) and updates its
// live columns.  The column that holds the NEXT pivot is updated first and broadcast before the rest of the step's
// updates, so that the shuffle -> reciprocal chain of step k+1 runs under the bulk of step k's arithmetic.
// Row halves (the registers hold 2C x F doubles of M at a time): phase T runs the steps 0..F-1 on the rows 0..F-1 (dP) of all
// columns and keeps the multipliers; phase B replays them on the rows F..2F-1 (dQ), the pivot columns' lower parts being
// broadcast as they become final; what is left in the d/dQ0 columns is the Schur complement, whose F-1 steps run TOGETHER
// with the F-1 steps of the complex elimination of 2K (two independent pivot chains).  Element by element the arithmetic
// is that of the one-piece right-looking elimination.  No pivot search: numerical safety is monitored instead (gm, gk =
// largest |multiplier| of a live column, IEEE high word); the caller repeats a step whose multipliers exceed its bound
// with the pivoted routine.
// Results on lane class step_lane(N-1): det M, and (Dre, Dim) = det(2K) |R|^2 with R the product of the reciprocal
// pivots: a positive multiple of det 2K; only its phase is used downstream (Eq. 10 drops |C_t|).
template <int F, int L>
__device__ __forceinline__ void lu_mk_cml(uint32_t tm, const LaneAddr &A, int l, double &detM, unsigned &gm_out, double &Dre,
                                          double &Dim, unsigned &gk_out) {
  using X = Cml<F, L>;
  constexpr int G = X::G, C = X::C, NS = X::NS;
  double Rm = 1.0;
  unsigned gm = 0u;
  double m[NS][F];  // m[s][k]: multiplier of column s in step k (entries of dead columns are never used)
  // ---- phase T: rows 0..F-1 ----
  {
    double W[NS][F];
    {
      double st[NS * F];
      tmem_ld_f64<NS * F>(tm, st);
#pragma unroll
      for (int s = 0; s < NS; s++)
#pragma unroll
        for (int i = 0; i < F; i++) W[s][i] = st[s * F + i];
    }
    double pc[F];
#pragma unroll
    for (int i = 0; i < F; i++) pc[i] = bcast<L>(W[0][i], A.g0);
    double r = rcp_nr2(pc[0]);
#pragma unroll
    for (int k = 0; k < F; k++) {
      Rm *= r;
      const int sn = (k + 1 < F) ? (k + 1) / L : -1;
      double pn[F], rn = 0.0;
      if (sn >= 0) {
        m[sn][k] = W[sn][k] * r;
        if (sn * L + l > k && (X::EXACT || sn * L + l < F)) gm = max(gm, abs_hi(m[sn][k]));
#pragma unroll
        for (int i = k + 1; i < F; i++) W[sn][i] = fma(-m[sn][k], pc[i], W[sn][i]);
#pragma unroll
        for (int i = k + 1; i < F; i++) pn[i] = bcast<L>(W[sn][i], A.g0 + ((k + 1) % L) * G);
        rn = rcp_nr2(pn[k + 1]);
      }
#pragma unroll
      for (int s = 0; s < NS; s++) {
        if (s == sn || !X::slot_live(s, k)) continue;
        m[s][k] = W[s][k] * r;
        const bool live = s >= C ? (X::EXACT || (s - C) * L + l < F) : (s * L + l > k && (X::EXACT || s * L + l < F));
        if (live) gm = max(gm, abs_hi(m[s][k]));
#pragma unroll
        for (int i = k + 1; i < F; i++) W[s][i] = fma(-m[s][k], pc[i], W[s][i]);
      }
      if (sn >= 0) {
        r = rn;
#pragma unroll
        for (int i = k + 2; i < F; i++) pc[i] = pn[i];
      }
    }
  }
  // ---- phase B: rows F..2F-1 (W[s][i] is row F + i) ----
  double W[NS][F];
  {
    double st[NS * F];
    tmem_ld_f64<NS * F>(tm + X::TH * 2, st);
#pragma unroll
    for (int s = 0; s < NS; s++)
#pragma unroll
      for (int i = 0; i < F; i++) W[s][i] = st[s * F + i];
  }
  {
    double pc[F];
#pragma unroll
    for (int i = 0; i < F; i++) pc[i] = bcast<L>(W[0][i], A.g0);
#pragma unroll
    for (int k = 0; k < F; k++) {
      const int sn = (k + 1 < F) ? (k + 1) / L : -1;
      double pn[F];
      if (sn >= 0) {
#pragma unroll
        for (int i = 0; i < F; i++) W[sn][i] = fma(-m[sn][k], pc[i], W[sn][i]);
#pragma unroll
        for (int i = 0; i < F; i++) pn[i] = bcast<L>(W[sn][i], A.g0 + ((k + 1) % L) * G);
      }
#pragma unroll
      for (int s = 0; s < NS; s++) {
        if (s == sn || !X::slot_live(s, k)) continue;
#pragma unroll
        for (int i = 0; i < F; i++) W[s][i] = fma(-m[s][k], pc[i], W[s][i]);
      }
      if (sn >= 0) {
#pragma unroll
        for (int i = 0; i < F; i++) pc[i] = pn[i];
      }
    }
  }
  // ---- the Schur complement S[s][i] = W[C + s][i] (F x F, column index s L + l) and 2K ----
  // the lane's columns of 2K = (M_qq + M_pp) + i (M_pq - M_qp) (Eq. 5, reading R2, reduced coordinates)
  double Kr[C][F], Ki[C][F];
#pragma unroll
  for (int s = 0; s < C; s++) {
    double c1p[F], c1q[F], c2p[F], c2q[F];  // columns d/dP0_a and d/dQ0_a of the lane's mode s, dP rows and dQ rows
    tmem_ld_f64<F>(tm + s * F * 2, c1p);
    tmem_ld_f64<F>(tm + (X::TH + s * F) * 2, c1q);
    tmem_ld_f64<F>(tm + (C + s) * F * 2, c2p);
    tmem_ld_f64<F>(tm + (X::TH + (C + s) * F) * 2, c2q);
#pragma unroll
    for (int i = 0; i < F; i++) {
      Kr[s][i] = c2q[i] + c1p[i];  // dQ2 + dP1
      Ki[s][i] = c2p[i] - c1q[i];  // dP2 - dQ1
    }
  }
  double Rr = 1.0, Ri = 0.0;
  unsigned gk = 0u;
  double pc[F], r = 1.0;
  double rr = 1.0, ri = 0.0, pr[F], pi[F];
  if (F > 1) {
#pragma unroll
    for (int i = 0; i < F; i++) pc[i] = bcast<L>(W[C][i], A.g0);
    r = rcp_nr2(pc[0]);
    KStep<F, L>::cast(0, 0, A.g0, Kr, Ki, rr, ri, pr, pi);
  }
#pragma unroll
  for (int j = 0; j < F - 1; j++) {
    Rm *= r;
    {
      const double t = Rr * rr - Ri * ri;
      Ri = fma(Rr, ri, Ri * rr);
      Rr = t;
    }
    const int sn = (j + 1 < F - 1) ? (j + 1) / L : -1;  // the slot of the next pivot, in both eliminations
    double pn[F], rn = 0.0, rrn = 0.0, rin = 0.0, prn[F], pin[F];
    if (sn >= 0) {
      const bool live = sn * L + l > j && (X::EXACT || sn * L + l < F);
      const int src = A.g0 + ((j + 1) % L) * G;
      {
        const double mm = W[C + sn][j] * r;
        if (live) gm = max(gm, abs_hi(mm));
#pragma unroll
        for (int i = j + 1; i < F; i++) W[C + sn][i] = fma(-mm, pc[i], W[C + sn][i]);
#pragma unroll
        for (int i = j + 1; i < F; i++) pn[i] = bcast<L>(W[C + sn][i], src);
        rn = rcp_nr2(pn[j + 1]);
      }
      KStep<F, L>::upd(j, sn, l, Kr, Ki, rr, ri, pr, pi, gk);
      KStep<F, L>::cast(j + 1, sn, src, Kr, Ki, rrn, rin, prn, pin);
    }
#pragma unroll
    for (int s = 0; s < C; s++) {
      if (s == sn || !X::slot_live(s, j)) continue;
      const bool live = s * L + l > j && (X::EXACT || s * L + l < F);
      const double mm = W[C + s][j] * r;
      if (live) gm = max(gm, abs_hi(mm));
#pragma unroll
      for (int i = j + 1; i < F; i++) W[C + s][i] = fma(-mm, pc[i], W[C + s][i]);
      KStep<F, L>::upd(j, s, l, Kr, Ki, rr, ri, pr, pi, gk);
    }
    if (sn >= 0) {
      r = rn;
      rr = rrn;
      ri = rin;
#pragma unroll
      for (int i = j + 2; i < F; i++) {
        pc[i] = pn[i];
        pr[i] = prn[i];
        pi[i] = pin[i];
      }
    }
  }
  detM = W[C + (F - 1) / L][F - 1] * rcp_nr2(Rm);
  // det 2K = p_{F-1} / R  ~  p_{F-1} conj(R)
  const double lr = Kr[(F - 1) / L][F - 1], li = Ki[(F - 1) / L][F - 1];
  Dre = fma(lr, Rr, li * Ri);
  Dim = fma(li, Rr, -lr * Ri);
  gk_out = gk;
  gm_out = gm;
}

// ---- a5 alone (time steps without the a7 check): det 2K by the same scheme; the lane's columns s = 0..C-1 are those of
// its modes.  Result on lane class step_lane(F-1).
template <int F, int L>
__device__ __forceinline__ void lu_k_cml(double (&Kr)[Cml<F, L>::C][F], double (&Ki)[Cml<F, L>::C][F], const LaneAddr &A, int l,
                                         double &Dre, double &Dim, unsigned &gk_out) {
  using X = Cml<F, L>;
  constexpr int G = X::G, C = X::C;
  double Rr = 1.0, Ri = 0.0;
  unsigned gk = 0u;
  double rr = 1.0, ri = 0.0, pr[F], pi[F];
  if (F > 1) KStep<F, L>::cast(0, 0, A.g0, Kr, Ki, rr, ri, pr, pi);
#pragma unroll
  for (int j = 0; j < F - 1; j++) {
    {
      const double t = Rr * rr - Ri * ri;
      Ri = fma(Rr, ri, Ri * rr);
      Rr = t;
    }
    const int sn = (j + 1 < F - 1) ? (j + 1) / L : -1;
    double rrn = 0.0, rin = 0.0, prn[F], pin[F];
    if (sn >= 0) {
      KStep<F, L>::upd(j, sn, l, Kr, Ki, rr, ri, pr, pi, gk);
      KStep<F, L>::cast(j + 1, sn, A.g0 + ((j + 1) % L) * G, Kr, Ki, rrn, rin, prn, pin);
    }
#pragma unroll
    for (int s = 0; s < C; s++) {
      if (s == sn || !X::slot_live(s, j)) continue;
      KStep<F, L>::upd(j, s, l, Kr, Ki, rr, ri, pr, pi, gk);
    }
    if (sn >= 0) {
      rr = rrn;
      ri = rin;
#pragma unroll
      for (int i = j + 2; i < F; i++) {
        pr[i] = prn[i];
        pi[i] = pin[i];
      }
    }
  }
  // det 2K = p_{F-1} / R  ~  p_{F-1} conj(R)
  const double lr = Kr[(F - 1) / L][F - 1], li = Ki[(F - 1) / L][F - 1];
  Dre = fma(lr, Rr, li * Ri);
  Dim = fma(li, Rr, -lr * Ri);
  gk_out = gk;
}

// ---- a5 + a7, rare path: both determinants with partial pivoting ------------------------------------------------------
// Every lane gathers the whole matrix M(c) of its trajectory from the TMEM state of the trajectory's lanes (warp
// shuffles) into local memory and eliminates it serially; the L lanes of a trajectory compute the same numbers.
template <int F, int L>
__device__ __noinline__ void pivoted_dets_cml(uint32_t tm, int g, bool with_m, double &Dre, double &Dim, double &dM) {
  using X = Cml<F, L>;
  constexpr int G = X::G, N = X::N, C = X::C, NS = X::NS;
  double A[N * N];
#pragma unroll 1
  for (int i = 0; i < N * N; i++) A[i] = 0.0;
#pragma unroll
  for (int s = 0; s < NS; s++) {
    double col[N];
    tmem_ld_col<F, L>(tm, s, col);
#pragma unroll
    for (int lp = 0; lp < L; lp++) {
      const int a = lp + (s % C) * L;
      if (a >= F) continue;
      const int j = (s / C) * F + a;
#pragma unroll
      for (int i = 0; i < N; i++) A[i * N + j] = __shfl_sync(0xffffffffu, col[i], lp * G + g);
    }
  }
  // 2K = (M_qq + M_pp) + i (M_pq - M_qp), rows/columns in (P, Q) order (Eq. 5, reading R2, reduced coordinates)
  double Br[F * F], Bi[F * F];
#pragma unroll 1
  for (int i = 0; i < F; i++)
#pragma unroll 1
    for (int a = 0; a < F; a++) {
      Br[i * F + a] = A[(F + i) * N + F + a] + A[i * N + a];
      Bi[i * F + a] = A[i * N + F + a] - A[(F + i) * N + a];
    }
  double dr = 1.0, di = 0.0;
#pragma unroll 1
  for (int k = 0; k < F; k++) {
    int p = k;
    double best = -1.0;
#pragma unroll 1
    for (int i = k; i < F; i++) {
      const double m = fma(Br[i * F + k], Br[i * F + k], Bi[i * F + k] * Bi[i * F + k]);
      if (m > best) {
        best = m;
        p = i;
      }
    }
    if (!(best > 0.0)) {  // singular column (0) or nothing but NaN below the diagonal
      dr = di = (best == 0.0) ? 0.0 : nan("");
      break;
    }
    if (p != k) {
#pragma unroll 1
      for (int j = k; j < F; j++) {
        double t = Br[k * F + j];
        Br[k * F + j] = Br[p * F + j];
        Br[p * F + j] = t;
        t = Bi[k * F + j];
        Bi[k * F + j] = Bi[p * F + j];
        Bi[p * F + j] = t;
      }
      dr = -dr;
      di = -di;
    }
    const double pr = Br[k * F + k], pi = Bi[k * F + k];
    {
      const double t = dr * pr - di * pi;
      di = dr * pi + di * pr;
      dr = t;
    }
    // keep the running product in range: only its phase is used
    {
      const double sc = fmax(fabs(dr), fabs(di));
      if (sc > 0.0 && isfinite(sc)) {
        int e;
        frexp(sc, &e);
        dr = ldexp(dr, -e);
        di = ldexp(di, -e);
      }
    }
    const double inv = 1.0 / best;
#pragma unroll 1
    for (int i = k + 1; i < F; i++) {
      const double xr = Br[i * F + k], xi = Bi[i * F + k];
      const double mr = (xr * pr + xi * pi) * inv, mi = (xi * pr - xr * pi) * inv;
#pragma unroll 1
      for (int j = k + 1; j < F; j++) {
        const double ur = Br[k * F + j], ui = Bi[k * F + j];
        Br[i * F + j] -= mr * ur - mi * ui;
        Bi[i * F + j] -= mr * ui + mi * ur;
      }
    }
  }
  Dre = dr;
  Dim = di;
  dM = 1.0;
  if (with_m) {
    double det = 1.0;
#pragma unroll 1
    for (int k = 0; k < N; k++) {
      int p = k;
      double best = -1.0;
#pragma unroll 1
      for (int i = k; i < N; i++) {
        const double m = fabs(A[i * N + k]);
        if (m > best) {
          best = m;
          p = i;
        }
      }
      if (!(best > 0.0)) {
        det = (best == 0.0) ? 0.0 : nan("");
        break;
      }
      if (p != k) {
#pragma unroll 1
        for (int j = k; j < N; j++) {
          const double t = A[k * N + j];
          A[k * N + j] = A[p * N + j];
          A[p * N + j] = t;
        }
        det = -det;
      }
      const double pv = A[k * N + k];
      det *= pv;
#pragma unroll 1
      for (int i = k + 1; i < N; i++) {
        const double m = A[i * N + k] / pv;
#pragma unroll 1
        for (int j = k + 1; j < N; j++) A[i * N + j] -= m * A[k * N + j];
      }
    }
    dM = det;
  }
}

// ---- snapshot: both determinants of M(c) from the TMEM state -----------------------------------------------------------
template <int F, int L, bool WITH_M>
__device__ __forceinline__ void dets_cml(uint32_t tm, const LaneAddr &A, int l, double &Dre, double &Dim, double &dM,
                                         unsigned &gk, unsigned &gm) {
  using X = Cml<F, L>;
  constexpr int C = X::C, N = X::N;
  dM = 1.0;
  gm = 0u;
  if constexpr (WITH_M) {
    lu_mk_cml<F, L>(tm, A, l, dM, gm, Dre, Dim, gk);
  } else {
  double Kr[C][F], Ki[C][F];
#pragma unroll
  for (int s = 0; s < C; s++) {
    double c1[N], c2[N];  // columns d/dP0_a and d/dQ0_a of the lane's mode s
    tmem_ld_col<F, L>(tm, s, c1);
    tmem_ld_col<F, L>(tm, C + s, c2);
#pragma unroll
    for (int i = 0; i < F; i++) {
      Kr[s][i] = c2[F + i] + c1[i];  // dQ2 + dP1
      Ki[s][i] = c2[i] - c1[F + i];  // dP2 - dQ1
    }
  }
  lu_k_cml<F, L>(Kr, Ki, A, l, Dre, Dim, gk);
  }
}

template <int F, int L, int KIND>
__global__ void __launch_bounds__(kThreadsC, 1) k_propagate_cml(const __grid_constant__ PropParams P) {
  using X = Cml<F, L>;
  constexpr int C = X::C, G = X::G, N = X::N, NS = X::NS;
  extern __shared__ double smem[];
  double *cs = smem;
  uint32_t *tm_slot = reinterpret_cast<uint32_t *>(smem + X::NCOEFP + kWarpsC * X::WS);
  {
    const int nco = (KIND == SC_IVR_PES_QFF) ? X::NCOEF_QFF : X::NCOEF_MORSE;
    for (int i = threadIdx.x; i < nco; i += kThreadsC) cs[i] = P.coef[i];
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (warp == 0) tmem_alloc_all(tm_slot);
  tmem_fence_before_sync();
  __syncthreads();
  tmem_fence_after_sync();
  const uint32_t tm_base = *tm_slot;
  // two warps per 32-lane quadrant: warp w owns lanes 32 (w % 4) .. +31, columns 256 (w / 4) .. +255
  const uint32_t tm = tm_base + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)((warp >> 2) * 256);

  const bool act = lane < X::ACT;
  const int l = act ? lane / G : 0, g = act ? lane - l * G : 0;
  double *ws = smem + X::NCOEFP + warp * X::WS;
  LaneAddr A;
  A.g = (uint32_t)__cvta_generic_to_shared(ws + g);
  A.hm = (uint32_t)__cvta_generic_to_shared(ws + X::WSG) + 16 * lane;
  A.g0 = g;
  unsigned gmask = 0u;
#pragma unroll
  for (int i = 0; i < L; i++) gmask |= 1u << (i * G + g);

  // launch shape: cta_full CTAs of kWarpsC warps (whole rounds of one CTA per SM), then the warps that are left spread
  // evenly over one more CTA per SM (cta_warps, +1 for the first cta_warps_rem of them): a step of a CTA takes as long as
  // that of its busiest scheduler, so a last round with one warp per scheduler costs 0.7 of a full one and a nearly
  // empty grid tail a whole one (131072 trajectories of config 4 are 11.07 rounds of 148 x 80)
  const int bt = (int)blockIdx.x - P.cta_full;
  const int nw = bt < 0 ? kWarpsC : P.cta_warps + (bt < P.cta_warps_rem ? 1 : 0);
  const int nthr = nw * 32;
  if (warp >= nw) return;  // after the barrier above; the barriers below count nthr threads
  const long long w0 = bt < 0 ? (long long)blockIdx.x * kWarpsC
                              : (long long)P.cta_full * kWarpsC + (long long)bt * P.cta_warps + min(bt, P.cta_warps_rem);
  const long long jj = (w0 + warp) * G + g;
  const bool valid = act && jj < P.nb;
  const long long jl = jj < P.nb ? jj : P.nb - 1;  // tail groups recompute the last trajectory and store nothing
  const long long jg = P.j0 + jl;

  double Pm[C], Q[C], mu_s[C], Peq_s[C], Qeq_s[C], gq[C];
#pragma unroll
  for (int s = 0; s < C; s++) {
    const int a = l + s * L;
    const bool real = X::EXACT || a < F;
    const int ae = real ? a : 0;
    mu_s[s] = real ? P.mu[ae] : 0.0;
    Peq_s[s] = P.Peq[ae];
    Qeq_s[s] = P.Qeq[ae];
    Pm[s] = real ? P.p0q0[(long long)ae * P.stride + jg] * P.isg[ae] : Peq_s[s];
    Q[s] = real ? P.p0q0[(long long)(F + ae) * P.stride + jg] * P.sg[ae] : Qeq_s[s];
  }
  double Sa = 0.0, Va;

  // M(0) = 1 in TMEM; nothing parked yet
#pragma unroll
  for (int s = 0; s < NS; s++) {
    double col[N];
    const int a = l + (s % C) * L;
#pragma unroll
    for (int i = 0; i < N; i++) col[i] = (i == (s / C) * F + a && (X::EXACT || a < F)) ? 1.0 : 0.0;
    tmem_st_col<F, L>(tm, s, col);
  }
#pragma unroll 1
  for (int e = 0; e < X::HMH; e++) sts2(A.hm + 512 * e, 0.0, 0.0);
  pes_cml<F, L, KIND>(cs, A, l, Q, gq, Va);
  __syncwarp();
  pass_cml<F, L, KIND>(tm, A, P, 0.0, 0.0, 0.0);

  const int lw = X::step_lane(N - 1);  // the lane class that ends up with the last pivots of both eliminations
  bool good = true;
  int det_count = 0;  // steps until the next check
  const int nsteps = P.nsteps;
  const bool has_raw = P.raw != nullptr, has_pq = P.pq_steps != nullptr;
#pragma unroll 1
  for (int c = 0;; c++) {
    if (SCI_CML_SYNC >= 6) {
      if (c == 0 && warp >= 4) asm volatile("bar.sync 7, %0;" ::"r"(nthr) : "memory");
      if (SCI_CML_SYNC == 7 && warp < 4 && c > 0) cta_sync(nthr);
    } else if (SCI_CML_SYNC == 1) {
      cta_sync(nthr);
    }
    const bool last = (c == nsteps);
    const bool check = (det_count == 0) || last;  // warp-uniform
    // a6 (Eq. 3): the lane's share of ln<chi|pq> and of the phase S + arg<chi|pq>, at the integer time c
    if (has_raw) {  // uniform branches only: a divergent one costs reconvergence barriers and an instruction-fetch restart
      double oa = 0.0, ob = Sa;
#pragma unroll
      for (int s = 0; s < C; s++) {
        const bool real = X::EXACT || l + s * L < F;
        const double dq = Qeq_s[s] - Q[s], dp = Peq_s[s] - Pm[s];
        const double ta = fma(-0.25, fma(dq, dq, dp * dp), oa), tb = fma(0.5 * (Peq_s[s] + Pm[s]), dq, ob);
        oa = real ? ta : oa;
        ob = real ? tb : ob;
      }
      if (has_pq) {  // several reference states: the record carries S alone, (P, Q) of the step go out beside it
#pragma unroll
        for (int s = 0; s < C; s++)
          if (valid && (X::EXACT || l + s * L < F))
            P.pq_steps[((long long)c * F + (l + s * L)) * P.raw_stride + jj] = make_double2(Pm[s], Q[s]);
      }
      if (P.raw_plain) {
        oa = 0.0;
        ob = Sa;
      }
      sts(A.g + 8 * (X::O_RED + 2 * l) * G, oa);
      sts(A.g + 8 * (X::O_RED + 2 * l + 1) * G, ob);
    }
    double Dre, Dim, dM;
    unsigned growK, growM;
    if (check) dets_cml<F, L, true>(tm, A, l, Dre, Dim, dM, growK, growM);
    else dets_cml<F, L, false>(tm, A, l, Dre, Dim, dM, growK, growM);
    {
      // static order not safe for this matrix (or forced by the caller): repeat with the pivoted eliminations
      // ... and a rejection by the static-order elimination is confirmed by the pivoted one before it sticks: for a strongly
      // stretched M (entries ~1e5, pivots from 1e5 down to 1e-5) the fixed order loses digits of det M that the multiplier
      // bound does not predict (13 of 131072 trajectories of config 5 at 8000 steps were rejected where the oracle's
      // pivoted elimination finds |det M - 1| ~ 1e-8: tests/test_gpu_parity.py, full-size case 2^17 x 8000)
      const bool suspect = check && good && l == lw && !(fabs(dM - 1.0) <= P.det_tol);
      const bool risky = act && ((growK >= P.grow_k_max) || (check && growM >= P.grow_m_max) || suspect);
      const unsigned rb = __ballot_sync(0xffffffffu, risky);
      if (rb != 0u) {
        double fDre, fDim, fdM;
        pivoted_dets_cml<F, L>(tm, g, check, fDre, fDim, fdM);
        if ((rb & gmask) != 0u) {
          Dre = fDre;
          Dim = fDim;
          dM = fdM;
          if (P.fb_count != nullptr && l == 0 && valid) atomicAdd(P.fb_count, 1ULL);  // statistics only
        }
      }
    }
    // a8 input record, written by the lane that holds the last pivots
    if (has_raw) {
      __syncwarp();
      double s0 = 0.0, s1 = 0.0;
#pragma unroll
      for (int i = 0; i < L; i++) {
        s0 += lds(A.g + 8 * (X::O_RED + 2 * i) * G);
        s1 += lds(A.g + 8 * (X::O_RED + 2 * i + 1) * G);
      }
      // only the phase of the determinant is used: bring it to unit scale (a power of two, exact)
      const int ex = (int)((max(abs_hi(Dre), abs_hi(Dim)) >> 20) & 0x7ffu);
      const double sc = (ex > 0 && ex < 0x7fe) ? __hiloint2double((0x7fe - ex) << 20, 0) : 1.0;  // 2^(1023 - ex)
      if (valid && l == lw) P.raw[(long long)c * P.raw_stride + jj] = make_double4(s0, s1, Dre * sc, Dim * sc);
    }
    if (SCI_CML_SYNC >= 6) {
      // the warps 4.. run half a time step behind the warps 0..3 (one of each per scheduler): while one does the
      // eliminations the other does the PES and the pass
      if (c == 0 && warp < 4) asm volatile("bar.arrive 7, %0;" ::"r"(nthr) : "memory");
      if (SCI_CML_SYNC == 7 && warp >= 4 && !last) cta_sync(nthr);
    }
    // a7: |det M - 1| <= tol and finite, every det_stride steps and at the end
    if (check) {
      // finite <=> exponent field below 0x7ff: one integer maximum over the high words
      unsigned hx = abs_hi(Sa);
#pragma unroll
      for (int s = 0; s < C; s++) hx = max(hx, max(abs_hi(Pm[s]), abs_hi(Q[s])));
      const bool okd = (l != lw) | (fabs(dM - 1.0) <= P.det_tol);
      good = good & okd & (hx < 0x7ff00000u);
      det_count = P.det_stride;
    }
    det_count--;
    if (last) break;
    // a2-a4 (R10, R11): evaluation points of the "kick b_s, drift a_s" composition
#pragma unroll 1
    for (int e = 0; e < P.npoints; e++) {
      const double post = P.pt_post[e], adt = P.pt_drift[e];
      const double pre = P.pt_pre[(e + 1 == P.npoints) ? 0 : e + 1];
      Sa = fma(-post, Va, Sa);
#pragma unroll
      for (int s = 0; s < C; s++) {
        Pm[s] = fma(-post, gq[s], Pm[s]);
        Sa = fma(0.5 * adt * mu_s[s], Pm[s] * Pm[s], Sa);
        Q[s] = fma(adt * mu_s[s], Pm[s], Q[s]);
      }
      __syncwarp();  // every lane is done with the previous Hessian
      pes_cml<F, L, KIND>(cs, A, l, Q, gq, Va);
      __syncwarp();
      pass_cml<F, L, KIND>(tm, A, P, post, adt, pre);
      Sa = fma(-pre, Va, Sa);
#pragma unroll
      for (int s = 0; s < C; s++) Pm[s] = fma(-pre, gq[s], Pm[s]);
    }
  }

  // outputs
  const unsigned bal = __ballot_sync(0xffffffffu, good);
  const bool group_good = ((bal & gmask) == gmask);
  double Stot = 0.0;
#pragma unroll
  for (int i = 0; i < L; i++) Stot += __shfl_sync(0xffffffffu, Sa, i * G + g);
  if (valid) {
    if (P.good != nullptr && l == 0) P.good[jj] = group_good ? 1 : 0;
    if (P.S_out != nullptr && l == 0) P.S_out[jg] = Stot;
    if (P.pq_out != nullptr) {
#pragma unroll
      for (int s = 0; s < C; s++) {
        const int a = l + s * L;
        if (!X::EXACT && a >= F) continue;
        P.pq_out[(long long)a * P.stride + jg] = Pm[s] * P.sg[a];
        P.pq_out[(long long)(F + a) * P.stride + jg] = Q[s] * P.isg[a];
      }
    }
  }
  if (P.M_out != nullptr) {
    // M_xy[i][a], reduced -> caller's units: p = sg P, q = Q / sg
#pragma unroll
    for (int s = 0; s < NS; s++) {
      double col[N];
      tmem_ld_col<F, L>(tm, s, col);
      const int a = l + (s % C) * L, h = s / C;
      if (!valid || (!X::EXACT && a >= F)) continue;
      const double ca = h == 0 ? P.isg[a] : P.sg[a];
      const long long blk = (long long)F * F * P.stride;
#pragma unroll
      for (int i = 0; i < F; i++) {
        const long long e = ((long long)i * F + a) * P.stride + jg;
        P.M_out[(h == 0 ? 0 : 1) * blk + e] = col[i] * P.sg[i] * ca;
        P.M_out[(h == 0 ? 2 : 3) * blk + e] = col[F + i] * P.isg[i] * ca;
      }
    }
  }
  tmem_fence_before_sync();
  cta_sync(nthr);
  if (warp == 0) tmem_free_all(tm_base);
}

// ---- debug kernel for a1: same pes_cml, caller's units out ---------------------------------------------------------------
template <int F, int L, int KIND>
__global__ void __launch_bounds__(kThreadsC) k_eval_pes_cml(const double *__restrict__ coef, const double *__restrict__ sgv,
                                                            const double *__restrict__ q, long long n, double *V,
                                                            double *gout, double *H) {
  using X = Cml<F, L>;
  constexpr int C = X::C, G = X::G;
  extern __shared__ double smem[];
  double *cs = smem;
  {
    const int nco = (KIND == SC_IVR_PES_QFF) ? X::NCOEF_QFF : X::NCOEF_MORSE;
    for (int i = threadIdx.x; i < nco; i += kThreadsC) cs[i] = coef[i];
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool act = lane < X::ACT;
  const int l = act ? lane / G : 0, g = act ? lane - l * G : 0;
  double *ws = smem + X::NCOEFP + warp * X::WS;
  LaneAddr A;
  A.g = (uint32_t)__cvta_generic_to_shared(ws + g);
  A.hm = 0;
  A.g0 = g;
  auto HSv = [&](int e) { return ws[(X::O_HS + e) * G + g]; };
  const long long jj = ((long long)blockIdx.x * kWarpsC + warp) * G + g;
  const bool valid = act && jj < n;
  const long long jl = jj < n ? jj : n - 1;
  double Q[C], gq[C], Va;
#pragma unroll
  for (int s = 0; s < C; s++) {
    const int a = l + s * L;
    Q[s] = (X::EXACT || a < F) ? q[(long long)a * n + jl] * sgv[a] : 0.0;
  }
  pes_cml<F, L, KIND>(cs, A, l, Q, gq, Va);
  __syncwarp();
  double Vt = 0.0;
#pragma unroll
  for (int i = 0; i < L; i++) Vt += __shfl_sync(0xffffffffu, Va, i * G + g);
  if (!valid) return;
  if (l == 0) V[jl] = Vt;
#pragma unroll
  for (int s = 0; s < C; s++) {
    const int a = l + s * L;
    if (!X::EXACT && a >= F) continue;
    gout[(long long)a * n + jl] = gq[s] * sgv[a];
    if (KIND != SC_IVR_PES_QFF) {
      for (int b = 0; b < F; b++) H[((long long)a * F + b) * n + jl] = (b == a) ? HSv(a) * sgv[a] * sgv[a] : 0.0;
    } else {
#pragma unroll
      for (int d = 0; d < X::ND; d++) {
        const int b = (a + d) % F;
        const double h = HSv(d * F + a) * sgv[a] * sgv[b];
        H[((long long)a * F + b) * n + jl] = h;
        H[((long long)b * F + a) * n + jl] = h;
      }
    }
  }
}

template <int F, int L, int KIND>
cudaError_t launch_prop_cml(const PropParams &P, cudaStream_t st) {
  using X = Cml<F, L>;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  // per device and cheap: set on every launch, no process-wide flag (as chirp.cu and spectrum.cu do)
  e = cudaFuncSetAttribute(k_propagate_cml<F, L, KIND>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)X::SMEM_LAUNCH);
  if (e != cudaSuccess) return e;
  int sm = 0;
  e = cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return e;
  const long long W = (P.nb + X::G - 1) / X::G;                                  // warps of work
  const long long per_round = (long long)sm * kWarpsC;
  const long long full = W / per_round * sm;                                     // CTAs of whole rounds
  const long long left = W - full * kWarpsC;                                     // warps of the last, partial round
  const long long tail = left < sm ? left : sm;
  PropParams Q = P;
  Q.cta_full = (int)full;
  Q.cta_warps = tail ? (int)(left / tail) : 0;
  Q.cta_warps_rem = tail ? (int)(left % tail) : 0;
  k_propagate_cml<F, L, KIND><<<(unsigned)(full + tail), kThreadsC, X::SMEM_LAUNCH, st>>>(Q);
  return cudaGetLastError();
}

template <int F, int L, int KIND>
cudaError_t launch_pes_cml(const double *coef, const double *sg, const double *q, long long n, double *V, double *g, double *H,
                           cudaStream_t st) {
  using X = Cml<F, L>;
  cudaError_t e = cudaFuncSetAttribute(k_eval_pes_cml<F, L, KIND>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)X::SMEM);
  if (e != cudaSuccess) return e;
  const int tpb = kWarpsC * X::G;
  const long long blocks = (n + tpb - 1) / tpb;
  k_eval_pes_cml<F, L, KIND><<<(unsigned)blocks, kThreadsC, X::SMEM, st>>>(coef, sg, q, n, V, g, H);
  return cudaGetLastError();
}

// Host: reduce the caller's coefficients to the packed block of Cml<F, L>.
//   Phi~_ijk = Phi_ijk / sqrt(g_i g_j g_k),  P~_ij = Phi_iijj / (g_i g_j),  w~_a^2 = w_a^2 / g_a   (QFF)
//   a~ = a / sqrt(g),  Q_e = sqrt(g) q_e                                                           (Morse)
template <int F, int L>
size_t pack_cml(int kind, const double *c, const double *gamma, double *out) {
  using X = Cml<F, L>;
  constexpr int C = X::C, ND = X::ND;
  if (kind != SC_IVR_PES_QFF) {
    const size_t n = X::NCOEF_MORSE;
    if (!out) return n;
    for (size_t i = 0; i < n; i++) out[i] = 0.0;
    for (int l = 0; l < L; l++)
      for (int s = 0; s < C; s++) {
        const int a = l + s * L;
        if (a >= F) continue;
        const double sg = sqrt(gamma[a]);
        out[(s * 3 + 0) * L + l] = c[4 * a];
        out[(s * 3 + 1) * L + l] = c[4 * a + 1] / sg;
        out[(s * 3 + 2) * L + l] = c[4 * a + 2] * sg;
      }
    return n;
  }
  const size_t n = X::NCOEF_QFF;
  if (!out) return n;
  for (size_t i = 0; i < n; i++) out[i] = 0.0;
  std::vector<double> phi((size_t)F * F * F, 0.0), pq((size_t)F * F, 0.0);
  const double *cub = c + F;
  size_t m = 0;
  for (int i = 0; i < F; i++)
    for (int j = i; j < F; j++)
      for (int k = j; k < F; k++) {
        const double v = cub[m++] / sqrt(gamma[i] * gamma[j] * gamma[k]);
        const int p[6][3] = {{i, j, k}, {i, k, j}, {j, i, k}, {j, k, i}, {k, i, j}, {k, j, i}};
        for (auto &t : p) phi[((size_t)t[0] * F + t[1]) * F + t[2]] = v;
      }
  const double *qua = cub + m;
  m = 0;
  for (int i = 0; i < F; i++)
    for (int j = i; j < F; j++) {
      const double v = qua[m++] / (gamma[i] * gamma[j]);
      pq[i * F + j] = pq[j * F + i] = v;
    }
  std::vector<double> list(X::LAP);
  for (int l = 0; l < L; l++)
    for (int s = 0; s < C; s++) {
      const int a = l + s * L;
      if (a >= F) continue;
      for (auto &x : list) x = 0.0;
      for (int d = 0; d < ND; d++)
        for (int k = 0; k < F; k++) list[X::L_C3 + d * F + k] = phi[((size_t)a * F + (a + d) % F) * F + k];
      for (int j = 0; j < F; j++) list[X::L_C4U + j] = pq[a * F + j];
      for (int d = 0; d < ND; d++) list[X::L_C4D + d] = pq[a * F + (a + d) % F];
      list[X::L_W2] = c[a] * c[a] / gamma[a];
      for (int i = 0; i < X::LAP; i++) out[((size_t)(s * (X::LAP / 2) + i / 2) * L + l) * 2 + (i & 1)] = list[i];
    }
  return n;
}

}  // namespace

#define SCI_CAT2(a, b) a##b
#define SCI_CAT(a, b) SCI_CAT2(a, b)

size_t SCI_CAT(sci_cml_pack_f, SCI_CML_INST_F)(int kind, const double *c, const double *gamma, double *out) {
  return pack_cml<SCI_CML_INST_F, SCI_CML_INST_L>(kind, c, gamma, out);
}

cudaError_t SCI_CAT(sci_cml_prop_f, SCI_CML_INST_F)(int kind, const PropParams &P, cudaStream_t st) {
  return kind == SC_IVR_PES_QFF ? launch_prop_cml<SCI_CML_INST_F, SCI_CML_INST_L, SC_IVR_PES_QFF>(P, st)
                                : launch_prop_cml<SCI_CML_INST_F, SCI_CML_INST_L, SC_IVR_PES_MORSE_UNCOUPLED>(P, st);
}

cudaError_t SCI_CAT(sci_cml_pes_f, SCI_CML_INST_F)(int kind, const double *coef, const double *sg, const double *q, long long n,
                                                   double *V, double *g, double *H, cudaStream_t st) {
  return kind == SC_IVR_PES_QFF ? launch_pes_cml<SCI_CML_INST_F, SCI_CML_INST_L, SC_IVR_PES_QFF>(coef, sg, q, n, V, g, H, st)
                                : launch_pes_cml<SCI_CML_INST_F, SCI_CML_INST_L, SC_IVR_PES_MORSE_UNCOUPLED>(coef, sg, q, n, V, g, H, st);
}

#else
// ======== dispatcher ========================================================================================================
#define X(f, l)                                                                                                      \
  size_t sci_cml_pack_f##f(int kind, const double *c, const double *gamma, double *out);                             \
  cudaError_t sci_cml_prop_f##f(int kind, const PropParams &P, cudaStream_t st);                                     \
  cudaError_t sci_cml_pes_f##f(int kind, const double *coef, const double *sg, const double *q, long long n, double *V, \
                               double *g, double *H, cudaStream_t st);
SCI_CML_FOR_EACH(X)
#undef X

int sci_cml_lanes(int F) {
  switch (F) {
#define X(f, l) case f: return l;
    SCI_CML_FOR_EACH(X)
#undef X
  }
  return 0;
}

int sci_cml_traj_per_block(int F) {
  const int L = sci_cml_lanes(F);
  return L ? kWarpsC * (32 / L) : 0;
}

size_t sci_cml_pack_coeffs(int F, int kind, const double *c, const double *gamma, double *out) {
  switch (F) {
#define X(f, l) case f: return sci_cml_pack_f##f(kind, c, gamma, out);
    SCI_CML_FOR_EACH(X)
#undef X
  }
  return 0;
}

cudaError_t sci_cml_launch_propagate(int F, int kind, const PropParams &P, cudaStream_t st) {
  switch (F) {
#define X(f, l) case f: return sci_cml_prop_f##f(kind, P, st);
    SCI_CML_FOR_EACH(X)
#undef X
  }
  return cudaErrorInvalidValue;
}

cudaError_t sci_cml_launch_eval_pes(int F, int kind, const double *coef, const double *sg, const double *q, long long n,
                                    double *V, double *g, double *H, cudaStream_t st) {
  switch (F) {
#define X(f, l) case f: return sci_cml_pes_f##f(kind, coef, sg, q, n, V, g, H, st);
    SCI_CML_FOR_EACH(X)
#undef X
  }
  return cudaErrorInvalidValue;
}
#endif
