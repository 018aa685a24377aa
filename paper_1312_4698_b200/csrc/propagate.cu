// Kernel A: fused PES (a1) + symplectic step (a2) + monodromy (a3) + action (a4) + Herman-Kluk
// determinant (a5) + coherent-state overlap exponent (a6) + det M quality flag (a7).
//
// Mapping: F lanes per trajectory, G = floor(32/F) trajectories per warp, lane = a * G + g
// (a = mode / column index, g = trajectory of the warp).
// Lane a of a group owns (P_a, Q_a), its share S_a of the action and the two tangent vectors
// d(P,Q)/dP0_a and d(P,Q)/dQ0_a (columns a and F+a of the monodromy matrix, 2F doubles each), all in
// registers.  The tangent map of a kick needs the full Hessian, so the lanes of a group compute
// disjoint Hessian entries and exchange them through a per-group shared-memory slot.
// Column a of the Herman-Kluk matrix lives entirely on lane a, so det K is a column-distributed
// elimination with column pivoting: the pivot column is broadcast with __shfl_sync from a dynamic
// source lane, no data is ever swapped.
//
// Everything runs in reduced coordinates Q = sqrt(gamma) q, P = p / sqrt(gamma).
#include "common.cuh"

namespace {

constexpr int kThreads = 128;

__device__ __forceinline__ double fast_rcp(double x) {
  // MUFU.RCP64H seed (2^-23 relative) + two Newton steps: ~1 ulp for normal x, no slow path.
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  return r;
}

template <int F>
struct Geo {
  static constexpr int G = 32 / F;         // trajectories per warp
  static constexpr int ACT = G * F;        // active lanes
  static constexpr unsigned AMASK = ACT == 32 ? 0xffffffffu : ((1u << ACT) - 1u);
  static constexpr int ND = F / 2 + 1;     // Hessian entries (a, (a+d)%F), d = 0..ND-1, computed by lane a
  static constexpr int NR = (F - 1) / 2;   // cubic-gradient terms received from lanes a-d
  static constexpr int FP = (F + 1) & ~1;  // F padded to even (16-byte alignment of the slots)
  static constexpr int NH = F * ND;
  static constexpr int NHP = (NH + 1) & ~1;
  static constexpr int KB = 2 * F;             // doubles per Herman-Kluk broadcast buffer (F double2)
  static constexpr int MB = 2 * F + 2;         // doubles per monodromy broadcast buffer (reciprocal + 2F-1 rows, even)
  static constexpr int WS = FP + NHP + 2 * F + 2 * KB + 2 * MB;  // doubles of scratch per group: qs, Hs, red, kb[2], mb[2]
  // packed coefficient block (QFF): lane a reads its own list of LA coefficients two at a time, pair t of lane a at
  // double2 index t * F + a (adjacent lanes read adjacent 16-byte words).  Positions within the list:
  static constexpr int L_C3 = 0;                // [ND][F]  (d, k) = Phi~[a][(a+d)%F][k]
  static constexpr int L_C4U = L_C3 + ND * F;   // [F]      j      = P~[a][j]
  static constexpr int L_C4D = L_C4U + F;       // [ND]     d      = P~[a][(a+d)%F]
  static constexpr int L_W2 = L_C4D + ND;       //                   omega_a^2 / gamma_a
  static constexpr int LA = L_W2 + 1;
  static constexpr int LAP = (LA + 1) & ~1;
  static constexpr int NCOEF_QFF = LAP * F;
  static constexpr int NCOEF_MORSE = 3 * F;     // D[F], a~[F], Qe[F]
  static constexpr int NCOEF = NCOEF_QFF > NCOEF_MORSE ? NCOEF_QFF : NCOEF_MORSE;
  static constexpr int NCOEFP = (NCOEF + 1) & ~1;
};

// ---- a1: potential, own gradient component, ND Hessian entries (reduced coordinates) --------------
// QFF (BASELINE.json configs 2-5, stand-in for the fitted surfaces of PAPER.md:157):
//   H3_ab = sum_k Phi_abk Q_k,  g3_a = 1/2 sum_b H3_ab Q_b,  u_a = sum_j P_aj Q_j^2,
//   g4_a = Q_a (u_a/2 - P_aa Q_a^2/3),  H4_aa = u_a/2,  H4_ab = P_ab Q_a Q_b,
//   V = sum_a Q_a (w_a^2 Q_a/2 + g3_a/3 + g4_a/4)   (Euler's theorem on the homogeneous parts).
// Morse: y = exp(-a (Q - Q_e)), V = D (1-y)^2, g = 2 D a y (1-y), H = 2 D a^2 y (2y-1).
// Writes the entries to Hs[d*F + a]; the caller reads them back after __syncwarp.
template <int F, int KIND>
__device__ __forceinline__ void pes_group(const double *__restrict__ cs, double *qs, double *Hs, int a, int gbase,
                                          const int (&fwd)[Geo<F>::ND], const int (&bwd)[Geo<F>::ND], double Q,
                                          double &g, double &Va, double (&Hent)[Geo<F>::ND]) {
  using X = Geo<F>;
  if (KIND == SC_IVR_PES_QFF) {
    double q[F];
    if (F > 1) {
      qs[a] = Q;
      __syncwarp(X::AMASK);
#pragma unroll
      for (int i = 0; i < F; i++) q[i] = qs[i];
    } else {
      q[0] = Q;
    }
    double qd[X::ND];
    qd[0] = Q;
#pragma unroll
    for (int d = 1; d < X::ND; d++) qd[d] = qs[fwd[d]];
    double cf[X::LAP];
    {
      const double2 *c2 = reinterpret_cast<const double2 *>(cs);
#pragma unroll
      for (int t = 0; t < X::LAP / 2; t++) {
        const double2 v = c2[t * F + a];
        cf[2 * t] = v.x;
        cf[2 * t + 1] = v.y;
      }
    }
    double u = 0.0;
#pragma unroll
    for (int j = 0; j < F; j++) u = fma(cf[X::L_C4U + j], q[j] * q[j], u);
    double h3[X::ND];
#pragma unroll
    for (int d = 0; d < X::ND; d++) {
      double s = 0.0;
#pragma unroll
      for (int k = 0; k < F; k++) s = fma(cf[X::L_C3 + d * F + k], q[k], s);
      h3[d] = s;
    }
    double s3 = 0.0;
#pragma unroll
    for (int d = 0; d < X::ND; d++) s3 = fma(h3[d], qd[d], s3);
#pragma unroll
    for (int d = 1; d <= X::NR; d++) s3 += __shfl_sync(X::AMASK, h3[d] * Q, bwd[d] * X::G + gbase);
    const double w2 = cf[X::L_W2];
    const double paa = cf[X::L_C4D];
    const double g3 = 0.5 * s3;
    const double g4 = Q * (0.5 * u - (1.0 / 3.0) * paa * Q * Q);
    g = fma(w2, Q, g3 + g4);
    Va = Q * (0.5 * w2 * Q + (1.0 / 3.0) * g3 + 0.25 * g4);
    Hent[0] = w2 + h3[0] + 0.5 * u;
#pragma unroll
    for (int d = 1; d < X::ND; d++) Hent[d] = fma(cf[X::L_C4D + d] * Q, qd[d], h3[d]);
#pragma unroll
    for (int d = 0; d < X::ND; d++) Hs[d * F + a] = Hent[d];
  } else {
    const double D = cs[a], at = cs[F + a], Qe = cs[2 * F + a];
    const double y = exp(-at * (Q - Qe));
    Va = D * (1.0 - y) * (1.0 - y);
    g = 2.0 * D * at * y * (1.0 - y);
    Hent[0] = 2.0 * D * at * at * y * (2.0 * y - 1.0);
#pragma unroll
    for (int d = 1; d < X::ND; d++) Hent[d] = 0.0;
    Hs[a] = Hent[0];
  }
}

// ---- a3 helper: HM1 = H dQ1, HM2 = H dQ2 from the group's shared Hessian slot ------------------------
template <int F, int KIND>
__device__ __forceinline__ void hessian_times_tangent(const double *Hs, const double (&dQ1)[F], const double (&dQ2)[F],
                                                      double (&HM1)[F], double (&HM2)[F]) {
  using X = Geo<F>;
#pragma unroll
  for (int i = 0; i < F; i++) {
    const double h = Hs[i];
    HM1[i] = h * dQ1[i];
    HM2[i] = h * dQ2[i];
  }
  if (KIND == SC_IVR_PES_QFF) {
#pragma unroll
    for (int d = 1; d < X::ND; d++) {
#pragma unroll
      for (int i = 0; i < F; i++) {
        if (F % 2 == 0 && d == F / 2 && i >= F / 2) continue;  // pair (i, i+F/2) already taken from lane i-F/2
        const int l = (i + d) % F;
        const double h = Hs[d * F + i];
        HM1[i] = fma(h, dQ1[l], HM1[i]);
        HM1[l] = fma(h, dQ1[i], HM1[l]);
        HM2[i] = fma(h, dQ2[l], HM2[i]);
        HM2[l] = fma(h, dQ2[i], HM2[l]);
      }
    }
  }
}

// ---- a5: det of the F x F complex matrix whose column a is on lane a (Eq. 5) -------------
// Elimination of rows k = 0..F-1 by column operations; the pivot for row k is the not-yet-used column with
// the largest |A[k][.]| (REDUX over the group's lanes on the high word of |.|^2, lane id in the low bits).
// det = sign(permutation) * product of pivots; the sign is the parity of the inversions of the pick order.
template <int F>
__device__ __forceinline__ void det_columns_complex(double (&Are)[F], double (&Aim)[F], int gbase, int a,
                                                    unsigned gmask, double &Dre, double &Dim) {
  using X = Geo<F>;
  if (F == 1) {
    Dre = Are[0];
    Dim = Aim[0];
    return;
  }
  unsigned umask = (1u << F) - 1u;
  bool used = false;
  unsigned par = 0;
  double dre = 1.0, dim = 0.0;
#pragma unroll
  for (int k = 0; k < F; k++) {
    const double mag = fma(Are[k], Are[k], Aim[k] * Aim[k]);
    const unsigned key = used ? 0u : ((((unsigned)__double2hiint(mag)) & 0xFFFFFFE0u) | (unsigned)a) + 32u;
    const unsigned best = __reduce_max_sync(gmask, key);
    const int srcg = (int)((best - 32u) & 31u);
    const int src = srcg * X::G + gbase;
    par ^= __popc(umask & ((1u << srcg) - 1u));
    umask &= ~(1u << srcg);
    double pr[F], pi[F];
#pragma unroll
    for (int i = k; i < F; i++) {
      pr[i] = __shfl_sync(X::AMASK, Are[i], src);
      pi[i] = __shfl_sync(X::AMASK, Aim[i], src);
    }
    const double t = dre * pr[k] - dim * pi[k];
    dim = fma(dre, pi[k], dim * pr[k]);
    dre = t;
    if (k < F - 1) {
      const double rn = fast_rcp(fma(pr[k], pr[k], pi[k] * pi[k]));
      const double ir = pr[k] * rn, ii = -pi[k] * rn;
      const double mr = Are[k] * ir - Aim[k] * ii;
      const double mi = fma(Are[k], ii, Aim[k] * ir);
#pragma unroll
      for (int i = k + 1; i < F; i++) {
        Are[i] = fma(-mr, pr[i], fma(mi, pi[i], Are[i]));
        Aim[i] = fma(-mr, pi[i], fma(-mi, pr[i], Aim[i]));
      }
    }
    if (a == srcg) used = true;
  }
  if (par & 1u) {
    dre = -dre;
    dim = -dim;
  }
  Dre = dre;
  Dim = dim;
}

// ---- a7: det of the 2F x 2F monodromy matrix; lane a holds columns a (in C[0..2F)) and F+a (C[2F..4F)) -----
// Same column-pivoted elimination, two local columns per lane.  Reads its input from local memory so
// that the caller's register state is not duplicated.
template <int F>
__device__ __noinline__ double det_columns_real2(const double *C, int gbase, int a, unsigned gmask) {
  using X = Geo<F>;
  constexpr int N = 2 * F;
  double C1[N], C2[N];
#pragma unroll
  for (int i = 0; i < N; i++) {
    C1[i] = C[i];
    C2[i] = C[N + i];
  }
  bool used1 = false, used2 = false;
  unsigned umask = (N >= 32) ? 0xffffffffu : ((1u << N) - 1u);
  unsigned par = 0;
  double det = 1.0;
#pragma unroll
  for (int k = 0; k < N; k++) {
    const double m1 = used1 ? -1.0 : fabs(C1[k]);
    const double m2 = used2 ? -1.0 : fabs(C2[k]);
    const bool sel = m2 > m1;
    const double m = sel ? m2 : m1;
    const unsigned col_mine = (unsigned)(sel ? F + a : a);
    const unsigned key = (m < 0.0) ? 0u : ((((unsigned)__double2hiint(m)) & 0xFFFFFFE0u) | col_mine) + 32u;
    const unsigned best = (F == 1) ? key : __reduce_max_sync(gmask, key);
    const int col = (int)((best - 32u) & 31u);
    const bool ssel = col >= F;
    const int srcg = ssel ? col - F : col;
    const int src = srcg * X::G + gbase;
    par ^= __popc(umask & ((1u << col) - 1u));
    umask &= ~(1u << col);
    double pv[N];
#pragma unroll
    for (int i = k; i < N; i++) {
      const double v = ssel ? C2[i] : C1[i];
      pv[i] = (F == 1) ? v : __shfl_sync(X::AMASK, v, src);
    }
    det *= pv[k];
    if (k < N - 1) {
      const double r = fast_rcp(pv[k]);
      const double mm1 = C1[k] * r, mm2 = C2[k] * r;
#pragma unroll
      for (int i = k + 1; i < N; i++) {
        C1[i] = fma(-mm1, pv[i], C1[i]);
        C2[i] = fma(-mm2, pv[i], C2[i]);
      }
    }
    if (a == srcg) {
      if (ssel) used2 = true; else used1 = true;
    }
  }
  return (par & 1u) ? -det : det;
}

// ---- a5 + a7, rare path: both determinants with pivoting, from the state AFTER the opening kick -------------------
// st = (dP1, dQ1, dP2, dQ2) of the calling lane with the kick of weight bdt0 already applied; it is undone here with
// H dQ recomputed from the group's Hessian slot (still the one of the current q).
template <int F, int KIND>
__device__ __noinline__ void pivoted_dets(const double *st, const double *Hs, double bdt0, int gbase, int a, unsigned gmask,
                                          bool with_m, double &Dre, double &Dim, double &dM) {
  double dP1[F], dQ1[F], dP2[F], dQ2[F], HM1[F], HM2[F];
#pragma unroll
  for (int i = 0; i < F; i++) {
    dP1[i] = st[i];
    dQ1[i] = st[F + i];
    dP2[i] = st[2 * F + i];
    dQ2[i] = st[3 * F + i];
  }
  hessian_times_tangent<F, KIND>(Hs, dQ1, dQ2, HM1, HM2);
  double buf[4 * F];
  double Are[F], Aim[F];
#pragma unroll
  for (int i = 0; i < F; i++) {
    const double p1 = fma(bdt0, HM1[i], dP1[i]), p2 = fma(bdt0, HM2[i], dP2[i]);
    buf[i] = p1;
    buf[F + i] = dQ1[i];
    buf[2 * F + i] = p2;
    buf[3 * F + i] = dQ2[i];
    Are[i] = dQ2[i] + p1;
    Aim[i] = p2 - dQ1[i];
  }
  det_columns_complex<F>(Are, Aim, gbase, a, gmask, Dre, Dim);
  dM = with_m ? det_columns_real2<F>(buf, gbase, a, gmask) : 1.0;
}

// ---- a5 + a7, common path: both determinants by LU in a STATIC pivot order ---------------------------------------
// Lane a owns column a of the F x F complex matrix 2K (Are, Aim) and columns a (C1) and F+a (C2) of the 2F x 2F
// monodromy matrix, rows in (P, Q) order.  Step k eliminates row k with the diagonal pivot: the owner of column k
// publishes (1/pivot, rest of its column) in a per-group shared-memory buffer (two buffers alternate, one
// __syncwarp per step), every lane scales its row-k element by the reciprocal and updates its column(s).  The two
// eliminations are independent and interleaved step by step so that each hides the other's latency.
// No pivot search: the order is fixed, so there is no data-dependent control flow or register selection.  Its
// numerical safety is monitored instead: grow = largest magnitude (IEEE high word) of any multiplier of a live
// column.  A caller that sees grow above its bound repeats the step with the pivoted routines above (rare:
// DESIGN.md "Static-order LU").  Results: on lane F-1, (Dre, Dim) = det(2K) * |R|^2 (a positive multiple of
// det 2K: only its phase is used downstream, Eq. 10) and detM = det M.
template <int F, bool WITH_M>
__device__ __forceinline__ void lu_static(double (&Are)[F], double (&Aim)[F], double (&C1)[2 * F], double (&C2)[2 * F],
                                          double2 *kb, double *mb, int a, unsigned amask, double &Dre, double &Dim,
                                          double &detM, unsigned &growK, unsigned &growM) {
  using X = Geo<F>;
  constexpr int N = 2 * F;
  constexpr int NSTEP = WITH_M ? N - 1 : F - 1;
  double Rr = 1.0, Ri = 0.0, Rm = 1.0;
  unsigned gk = 0u, gm = 0u;
#pragma unroll
  for (int k = 0; k < NSTEP; k++) {
    const bool doK = k < F - 1;
    if (doK) {
      double2 *b = kb + (k & 1) * F;
      const double rn = fast_rcp(fma(Are[k], Are[k], Aim[k] * Aim[k]));
      if (a == k) {
        b[0] = make_double2(Are[k] * rn, -Aim[k] * rn);
#pragma unroll
        for (int i = k + 1; i < F; i++) b[i - k] = make_double2(Are[i], Aim[i]);
      }
    }
    if (WITH_M) {
      double2 *b = reinterpret_cast<double2 *>(mb + (k & 1) * X::MB);
      const bool own = (k < F) ? (a == k) : (a == k - F);
      double(&C)[N] = (k < F) ? C1 : C2;
      const double r = fast_rcp(C[k]);
      if (own) {
#pragma unroll
        for (int t = 0; 2 * t < N - k; t++) {
          const double x = (t == 0) ? r : C[k + 2 * t];
          const double y = (k + 2 * t + 1 < N) ? C[k + 2 * t + 1] : 0.0;
          b[t] = make_double2(x, y);
        }
      }
    }
    if (F > 1) __syncwarp(amask);
    if (doK) {
      const double2 *b = kb + (k & 1) * F;
      const double2 r = b[0];
      const double mr = Are[k] * r.x - Aim[k] * r.y;
      const double mi = fma(Are[k], r.y, Aim[k] * r.x);
      if (a > k) gk = max(gk, max((unsigned)__double2hiint(mr) & 0x7fffffffu, (unsigned)__double2hiint(mi) & 0x7fffffffu));
      const double t = Rr * r.x - Ri * r.y;
      Ri = fma(Rr, r.y, Ri * r.x);
      Rr = t;
#pragma unroll
      for (int i = k + 1; i < F; i++) {
        const double2 pv = b[i - k];
        Are[i] = fma(-mr, pv.x, fma(mi, pv.y, Are[i]));
        Aim[i] = fma(-mr, pv.y, fma(-mi, pv.x, Aim[i]));
      }
    }
    if (WITH_M) {
      const double2 *b = reinterpret_cast<const double2 *>(mb + (k & 1) * X::MB);
      double2 pv = b[0];
      const double r = pv.x;
      Rm *= r;
      const double m2 = C2[k] * r;
      if (k < F || a > k - F) gm = max(gm, (unsigned)__double2hiint(m2) & 0x7fffffffu);
      if (k < F) {
        const double m1 = C1[k] * r;
        if (a > k) gm = max(gm, (unsigned)__double2hiint(m1) & 0x7fffffffu);
#pragma unroll
        for (int i = k + 1; i < N; i++) {
          const int e = i - k;
          if ((e & 1) == 0) pv = b[e >> 1];
          const double x = (e & 1) ? pv.y : pv.x;
          C1[i] = fma(-m1, x, C1[i]);
          C2[i] = fma(-m2, x, C2[i]);
        }
      } else {
#pragma unroll
        for (int i = k + 1; i < N; i++) {
          const int e = i - k;
          if ((e & 1) == 0) pv = b[e >> 1];
          const double x = (e & 1) ? pv.y : pv.x;
          C2[i] = fma(-m2, x, C2[i]);
        }
      }
    }
  }
  // det 2K = p_{F-1} / R  ~  p_{F-1} conj(R);   det M = p_{2F-1} / R_m
  Dre = fma(Are[F - 1], Rr, Aim[F - 1] * Ri);
  Dim = fma(Aim[F - 1], Rr, -Are[F - 1] * Ri);
  detM = WITH_M ? C2[N - 1] * fast_rcp(Rm) : 1.0;
  growK = gk;
  growM = gm;
}

template <int F, int KIND>
__global__ void __launch_bounds__(kThreads) k_propagate(const __grid_constant__ PropParams P) {
  using X = Geo<F>;
  extern __shared__ double smem[];
  double *cs = smem;
  {
    const int nco = (KIND == SC_IVR_PES_QFF) ? X::NCOEF_QFF : X::NCOEF_MORSE;
    for (int i = threadIdx.x; i < nco; i += kThreads) cs[i] = P.coef[i];
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane >= X::ACT) return;
  // lane = a * G + g: the lanes that own the same column of the warp's G trajectories are adjacent, so that the
  // owner's shared-memory stores of an elimination step fall into one quarter-warp (one wavefront instead of G)
  const int a = lane / X::G, g = lane - a * X::G, gbase = g;
  unsigned gmask = 0u;
#pragma unroll
  for (int i = 0; i < F; i++) gmask |= 1u << (i * X::G + g);
  double *ws = smem + X::NCOEFP + (warp * X::G + g) * X::WS;
  double *qs = ws, *Hs = ws + X::FP;
  double2 *red = reinterpret_cast<double2 *>(ws + X::FP + X::NHP);

  const long long jj = (long long)blockIdx.x * (kThreads / 32 * X::G) + warp * X::G + g;
  const bool valid = jj < P.nb;
  const long long jl = valid ? jj : P.nb - 1;  // tail groups recompute the last trajectory and store nothing
  const long long jg = P.j0 + jl;

  int fwd[X::ND], bwd[X::ND];
#pragma unroll
  for (int d = 0; d < X::ND; d++) {
    fwd[d] = (a + d) % F;
    bwd[d] = (a - d + F) % F;
  }
  const double sg_a = P.sg[a], isg_a = P.isg[a], mu_a = P.mu[a];
  const double Peq_a = P.Peq[a], Qeq_a = P.Qeq[a];

  double Pm = P.p0q0[(long long)a * P.stride + jg] * isg_a;
  double Q = P.p0q0[(long long)(F + a) * P.stride + jg] * sg_a;
  double Sa = 0.0;
  double dP1[F], dQ1[F], dP2[F], dQ2[F], HM1[F], HM2[F];
#pragma unroll
  for (int i = 0; i < F; i++) {
    dP1[i] = (i == a) ? 1.0 : 0.0;
    dQ1[i] = 0.0;
    dP2[i] = 0.0;
    dQ2[i] = (i == a) ? 1.0 : 0.0;
  }
  double gq, Va, Hent[X::ND];
  pes_group<F, KIND>(cs, qs, Hs, a, gbase, fwd, bwd, Q, gq, Va, Hent);
  __syncwarp(X::AMASK);
  hessian_times_tangent<F, KIND>(Hs, dQ1, dQ2, HM1, HM2);

  double2 *kb = reinterpret_cast<double2 *>(ws + X::FP + X::NHP + 2 * F);
  double *mb = ws + X::FP + X::NHP + 2 * F + 2 * X::KB;

  bool good = true;
  bool dirty = false;
  int det_count = 0;  // steps until the next check
  const int nsteps = P.nsteps;
#pragma unroll 1
  for (int c = 0;; c++) {
    const bool last = (c == nsteps);
    const bool check = (det_count == 0) || last;  // warp-uniform
    // a6 (Eq. 3): per-mode share of ln<chi|pq> and of the phase S + arg<chi|pq>, at the integer time c
    double oa = 0.0, ob = 0.0;
    if (P.raw != nullptr) {
      const double dq = Qeq_a - Q, dp = Peq_a - Pm;
      oa = -0.25 * fma(dq, dq, dp * dp);
      ob = fma(0.5 * (Peq_a + Pm), dq, Sa);
      if (P.raw_plain) {  // several reference states: the record carries S alone, (P, Q) of the step go out beside it
        oa = 0.0;
        ob = Sa;
      }
      if (P.pq_steps != nullptr && valid) P.pq_steps[((long long)c * F + a) * P.raw_stride + jj] = make_double2(Pm, Q);
      if (F > 1) red[a] = make_double2(oa, ob);
    }
    // working copies for the two eliminations: column a of 2K (a5; Eq. 5, R2) and columns a, F+a of M (a7)
    double Are[F], Aim[F], C1[2 * F], C2[2 * F];
#pragma unroll
    for (int i = 0; i < F; i++) {
      Are[i] = dQ2[i] + dP1[i];
      Aim[i] = dP2[i] - dQ1[i];
      C1[i] = dP1[i];
      C1[F + i] = dQ1[i];
      C2[i] = dP2[i];
      C2[F + i] = dQ2[i];
    }
    // opening kick of the next step (stage 0), applied now so that H dQ is dead during the eliminations
    const double bdt0 = last ? 0.0 : P.kick[0];
    Sa = fma(-bdt0, Va, Sa);
    Pm = fma(-bdt0, gq, Pm);
#pragma unroll
    for (int i = 0; i < F; i++) {
      dP1[i] = fma(-bdt0, HM1[i], dP1[i]);
      dP2[i] = fma(-bdt0, HM2[i], dP2[i]);
    }
    double Dre, Dim, dM;
    unsigned growK, growM;
    if (check) lu_static<F, true>(Are, Aim, C1, C2, kb, mb, a, X::AMASK, Dre, Dim, dM, growK, growM);
    else lu_static<F, false>(Are, Aim, C1, C2, kb, mb, a, X::AMASK, Dre, Dim, dM, growK, growM);
    {
      // static order not safe for this matrix (or forced by the caller): repeat with the pivoted eliminations
      const bool risky = (growK >= P.grow_k_max) || (check && growM >= P.grow_m_max);
      const unsigned rb = __ballot_sync(X::AMASK, risky);
      if (rb != 0u) {
        double buf[4 * F];
#pragma unroll
        for (int i = 0; i < F; i++) {
          buf[i] = dP1[i];
          buf[F + i] = dQ1[i];
          buf[2 * F + i] = dP2[i];
          buf[3 * F + i] = dQ2[i];
        }
        double fDre, fDim, fdM;
        pivoted_dets<F, KIND>(buf, Hs, bdt0, gbase, a, gmask, check, fDre, fDim, fdM);
        if ((rb & gmask) != 0u) {
          Dre = fDre;
          Dim = fDim;
          dM = fdM;
          if (P.fb_count != nullptr && a == 0 && valid) atomicAdd(P.fb_count, 1ULL);  // statistics only
        }
      }
    }
    // a8 input record, written by the lane that holds the last pivots
    if (P.raw != nullptr) {
      if (F > 1) {
        if (a == F - 1) {
          double s0 = 0.0, s1 = 0.0;
#pragma unroll
          for (int i = 0; i < F; i++) {
            const double2 v = red[i];
            s0 += v.x;
            s1 += v.y;
          }
          if (valid) P.raw[(long long)c * P.raw_stride + jj] = make_double4(s0, s1, Dre, Dim);
        }
      } else {
        if (valid) P.raw[(long long)c * P.raw_stride + jj] = make_double4(oa, ob, Dre, Dim);
      }
    }
    // a7: |det M - 1| <= tol and finite, every det_stride steps and at the end
    if (check) {
      const bool okd = (a == F - 1) ? (fabs(dM - 1.0) <= P.det_tol) : true;
      good = good && okd && isfinite(Sa) && isfinite(Pm) && isfinite(Q);
      det_count = P.det_stride;
    }
    det_count--;
    if (last) break;
    // a2-a4 (R10, R11): stages "kick b_s then drift a_s"; stage 0's kick is already in; the PES is re-evaluated
    // only after q moved
#pragma unroll 1
    for (int st = 0; st < P.nstages; st++) {
      if (st > 0) {
        if (dirty) {
          pes_group<F, KIND>(cs, qs, Hs, a, gbase, fwd, bwd, Q, gq, Va, Hent);
          __syncwarp(X::AMASK);
          hessian_times_tangent<F, KIND>(Hs, dQ1, dQ2, HM1, HM2);
          dirty = false;
        }
        const double bdt = P.kick[st];
        Sa = fma(-bdt, Va, Sa);
        Pm = fma(-bdt, gq, Pm);
#pragma unroll
        for (int i = 0; i < F; i++) {
          dP1[i] = fma(-bdt, HM1[i], dP1[i]);
          dP2[i] = fma(-bdt, HM2[i], dP2[i]);
        }
      }
      const double adt = P.drift[st];
      if (adt != 0.0) {
        Sa = fma(0.5 * adt * mu_a, Pm * Pm, Sa);
        Q = fma(adt * mu_a, Pm, Q);
#pragma unroll
        for (int i = 0; i < F; i++) {
          const double am = adt * P.mu[i];
          dQ1[i] = fma(am, dP1[i], dQ1[i]);
          dQ2[i] = fma(am, dP2[i], dQ2[i]);
        }
        dirty = true;
      }
    }
    if (dirty) {  // schemes whose last drift is non-zero: the next step's opening kick needs the PES at the new q
      pes_group<F, KIND>(cs, qs, Hs, a, gbase, fwd, bwd, Q, gq, Va, Hent);
      __syncwarp(X::AMASK);
      hessian_times_tangent<F, KIND>(Hs, dQ1, dQ2, HM1, HM2);
      dirty = false;
    }
  }

  // outputs
  const unsigned bal = __ballot_sync(X::AMASK, good);
  const bool group_good = ((bal & gmask) == gmask);
  double Stot = Sa;
  if (F > 1) {
    Stot = 0.0;
#pragma unroll
    for (int i = 0; i < F; i++) Stot += __shfl_sync(X::AMASK, Sa, i * X::G + gbase);
  }
  if (!valid) return;
  if (P.good != nullptr && a == 0) P.good[jj] = group_good ? 1 : 0;
  if (P.S_out != nullptr && a == 0) P.S_out[jg] = Stot;
  if (P.pq_out != nullptr) {
    P.pq_out[(long long)a * P.stride + jg] = Pm * sg_a;
    P.pq_out[(long long)(F + a) * P.stride + jg] = Q * isg_a;
  }
  if (P.M_out != nullptr) {
    // M_xy[i][a], reduced -> caller's units: p = sg P, q = Q / sg
#pragma unroll
    for (int i = 0; i < F; i++) {
      const double si = P.sg[i], ii = P.isg[i];
      const long long e = ((long long)i * F + a) * P.stride + jg;
      const long long blk = (long long)F * F * P.stride;
      P.M_out[0 * blk + e] = dP1[i] * si * isg_a;
      P.M_out[1 * blk + e] = dP2[i] * si * sg_a;
      P.M_out[2 * blk + e] = dQ1[i] * ii * isg_a;
      P.M_out[3 * blk + e] = dQ2[i] * ii * sg_a;
    }
  }
}

// ---- debug kernel for a1: same pes_group, caller's units out -----------------------------------------------
template <int F, int KIND>
__global__ void __launch_bounds__(kThreads) k_eval_pes(const double *__restrict__ coef, const double *__restrict__ sgv,
                                                       const double *__restrict__ q, long long n, double *V, double *gout,
                                                       double *H) {
  using X = Geo<F>;
  extern __shared__ double smem[];
  double *cs = smem;
  {
    const int nco = (KIND == SC_IVR_PES_QFF) ? X::NCOEF_QFF : X::NCOEF_MORSE;
    for (int i = threadIdx.x; i < nco; i += kThreads) cs[i] = coef[i];
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane >= X::ACT) return;
  const int a = lane / X::G, g = lane - a * X::G, gbase = g;
  double *ws = smem + X::NCOEFP + (warp * X::G + g) * X::WS;
  double *qs = ws, *Hs = ws + X::FP;
  const long long jj = (long long)blockIdx.x * (kThreads / 32 * X::G) + warp * X::G + g;
  const bool valid = jj < n;
  const long long jl = valid ? jj : n - 1;
  int fwd[X::ND], bwd[X::ND];
#pragma unroll
  for (int d = 0; d < X::ND; d++) {
    fwd[d] = (a + d) % F;
    bwd[d] = (a - d + F) % F;
  }
  const double sg_a = sgv[a];
  const double Q = q[(long long)a * n + jl] * sg_a;
  double gq, Va, Hent[X::ND];
  pes_group<F, KIND>(cs, qs, Hs, a, gbase, fwd, bwd, Q, gq, Va, Hent);
  double Vt = 0.0;
#pragma unroll
  for (int i = 0; i < F; i++) Vt += __shfl_sync(X::AMASK, Va, i * X::G + gbase);
  if (!valid) return;
  if (a == 0) V[jl] = Vt;
  gout[(long long)a * n + jl] = gq * sg_a;
  if (KIND != SC_IVR_PES_QFF) {
    for (int b = 0; b < F; b++) H[((long long)a * F + b) * n + jl] = (b == a) ? Hent[0] * sg_a * sg_a : 0.0;
  } else {
#pragma unroll
    for (int d = 0; d < X::ND; d++) {
      const int b = fwd[d];
      const double h = Hent[d] * sg_a * sgv[b];
      H[((long long)a * F + b) * n + jl] = h;
      H[((long long)b * F + a) * n + jl] = h;
    }
  }
}

template <int F>
size_t smem_bytes() {
  return sizeof(double) * (Geo<F>::NCOEFP + (kThreads / 32) * Geo<F>::G * Geo<F>::WS);
}

template <int F, int KIND>
cudaError_t launch_prop(const PropParams &P, cudaStream_t st) {
  const int tpb = (kThreads / 32) * Geo<F>::G;
  const long long blocks = (P.nb + tpb - 1) / tpb;
  k_propagate<F, KIND><<<(unsigned)blocks, kThreads, smem_bytes<F>(), st>>>(P);
  return cudaGetLastError();
}

template <int F, int KIND>
cudaError_t launch_pes(const double *coef, const double *sg, const double *q, long long n, double *V, double *g, double *H,
                       cudaStream_t st) {
  const int tpb = (kThreads / 32) * Geo<F>::G;
  const long long blocks = (n + tpb - 1) / tpb;
  k_eval_pes<F, KIND><<<(unsigned)blocks, kThreads, smem_bytes<F>(), st>>>(coef, sg, q, n, V, g, H);
  return cudaGetLastError();
}

template <int F, int KIND>
int occupancy() {
  int nb = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_propagate<F, KIND>, kThreads, smem_bytes<F>()) != cudaSuccess) nb = 1;
  return nb < 1 ? 1 : nb;
}

}  // namespace

// F <= SCI_TPT_MAXF is served by the thread-per-trajectory kernels (propagate_tpt.cu)
#define SCI_FOR_EACH_F(X) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12)

int sci_prop_traj_per_block(int F) { return (kThreads / 32) * (32 / F); }

int sci_prop_blocks_per_sm(int F, int kind) {
  const bool qff = kind == SC_IVR_PES_QFF;
  switch (F) {
#define X(f) case f: return qff ? occupancy<f, SC_IVR_PES_QFF>() : occupancy<f, SC_IVR_PES_MORSE_UNCOUPLED>();
    SCI_FOR_EACH_F(X)
#undef X
  }
  return 1;
}

cudaError_t sci_launch_propagate(int F, int kind, const PropParams &P, cudaStream_t st) {
  const bool qff = kind == SC_IVR_PES_QFF;
  switch (F) {
#define X(f) case f: return qff ? launch_prop<f, SC_IVR_PES_QFF>(P, st) : launch_prop<f, SC_IVR_PES_MORSE_UNCOUPLED>(P, st);
    SCI_FOR_EACH_F(X)
#undef X
  }
  return cudaErrorInvalidValue;
}

cudaError_t sci_launch_eval_pes(int F, int kind, const double *coef, const double *sg, const double *q, long long n,
                                double *V, double *g, double *H, cudaStream_t st) {
  const bool qff = kind == SC_IVR_PES_QFF;
  switch (F) {
#define X(f) case f: return qff ? launch_pes<f, SC_IVR_PES_QFF>(coef, sg, q, n, V, g, H, st) \
                                : launch_pes<f, SC_IVR_PES_MORSE_UNCOUPLED>(coef, sg, q, n, V, g, H, st);
    SCI_FOR_EACH_F(X)
#undef X
  }
  return cudaErrorInvalidValue;
}

// Host: reduce the caller's coefficients to the kernel's packed block (layout in Geo<F>).
//   Phi~_ijk = Phi_ijk / sqrt(g_i g_j g_k),  P~_ij = Phi_iijj / (g_i g_j),  w~_a^2 = w_a^2 / g_a   (QFF)
//   a~ = a / sqrt(g),  Q_e = sqrt(g) q_e                                                           (Morse)
size_t sci_pack_coeffs(int F, int kind, const double *c, const double *gamma, double *out) {
  const int ND = F / 2 + 1;
  if (kind != SC_IVR_PES_QFF) {
    const size_t n = 3 * (size_t)F;
    if (!out) return n;
    for (int a = 0; a < F; a++) {
      const double sg = sqrt(gamma[a]);
      out[a] = c[4 * a];
      out[F + a] = c[4 * a + 1] / sg;
      out[2 * F + a] = c[4 * a + 2] * sg;
    }
    return n;
  }
  const int L_C3 = 0, L_C4U = L_C3 + ND * F, L_C4D = L_C4U + F, L_W2 = L_C4D + ND, LA = L_W2 + 1, LAP = (LA + 1) & ~1;
  const size_t n = (size_t)LAP * F;
  if (!out) return n;
  // unpack the symmetric tensors
  double *phi = new double[(size_t)F * F * F];
  double *pq = new double[(size_t)F * F];
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
  double *list = new double[LAP];
  for (int a = 0; a < F; a++) {
    for (int i = 0; i < LAP; i++) list[i] = 0.0;
    for (int d = 0; d < ND; d++)
      for (int k = 0; k < F; k++) list[L_C3 + d * F + k] = phi[((size_t)a * F + (a + d) % F) * F + k];
    for (int j = 0; j < F; j++) list[L_C4U + j] = pq[a * F + j];
    for (int d = 0; d < ND; d++) list[L_C4D + d] = pq[a * F + (a + d) % F];
    list[L_W2] = c[a] * c[a] / gamma[a];
    for (int i = 0; i < LAP; i++) out[((size_t)(i / 2) * F + a) * 2 + (i & 1)] = list[i];
  }
  delete[] list;
  delete[] phi;
  delete[] pq;
  return n;
}
