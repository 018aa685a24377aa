/*
 * CPU FP64 ORACLE for the TA-SC-IVR hot path (arxiv 1312.4698).  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code with the CUDA path
 * (paper_1312_4698_b200/csrc): no common header, helper, table or constant.
 *
 * The method is an approximation chain (SC-IVR -> Herman-Kluk -> time averaging -> separable
 * prefactor -> Monte Carlo -> time discretisation), so this file follows the algorithm step by
 * step in the paper's order and notation, one plain loop nest per formula:
 *
 *   Eq. 11      I(E_i) = norm * sum_j w_j | sum_c <chi|p_j q_j> e^{i(S + E_i c dt + phi)} |^2
 *   Eq. 10    what Eq. 11 discretises
 *   Eq. 5       Herman-Kluk prefactor C_t = sqrt(det K), K from the monodromy blocks
 *   Eq. 3    coherent states; their closed-form overlap <chi|p q>
 *   PAPER.md:64                 monodromy matrix M = d(p_t,q_t)/d(p_0,q_0), rejection |det M - 1| > 1e-6
 *   PAPER.md:86                 phi(t) = phase[C_t], separable approximation (continuous branch)
 *   PAPER.md:109                symplectic integrator, n_good
 *   PAPER.md:117, :135          only trajectories that completed contribute
 *
 * Readings of the paper where it is silent or garbled are DESIGN.md R1..R21 (cited inline).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P0..P12 of DESIGN.md.  Parity unpinned: the
 * absolute normalisation constant of I(E) (R4) - immaterial, parity is relative to max(I).
 *
 * Layouts (same as include/sc_ivr.h so the same seeded inputs serve both sides):
 *   p0q0   [2F][ntraj]  rows 0..F-1 = p_k, rows F..2F-1 = q_k
 *   chi    [2F]         p_eq[F] then q_eq[F]
 *   M_out  [4][F][F][ntraj] blocks pp, pq, qp, qq;  M_xy[a][b] = d x_a(t) / d y_b(0)
 *   z_out  [ntraj][nsteps+1][2]  (re, im)
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define SCO_MAXF 16
#define SCO_OK 0
#define SCO_EINVAL 1
#define SCO_ENOMEM 2
#define SCO_ENOGOOD 5

enum { PES_MORSE1D = 0, PES_QFF = 1, PES_MORSE_UNCOUPLED = 2 };

typedef struct {
  int F, kind;
  double mass[SCO_MAXF];
  /* QFF (mass-weighted normal coordinates, m = 1) */
  double omega[SCO_MAXF];
  double phi3[SCO_MAXF][SCO_MAXF][SCO_MAXF]; /* fully symmetric cubic tensor Phi_ijk */
  double P[SCO_MAXF][SCO_MAXF];              /* P_ij = Phi_iijj (symmetric), P_ii = Phi_iiii */
  /* Morse, per mode */
  double mD[SCO_MAXF], ma[SCO_MAXF], mqe[SCO_MAXF];
} pes_t;

static long n_coeffs_expected(int F, int kind) {
  if (kind == PES_MORSE1D) return 4;
  if (kind == PES_QFF) return F + (long)F * (F + 1) * (F + 2) / 6 + (long)F * (F + 1) / 2;
  if (kind == PES_MORSE_UNCOUPLED) return 4L * F;
  return -1;
}

/* Unpack the coefficient block (layout: include/sc_ivr.h "pes_coeffs layouts"). */
static int pes_init(pes_t *P, int F, int kind, const double *c, long nc) {
  if (F < 1 || F > SCO_MAXF) return SCO_EINVAL;
  if (nc != n_coeffs_expected(F, kind)) return SCO_EINVAL;
  if (kind == PES_MORSE1D && F != 1) return SCO_EINVAL;
  memset(P, 0, sizeof(*P));
  P->F = F;
  P->kind = kind;
  if (kind == PES_MORSE1D) {
    P->mD[0] = c[0]; P->ma[0] = c[1]; P->mqe[0] = c[2]; P->mass[0] = c[3];
  } else if (kind == PES_MORSE_UNCOUPLED) {
    for (int k = 0; k < F; k++) {
      P->mD[k] = c[4 * k]; P->ma[k] = c[4 * k + 1]; P->mqe[k] = c[4 * k + 2]; P->mass[k] = c[4 * k + 3];
    }
  } else {
    for (int k = 0; k < F; k++) { P->omega[k] = c[k]; P->mass[k] = 1.0; }
    const double *cub = c + F;
    long n = 0;
    for (int i = 0; i < F; i++)
      for (int j = i; j < F; j++)
        for (int k = j; k < F; k++) {
          double v = cub[n++];
          P->phi3[i][j][k] = P->phi3[i][k][j] = P->phi3[j][i][k] = v;
          P->phi3[j][k][i] = P->phi3[k][i][j] = P->phi3[k][j][i] = v;
        }
    const double *qua = cub + n;
    n = 0;
    for (int i = 0; i < F; i++)
      for (int j = i; j < F; j++) {
        double v = qua[n++];
        P->P[i][j] = P->P[j][i] = v;
      }
  }
  return SCO_OK;
}

/*
 * a1. Potential, gradient, Hessian at q.
 * Morse: V = D (1 - y)^2, y = exp(-a (q - q_e)).
 * QFF (BASELINE.json configs 2-4, stand-in for the fitted surfaces of PAPER.md:157):
 *   V = 1/2 sum w_i^2 q_i^2 + 1/6 sum_ijk Phi_ijk q_i q_j q_k + 1/24 sum_ijkl Phi_ijkl q_i q_j q_k q_l
 * with UNRESTRICTED sums, Phi fully symmetric, and the only non-zero quartic entries those whose
 * indices form two pairs (Phi_iijj and permutations).  The cubic part is the unrestricted sum
 * written out; the quartic part is the unrestricted sum collected by pairs:
 *   1/24 sum_ijkl = 1/24 sum_i P_ii q_i^4 + 1/4 sum_{i<j} P_ij q_i^2 q_j^2
 * (six arrangements of (i,i,j,j) for i != j, one for i == j).
 * H is returned full, row-major [F][F].
 */
static void pes_eval(const pes_t *P, const double *q, double *V, double *g, double *H) {
  const int F = P->F;
  if (P->kind == PES_MORSE1D || P->kind == PES_MORSE_UNCOUPLED) {
    double v = 0.0;
    for (int a = 0; a < F; a++)
      for (int b = 0; b < F; b++) H[a * F + b] = 0.0;
    for (int k = 0; k < F; k++) {
      double D = P->mD[k], a = P->ma[k];
      double y = exp(-a * (q[k] - P->mqe[k]));
      v += D * (1.0 - y) * (1.0 - y);
      g[k] = 2.0 * D * a * y * (1.0 - y);
      H[k * F + k] = 2.0 * D * a * a * y * (2.0 * y - 1.0);
    }
    *V = v;
    return;
  }
  double v2 = 0.0, v3 = 0.0, v4 = 0.0;
  for (int i = 0; i < F; i++) v2 += 0.5 * P->omega[i] * P->omega[i] * q[i] * q[i];
  for (int i = 0; i < F; i++)
    for (int j = 0; j < F; j++)
      for (int k = 0; k < F; k++) v3 += P->phi3[i][j][k] * q[i] * q[j] * q[k];
  v3 /= 6.0;
  for (int i = 0; i < F; i++) {
    v4 += P->P[i][i] * q[i] * q[i] * q[i] * q[i] / 24.0;
    for (int j = i + 1; j < F; j++) v4 += 0.25 * P->P[i][j] * q[i] * q[i] * q[j] * q[j];
  }
  *V = v2 + v3 + v4;
  for (int a = 0; a < F; a++) {
    /* dV/dq_a = w_a^2 q_a + 1/2 sum_jk Phi_ajk q_j q_k + [1/6 P_aa q_a^3 + 1/2 q_a sum_{j!=a} P_aj q_j^2] */
    double s3 = 0.0, s4 = 0.0;
    for (int j = 0; j < F; j++)
      for (int k = 0; k < F; k++) s3 += P->phi3[a][j][k] * q[j] * q[k];
    for (int j = 0; j < F; j++)
      if (j != a) s4 += P->P[a][j] * q[j] * q[j];
    g[a] = P->omega[a] * P->omega[a] * q[a] + 0.5 * s3 + P->P[a][a] * q[a] * q[a] * q[a] / 6.0 + 0.5 * q[a] * s4;
    for (int b = 0; b < F; b++) {
      /* d2V/dq_a dq_b = w_a^2 delta_ab + sum_k Phi_abk q_k + quartic */
      double h = 0.0;
      for (int k = 0; k < F; k++) h += P->phi3[a][b][k] * q[k];
      if (a == b) h += P->omega[a] * P->omega[a] + 0.5 * P->P[a][a] * q[a] * q[a] + 0.5 * s4;
      else h += P->P[a][b] * q[a] * q[b];
      H[a * F + b] = h;
    }
  }
}

/* Integrator = composition of stages "kick b_i, then drift a_i" (R10).  Velocity-Verlet is
 * (1/2, 1), (1/2, 0).  The 4-stage 4th-order table (NEXT f2) is McLachlan-Atela's. */
typedef struct { int n; double b[4], a[4]; } scheme_t;

static int scheme_init(scheme_t *s, int integrator) {
  if (integrator == 0) {
    s->n = 2; s->b[0] = 0.5; s->a[0] = 1.0; s->b[1] = 0.5; s->a[1] = 0.0;
    return SCO_OK;
  }
  if (integrator == 1) {
    s->n = 4;
    s->b[0] = 0.1344961992774310892;  s->a[0] = 0.5153528374311229364;
    s->b[1] = -0.2248198030794208058; s->a[1] = -0.085782019412973646;
    s->b[2] = 0.7563200005156682911;  s->a[2] = 0.4415830236164665242;
    s->b[3] = 0.3340036032863214255;  s->a[3] = 0.1288461583653841854;
    return SCO_OK;
  }
  return SCO_EINVAL;
}

typedef struct {
  int F;
  double p[SCO_MAXF], q[SCO_MAXF], S;
  double Mpp[SCO_MAXF * SCO_MAXF], Mpq[SCO_MAXF * SCO_MAXF], Mqp[SCO_MAXF * SCO_MAXF], Mqq[SCO_MAXF * SCO_MAXF];
} state_t;

/* a2 + a3 + a4 (step vi of DESIGN.md "Algorithm"): one time step of (p, q, S, M).
 * kick  b: S -= b dt V(q);        p -= b dt g(q);     M_pp -= b dt H M_qp;  M_pq -= b dt H M_qq
 * drift a: S += a dt 1/2 p^T p/m; q += a dt p/m;      M_qp += a dt M_pp/m;  M_qq += a dt M_pq/m
 * (R11: each sub-flow contributes its exact action.)  The PES is evaluated afresh before
 * every kick: nothing is cached, so the step is the composition as written. */
static void step(const pes_t *P, const scheme_t *sc, double dt, state_t *s) {
  const int F = s->F;
  double V, g[SCO_MAXF], H[SCO_MAXF * SCO_MAXF], T1[SCO_MAXF * SCO_MAXF], T2[SCO_MAXF * SCO_MAXF];
  for (int st = 0; st < sc->n; st++) {
    const double b = sc->b[st], a = sc->a[st];
    if (b != 0.0) {
      pes_eval(P, s->q, &V, g, H);
      s->S -= b * dt * V;
      for (int k = 0; k < F; k++) s->p[k] -= b * dt * g[k];
      for (int i = 0; i < F; i++)
        for (int j = 0; j < F; j++) {
          double t1 = 0.0, t2 = 0.0;
          for (int l = 0; l < F; l++) { t1 += H[i * F + l] * s->Mqp[l * F + j]; t2 += H[i * F + l] * s->Mqq[l * F + j]; }
          T1[i * F + j] = t1; T2[i * F + j] = t2;
        }
      for (int i = 0; i < F * F; i++) { s->Mpp[i] -= b * dt * T1[i]; s->Mpq[i] -= b * dt * T2[i]; }
    }
    if (a != 0.0) {
      double ke = 0.0;
      for (int k = 0; k < F; k++) ke += 0.5 * s->p[k] * s->p[k] / P->mass[k];
      s->S += a * dt * ke;
      for (int k = 0; k < F; k++) s->q[k] += a * dt * s->p[k] / P->mass[k];
      for (int i = 0; i < F; i++)
        for (int j = 0; j < F; j++) {
          s->Mqp[i * F + j] += a * dt * s->Mpp[i * F + j] / P->mass[i];
          s->Mqq[i * F + j] += a * dt * s->Mpq[i * F + j] / P->mass[i];
        }
    }
  }
}

/* Determinant of an n x n complex matrix by LU with partial pivoting (max modulus). A is destroyed. */
static double complex cdet(double complex *A, int n) {
  double complex det = 1.0;
  for (int k = 0; k < n; k++) {
    int piv = k;
    double best = cabs(A[k * n + k]);
    for (int i = k + 1; i < n; i++) {
      double m = cabs(A[i * n + k]);
      if (m > best) { best = m; piv = i; }
    }
    if (best == 0.0) return 0.0;
    if (piv != k) {
      for (int j = 0; j < n; j++) { double complex t = A[k * n + j]; A[k * n + j] = A[piv * n + j]; A[piv * n + j] = t; }
      det = -det;
    }
    det *= A[k * n + k];
    for (int i = k + 1; i < n; i++) {
      double complex l = A[i * n + k] / A[k * n + k];
      for (int j = k + 1; j < n; j++) A[i * n + j] -= l * A[k * n + j];
    }
  }
  return det;
}

/* Determinant of an n x n real matrix, same algorithm. A is destroyed. */
static double rdet(double *A, int n) {
  double det = 1.0;
  for (int k = 0; k < n; k++) {
    int piv = k;
    double best = fabs(A[k * n + k]);
    for (int i = k + 1; i < n; i++) {
      double m = fabs(A[i * n + k]);
      if (m > best) { best = m; piv = i; }
    }
    if (!(best > 0.0)) return (best == 0.0) ? 0.0 : NAN;
    if (piv != k) {
      for (int j = 0; j < n; j++) { double t = A[k * n + j]; A[k * n + j] = A[piv * n + j]; A[piv * n + j] = t; }
      det = -det;
    }
    det *= A[k * n + k];
    for (int i = k + 1; i < n; i++) {
      double l = A[i * n + k] / A[k * n + k];
      for (int j = k + 1; j < n; j++) A[i * n + j] -= l * A[k * n + j];
    }
  }
  return det;
}

/* a5, step i: Herman-Kluk matrix (Eq. 5, read as R2):
 * K_ab = 1/2 [ M_qq,ab + (g_b/g_a) M_pp,ab ] + (i/2) [ M_pq,ab / g_a - g_b M_qp,ab ],  det K_0 = 1. */
static double complex hk_det(const state_t *s, const double *gamma) {
  const int F = s->F;
  double complex K[SCO_MAXF * SCO_MAXF];
  for (int a = 0; a < F; a++)
    for (int b = 0; b < F; b++) {
      double re = 0.5 * (s->Mqq[a * F + b] + gamma[b] / gamma[a] * s->Mpp[a * F + b]);
      double im = 0.5 * (s->Mpq[a * F + b] / gamma[a] - gamma[b] * s->Mqp[a * F + b]);
      K[a * F + b] = re + I * im;
    }
  return cdet(K, F);
}

/* a7: det of the 2F x 2F monodromy matrix [[M_pp, M_pq], [M_qp, M_qq]] ((p,q) order). */
static double monodromy_det(const state_t *s) {
  const int F = s->F, n = 2 * F;
  double A[4 * SCO_MAXF * SCO_MAXF];
  for (int a = 0; a < F; a++)
    for (int b = 0; b < F; b++) {
      A[a * n + b] = s->Mpp[a * F + b];
      A[a * n + F + b] = s->Mpq[a * F + b];
      A[(F + a) * n + b] = s->Mqp[a * F + b];
      A[(F + a) * n + F + b] = s->Mqq[a * F + b];
    }
  return rdet(A, n);
}

static int state_finite(const state_t *s) {
  const int F = s->F;
  if (!isfinite(s->S)) return 0;
  for (int k = 0; k < F; k++) if (!isfinite(s->p[k]) || !isfinite(s->q[k])) return 0;
  for (int i = 0; i < F * F; i++)
    if (!isfinite(s->Mpp[i]) || !isfinite(s->Mpq[i]) || !isfinite(s->Mqp[i]) || !isfinite(s->Mqq[i])) return 0;
  return 1;
}

/* a6: <chi | p q> for chi = |p_eq, q_eq> (Eq. 3; chi: PAPER.md:80), ln of it:
 * a = sum_k [ -g_k/4 (q_eq,k - q_k)^2 - (p_eq,k - p_k)^2 / (4 g_k) ],  b = 1/2 sum_k (p_eq,k + p_k)(q_eq,k - q_k). */
static double complex overlap(const state_t *s, const double *gamma, const double *chi) {
  const int F = s->F;
  double a = 0.0, b = 0.0;
  for (int k = 0; k < F; k++) {
    double dq = chi[F + k] - s->q[k], dp = chi[k] - s->p[k];
    a += -0.25 * gamma[k] * dq * dq - dp * dp / (4.0 * gamma[k]);
    b += 0.5 * (chi[k] + s->p[k]) * dq;
  }
  return exp(a) * cexp(I * b);
}

/* Reference state as a combination of coherent states, |chi> = sum_m eps_m |p_m, q_m>  (Fig. 4: "different
 * coherent state combinations for the same irreducible representation"):  <chi|p q> = sum_m conj(eps_m) <p_m q_m|p q>.
 * chi: [ncs][2F], eps: [ncs][2] (re, im); eps == NULL is the single coherent state chi[0] of PAPER.md:80. */
static double complex reference_overlap(const state_t *s, const double *gamma, const double *chi, int ncs, const double *eps) {
  if (!eps) return overlap(s, gamma, chi);
  double complex sum = 0.0;
  for (int m = 0; m < ncs; m++)
    sum += (eps[2 * m] - I * eps[2 * m + 1]) * overlap(s, gamma, chi + 2 * (size_t)s->F * m);
  return sum;
}

static double wrap_pi(double x) { /* to (-pi, pi] */
  while (x > M_PI) x -= 2.0 * M_PI;
  while (x <= -M_PI) x += 2.0 * M_PI;
  return x;
}

/*
 * One trajectory, steps i..vi of DESIGN.md "Algorithm" for c = 0..nsteps:
 *   i.   K from M                      (hk_det)
 *   ii.  D = det K; u^ = principal sqrt(D/|D|); if Re(u^ conj(u)) < 0 then u^ = -u^; u = u^   (R6)
 *        and, in parallel, the equivalent unwrapped angle theta_c = theta_{c-1} + wrap(arg D_c - arg D_{c-1})
 *   iii. overlap;  iv. z_c = <chi|p q> e^{i S} u;  v. quality flag;  vi. time step.
 * z (may be NULL): [nsteps+1][2].  Returns good flag.
 */
static int propagate_one(const pes_t *P, const scheme_t *sc, const double *gamma, const double *chi, int ncs, const double *eps,
                         double dt, int nsteps, int det_stride, double det_tol,
                         const double *p0, const double *q0, double *z, state_t *final, double *theta_out) {
  const int F = P->F;
  state_t s;
  memset(&s, 0, sizeof(s));
  s.F = F;
  for (int k = 0; k < F; k++) { s.p[k] = p0[k]; s.q[k] = q0[k]; }
  for (int k = 0; k < F; k++) { s.Mpp[k * F + k] = 1.0; s.Mqq[k * F + k] = 1.0; }
  s.S = 0.0;
  double complex u = 1.0;
  double theta = 0.0, argD_prev = 0.0;
  int good = 1;
  for (int c = 0; c <= nsteps; c++) {
    double complex D = hk_det(&s, gamma);
    double complex un = csqrt(D / cabs(D));
    if (creal(un * conj(u)) < 0.0) un = -un;
    u = un;
    double argD = carg(D);
    theta += wrap_pi(argD - argD_prev);
    argD_prev = argD;
    if (z) {
      double complex zc = reference_overlap(&s, gamma, chi, ncs, eps) * cexp(I * s.S) * u;
      z[2 * c] = creal(zc);
      z[2 * c + 1] = cimag(zc);
    }
    if (c % det_stride == 0 || c == nsteps) {
      int ok = state_finite(&s);
      if (ok) {
        double dM = monodromy_det(&s);
        ok = isfinite(dM) && fabs(dM - 1.0) <= det_tol;
      }
      good = good && ok;
    }
    if (c < nsteps) step(P, sc, dt, &s);
  }
  if (final) *final = s;
  if (theta_out) *theta_out = theta;
  return good;
}

/* ---------------------------------------------------------------- C ABI (host pointers only) */

int sc_ivr_oracle_max_f(void) { return SCO_MAXF; }

int sc_ivr_oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* V[n], g[F][n], H[F][F][n] at q[F][n]. */
int sc_ivr_oracle_eval_pes(int F, int kind, const double *coeffs, long ncoef, const double *q, long n,
                           double *V, double *g, double *H) {
  pes_t P;
  int rc = pes_init(&P, F, kind, coeffs, ncoef);
  if (rc) return rc;
  for (long j = 0; j < n; j++) {
    double qq[SCO_MAXF], gg[SCO_MAXF], HH[SCO_MAXF * SCO_MAXF], v;
    for (int k = 0; k < F; k++) qq[k] = q[k * n + j];
    pes_eval(&P, qq, &v, gg, HH);
    V[j] = v;
    for (int k = 0; k < F; k++) g[k * n + j] = gg[k];
    for (int a = 0; a < F * F; a++) H[a * n + j] = HH[a];
  }
  return SCO_OK;
}

/*
 * Propagate ntraj trajectories for nsteps steps.  Any output pointer may be NULL.
 *   pq_out [2F][ntraj], S_out [ntraj], M_out [4][F][F][ntraj], theta_out [ntraj] (unwrapped arg det K = 2 phi),
 *   good_out [ntraj] (bytes), z_out [ntraj][nsteps+1][2].
 */
int sc_ivr_oracle_propagate(int F, int kind, const double *coeffs, long ncoef, const double *gamma, double dt,
                            int nsteps, int integrator, int det_stride, double det_tol, const double *p0q0,
                            long ntraj, const double *chi, double *pq_out, double *S_out, double *M_out,
                            double *theta_out, unsigned char *good_out, double *z_out) {
  pes_t P;
  scheme_t sc;
  int rc = pes_init(&P, F, kind, coeffs, ncoef);
  if (rc) return rc;
  if (scheme_init(&sc, integrator)) return SCO_EINVAL;
  if (!(dt > 0.0) || nsteps < 0 || ntraj < 1 || det_stride < 1) return SCO_EINVAL;
  for (int k = 0; k < F; k++) if (!(gamma[k] > 0.0)) return SCO_EINVAL;
  double zero_chi[2 * SCO_MAXF];
  memset(zero_chi, 0, sizeof(zero_chi));
  const double *chi_use = chi ? chi : zero_chi;
#pragma omp parallel for schedule(dynamic, 4)
  for (long j = 0; j < ntraj; j++) {
    double p0[SCO_MAXF], q0[SCO_MAXF], th;
    state_t fin;
    for (int k = 0; k < F; k++) { p0[k] = p0q0[k * ntraj + j]; q0[k] = p0q0[(F + k) * ntraj + j]; }
    double *z = z_out ? z_out + 2 * (size_t)j * (size_t)(nsteps + 1) : NULL;
    int good = propagate_one(&P, &sc, gamma, chi_use, 1, NULL, dt, nsteps, det_stride, det_tol, p0, q0, z, &fin, &th);
    if (pq_out)
      for (int k = 0; k < F; k++) { pq_out[k * ntraj + j] = fin.p[k]; pq_out[(F + k) * ntraj + j] = fin.q[k]; }
    if (S_out) S_out[j] = fin.S;
    if (M_out)
      for (int a = 0; a < F * F; a++) {
        M_out[((size_t)0 * F * F + a) * ntraj + j] = fin.Mpp[a];
        M_out[((size_t)1 * F * F + a) * ntraj + j] = fin.Mpq[a];
        M_out[((size_t)2 * F * F + a) * ntraj + j] = fin.Mqp[a];
        M_out[((size_t)3 * F * F + a) * ntraj + j] = fin.Mqq[a];
      }
    if (theta_out) theta_out[j] = th;
    if (good_out) good_out[j] = (unsigned char)good;
  }
  return SCO_OK;
}

/*
 * a8: A_j(E_i) = sum_{c=0}^{nsteps} z_{j,c} e^{i E_i c dt}  (Eq. 11).
 * fourier_mode 0 ("exact"): the definition, one cexp per term.
 * fourier_mode 1 ("recur"): the same sum with the twiddle advanced by w <- w r, r = e^{i E_i dt},
 *   re-seeded with an exact cexp every 256 steps (error <= 256 eps per term); pinned to mode 0 by
 *   tests/test_oracle_pins.py (test_p10_*).  Used where mode 0 would take hours.
 * Asq[i] += wj * |A_j(E_i)|^2 for one trajectory.
 */
static void fourier_accumulate(const double *z, int nsteps, double dt, const double *E, int k, int mode,
                               double wj, double *Isum, int i0, int i1) {
  for (int i = i0; i < i1; i++) {
    double complex A = 0.0;
    if (mode == 0) {
      for (int c = 0; c <= nsteps; c++) A += (z[2 * c] + I * z[2 * c + 1]) * cexp(I * (E[i] * (c * dt)));
    } else {
      double complex r = cexp(I * (E[i] * dt)), w = 1.0;
      for (int c = 0; c <= nsteps; c++) {
        if ((c & 255) == 0) w = cexp(I * (E[i] * (c * dt)));
        A += (z[2 * c] + I * z[2 * c + 1]) * w;
        w *= r;
      }
    }
    Isum[i] += wj * (creal(A) * creal(A) + cimag(A) * cimag(A));
  }
  (void)k;
}

/* Fourier amplitudes of given series, for the pins: A_out [n][k][2] from z [n][nsteps+1][2]. */
int sc_ivr_oracle_fourier(const double *z, long n, int nsteps, double dt, const double *E, int k, int mode,
                          double *A_out) {
  if (n < 1 || nsteps < 0 || k < 1) return SCO_EINVAL;
  for (long j = 0; j < n; j++) {
    const double *zj = z + 2 * (size_t)j * (size_t)(nsteps + 1);
    for (int i = 0; i < k; i++) {
      double complex A = 0.0;
      if (mode == 0) {
        for (int c = 0; c <= nsteps; c++) A += (zj[2 * c] + I * zj[2 * c + 1]) * cexp(I * (E[i] * (c * dt)));
      } else {
        double complex r = cexp(I * (E[i] * dt)), w = 1.0;
        for (int c = 0; c <= nsteps; c++) {
          if ((c & 255) == 0) w = cexp(I * (E[i] * (c * dt)));
          A += (zj[2 * c] + I * zj[2 * c + 1]) * w;
          w *= r;
        }
      }
      A_out[2 * ((size_t)j * k + i)] = creal(A);
      A_out[2 * ((size_t)j * k + i) + 1] = cimag(A);
    }
  }
  return SCO_OK;
}

/*
 * The whole path: I(E_i) = dt^2 / ((2 pi)^{F+1} T n_good) * sum_j w_j good_j |A_j(E_i)|^2,  T = nsteps dt
 * (Eq. 11 with R4's dt^2, R5's nsteps+1 unit-weight samples, R7's weights).  Trajectories are summed in
 * index order: they are processed in chunks (threads share the chunk's propagation, then split the
 * energies; within an energy the loop over j is sequential and chunks follow one another).
 * weights may be NULL (= 1).  Returns SCO_ENOGOOD with I = 0 when no trajectory survives (R18).
 */
static int run_impl(int F, int kind, const double *coeffs, long ncoef, const double *gamma, double dt,
                    int nsteps, int integrator, int det_stride, double det_tol, const double *p0q0,
                    const double *weights, long ntraj, const double *chi, int ncs, const double *eps, const double *E, int k,
                    int fourier_mode, double *I_out, long long *n_good_out) {
  pes_t P;
  scheme_t sc;
  int rc = pes_init(&P, F, kind, coeffs, ncoef);
  if (rc) return rc;
  if (scheme_init(&sc, integrator)) return SCO_EINVAL;
  if (!(dt > 0.0) || nsteps < 1 || ntraj < 1 || k < 1 || det_stride < 1 || !chi || !E || !I_out) return SCO_EINVAL;
  for (int a = 0; a < F; a++) if (!(gamma[a] > 0.0)) return SCO_EINVAL;
  const long CH = 256;
  double *z = (double *)malloc(sizeof(double) * 2 * (size_t)CH * (size_t)(nsteps + 1));
  unsigned char *good = (unsigned char *)malloc((size_t)CH);
  if (!z || !good) { free(z); free(good); return SCO_ENOMEM; }
  for (int i = 0; i < k; i++) I_out[i] = 0.0;
  long long n_good = 0;
  for (long j0 = 0; j0 < ntraj; j0 += CH) {
    long nj = ntraj - j0 < CH ? ntraj - j0 : CH;
#pragma omp parallel for schedule(dynamic, 1)
    for (long jj = 0; jj < nj; jj++) {
      long j = j0 + jj;
      double p0[SCO_MAXF], q0[SCO_MAXF];
      for (int a = 0; a < F; a++) { p0[a] = p0q0[a * ntraj + j]; q0[a] = p0q0[(F + a) * ntraj + j]; }
      good[jj] = (unsigned char)propagate_one(&P, &sc, gamma, chi, ncs, eps, dt, nsteps, det_stride, det_tol, p0, q0,
                                              z + 2 * (size_t)jj * (size_t)(nsteps + 1), NULL, NULL);
    }
    for (long jj = 0; jj < nj; jj++) n_good += good[jj];
    /* split the energies over threads; each I_out[i] sees j in index order */
#pragma omp parallel
    {
#ifdef _OPENMP
      int nt = omp_get_num_threads(), t = omp_get_thread_num();
#else
      int nt = 1, t = 0;
#endif
      int i0 = (int)((long)k * t / nt), i1 = (int)((long)k * (t + 1) / nt);
      for (long jj = 0; jj < nj; jj++) {
        if (!good[jj]) continue;
        double wj = weights ? weights[j0 + jj] : 1.0;
        fourier_accumulate(z + 2 * (size_t)jj * (size_t)(nsteps + 1), nsteps, dt, E, k, fourier_mode, wj, I_out, i0, i1);
      }
    }
  }
  free(z);
  free(good);
  if (n_good_out) *n_good_out = n_good;
  if (n_good == 0) {
    for (int i = 0; i < k; i++) I_out[i] = 0.0;
    return SCO_ENOGOOD;
  }
  double T = nsteps * dt;
  double norm = dt * dt / (pow(2.0 * M_PI, F + 1) * T * (double)n_good);
  for (int i = 0; i < k; i++) I_out[i] *= norm;
  return SCO_OK;
}

int sc_ivr_oracle_run(int F, int kind, const double *coeffs, long ncoef, const double *gamma, double dt,
                      int nsteps, int integrator, int det_stride, double det_tol, const double *p0q0,
                      const double *weights, long ntraj, const double *chi, const double *E, int k,
                      int fourier_mode, double *I_out, long long *n_good_out) {
  return run_impl(F, kind, coeffs, ncoef, gamma, dt, nsteps, integrator, det_stride, det_tol, p0q0, weights, ntraj, chi, 1, NULL,
                  E, k, fourier_mode, I_out, n_good_out);
}

/* The same path with the reference state |chi> = sum_m eps_m |p_m, q_m>  (chi [ncs][2F], eps [ncs][2]): PAPER.md:167-173. */
int sc_ivr_oracle_run_combo(int F, int kind, const double *coeffs, long ncoef, const double *gamma, double dt,
                            int nsteps, int integrator, int det_stride, double det_tol, const double *p0q0,
                            const double *weights, long ntraj, const double *chi, int ncs, const double *eps,
                            const double *E, int k, int fourier_mode, double *I_out, long long *n_good_out) {
  if (ncs < 1 || !eps) return SCO_EINVAL;
  return run_impl(F, kind, coeffs, ncoef, gamma, dt, nsteps, integrator, det_stride, det_tol, p0q0, weights, ntraj, chi, ncs, eps,
                  E, k, fourier_mode, I_out, n_good_out);
}
