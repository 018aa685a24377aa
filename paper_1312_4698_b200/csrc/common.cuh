// Internal declarations shared by the translation units of libsc_ivr (CUDA path only; the CPU
// oracle under oracle/ shares nothing with this directory).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/sc_ivr.h"

#define SCI_MAXF SC_IVR_MAX_F
#define SCI_MAX_STAGES 4

// ---- kernel A (propagate) parameters: passed by value, read through the constant bank ----------
// All per-mode quantities are in REDUCED coordinates Q_k = sqrt(gamma_k) q_k, P_k = p_k / sqrt(gamma_k)
// (pin P8): the Herman-Kluk matrix becomes
// 2K = (M_qq + M_pp) + i (M_pq - M_qp) with no gamma factors.
struct PropParams {
  const double *p0q0;   // [2F][stride]
  long long stride;     // ntraj of the caller's array
  long long j0;         // first trajectory of this launch
  long long nb;         // trajectories in this launch
  int nsteps;
  int det_stride;
  double det_tol;
  unsigned grow_k_max, grow_m_max;  // static-order LU: largest tolerated multiplier, as the high word of the double
  int nstages;
  double kick[SCI_MAX_STAGES];   // b_i * dt
  double drift[SCI_MAX_STAGES];  // a_i * dt
  // the same composition as a table of evaluation points (propagate_cml.cu): a step visits npoints positions; at point e
  // the kicks up to the snapshot sum to pt_pre[e] (point 0 only: the end of the previous step), those after it to
  // pt_post[e], and the drift that leaves the point is pt_drift[e]
  int npoints;
  double pt_pre[SCI_MAX_STAGES], pt_post[SCI_MAX_STAGES], pt_drift[SCI_MAX_STAGES];
  double sg[SCI_MAXF];           // sqrt(gamma)
  double isg[SCI_MAXF];          // 1/sqrt(gamma)
  double mu[SCI_MAXF];           // gamma/mass: dQ/dt = mu P, T = 1/2 sum mu P^2
  double Peq[SCI_MAXF], Qeq[SCI_MAXF];
  const double *coef;            // packed reduced PES coefficients (device)
  double4 *raw;                  // [nsteps+1][raw_stride]: (ln|<chi|pq>|, S + arg<chi|pq>, Re det 2K, Im det 2K); may be NULL
  long long raw_stride;
  // several reference states per run (row f4): when pq_steps != NULL the kernel also stores (P_a, Q_a) (reduced) of every
  // step, [nsteps+1][F][raw_stride], and with raw_plain != 0 the record is (0, S, Re det 2K, Im det 2K): the overlaps are
  // then formed per reference state by the z assembly
  double2 *pq_steps;
  int raw_plain;
  int cta_full, cta_warps, cta_warps_rem;  // propagate_cml.cu: launch shape, set by the launcher
  unsigned long long *fb_count;  // may be NULL: number of trajectory-steps repeated with the pivoted eliminations
  unsigned char *good;           // [nb]; may be NULL
  // debug outputs (may be NULL), indexed by the GLOBAL trajectory number j0 + jj with stride `stride`
  double *pq_out, *S_out, *M_out;
};

// thread-per-trajectory kernels (F <= SCI_TPT_MAXF, propagate_tpt.cu): parameters + dense reduced PES constants, all
// passed by value so that the constants are constant-bank operands
#define SCI_TPT_MAXF 3
#define SCI_TPT_NCOEF 40
struct TptParams {
  PropParams P;
  double coef[SCI_TPT_NCOEF];
};

struct sc_ivr_ctx {
  int F, kind, nsteps, det_stride, integrator, fourier_mode;
  double dt, det_tol, lu_growth_max;
  double gamma[SCI_MAXF], mass[SCI_MAXF];
  int nstages;
  double sa[SCI_MAX_STAGES], sb[SCI_MAX_STAGES];
  double *d_coef;
  size_t n_coef;
  double tpt_coef[SCI_TPT_NCOEF];  // F <= SCI_TPT_MAXF only
  int device, sm_count;
  long long wave;  // trajectories one full wave of kernel A holds (batch granularity)
  char err[512];
  int timing;
  double tms[6];
  long long last_fallbacks;  // of the most recent synchronising sc_ivr_run; -1 = not read back
  // stage timing: (start, stop) event pairs recorded without synchronising, resolved by sc_ivr_last_timings
  std::vector<cudaEvent_t> ev;
  std::vector<int> ev_slot;
  size_t ev_used;
};

// C-modes-per-lane kernels with the monodromy state in tensor memory (propagate_cml.cu)
int sci_cml_lanes(int F);  // lanes per trajectory, 0 = F is not served by these kernels
int sci_cml_traj_per_block(int F);
size_t sci_cml_pack_coeffs(int F, int kind, const double *coeffs, const double *gamma, double *out /*may be NULL: size query*/);
cudaError_t sci_cml_launch_propagate(int F, int kind, const PropParams &P, cudaStream_t st);
cudaError_t sci_cml_launch_eval_pes(int F, int kind, const double *coef, const double *sg, const double *q,
                                    long long n, double *V, double *g, double *H, cudaStream_t st);

// thread-per-trajectory kernels (propagate_tpt.cu)
int sci_tpt_traj_per_block();
int sci_tpt_blocks_per_sm(int F, int kind);
int sci_tpt_pack_coeffs(int F, int kind, const double *coeffs, const double *gamma, double *out /*[SCI_TPT_NCOEF]*/);
cudaError_t sci_tpt_launch_propagate(int F, int kind, const TptParams &TP, cudaStream_t st);
cudaError_t sci_tpt_launch_eval_pes(int F, int kind, const TptParams &TP, const double *q, long long n, double *V, double *g,
                                    double *H, cudaStream_t st);

// spectrum stage (spectrum.cu)
#define SCI_TJ 128  // trajectories per Fourier tile
#define SCI_TI 64   // energies per Fourier tile
#define SCI_KC 16   // time samples per pipeline stage
cudaError_t sci_launch_zassemble(const double4 *raw, long long raw_stride, long long nb, int nsteps, double2 *z,
                                 long long zstride, long long zcols, int zrows, double *theta_out, cudaStream_t st);
cudaError_t sci_launch_twiddle(const double *E_dev, int k, int kp, int rows, double dt, double2 *W, cudaStream_t st);
cudaError_t sci_launch_fourier(const double2 *z, long long zstride, long long zcols, int zrows, const double2 *W, int kp, long long nb,
                               const double *wg /*[nb] weight*good*/, double *partial /*[tiles][kp]*/,
                               double2 *A_out /*debug [nb][k] or NULL*/, int k, cudaStream_t st);
cudaError_t sci_launch_weights(const double *w, const unsigned char *good, long long n, double *wg, cudaStream_t st);
cudaError_t sci_launch_count_good(const unsigned char *good, long long n, long long *ngood, int accumulate, cudaStream_t st);
cudaError_t sci_launch_final(const double *partial, long long ntiles, int kp, int k, const long long *ngood, double norm_no_ngood,
                             double *I_out, cudaStream_t st);
cudaError_t sci_fp64_probe(int mode, int iters, double *flops, double *ms);

// chirp-z Fourier stage for equally spaced energy grids (chirp.cu)
#define SCI_CHIRP_L 8192        // circular convolution length; blocks of SCI_CHIRP_L - k + 1 time samples
#define SCI_CHIRP_MIN_BLOCK 1024 // shorter blocks (k > 7169) or more than SCI_CHIRP_MAX_BLOCKS of them: direct sum instead
#define SCI_CHIRP_MAX_BLOCKS 16
size_t sci_chirp_smem_bytes();
cudaError_t sci_launch_chirp_tables(double e0dt, double theta, int n1, int k, int nblocks, int bsz, double2 *pc, double2 *hrow,
                                    cudaStream_t st);
cudaError_t sci_launch_zassemble_rows(const double4 *raw, long long raw_stride, long long nb, int nsteps, const double2 *pc,
                                      double2 *xrows, long long xstride, cudaStream_t st);
cudaError_t sci_launch_overlap_phase(const double4 *raw, const double2 *pq_steps, long long raw_stride, long long nb, int nsteps, int F,
                                     const double *chis_reduced /*[ncs][2F]: P_eq then Q_eq*/, int ncs, const double2 *pc,
                                     double2 *ovph /*[nsteps+1][ncs+1][raw_stride]*/, cudaStream_t st);
cudaError_t sci_launch_combine_rows(const double2 *ovph, long long raw_stride, long long nb, int nsteps, const double *eps /*[ncs][2]*/,
                                    int ncs, double2 *xrows, long long xstride, cudaStream_t st);
cudaError_t sci_launch_rows_from_z(const double2 *z, long long n, int n1, const double2 *pc, double2 *xrows, long long xstride,
                                   cudaStream_t st);
cudaError_t sci_launch_chirp_fft(int mode, const double2 *x, long long xstride, int n1, long long nrows, const double2 *HpT,
                                 const double *wg, int k, int kp, double *out, double2 *spec_out, int nblocks, int bsz,
                                 double2 *yscr, int grid, cudaStream_t st);

#ifdef __CUDACC__
// 1 / |D| for D = (re, im) without overflow or underflow of the squares: the determinant record carries an arbitrary positive
// factor (the static elimination hands over det 2K times |prod 1/pivot|^2), so it is brought to unit scale by a power of two
// taken from the larger component's exponent before it is squared (the oracle uses cabs).  The power 2^(1023 - ex) is a normal
// double for every ex <= 0x7fd, subnormal inputs (ex = 0) included: they come out in [2^-51, 2), whose squares are far from
// underflow.  For ex = 0x7fe (|D| >= 2^1023) it would be 2^-1023, which is not, so such a record is quartered first.  ex = 0x7ff
// (inf, NaN) yields NaN, as it must: that trajectory is rejected by the finite check of a7.  D = 0 exactly yields NaN too (det K
// = 0 has no phase; the oracle's division by cabs = 0 does the same).
__device__ __forceinline__ double unit_scale(double &re, double &im) {
  int ex = (int)((max((unsigned)__double2hiint(re) & 0x7fffffffu, (unsigned)__double2hiint(im) & 0x7fffffffu) >> 20) & 0x7ffu);
  if (ex >= 0x7fe) {
    re *= 0.25;
    im *= 0.25;
    ex -= 2;
  }
  const double sc = __hiloint2double((0x7fe - ex) << 20, 0);  // 2^(1023 - ex)
  re *= sc;
  im *= sc;
  return 1.0 / sqrt(fma(re, re, im * im));
}
#endif
