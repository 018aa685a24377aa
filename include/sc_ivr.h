/*
 * sc_ivr.h - C ABI of the B200 (sm_100a) TA-SC-IVR power-spectrum library.
 *
 * What it computes (arxiv 1312.4698; citations are PAPER.md line numbers):
 *
 *   I(E_i) = dt^2 / ((2 pi)^(F+1) T n_good) * sum_j w_j good_j | sum_{c=0}^{nsteps} z_{j,c} e^{i E_i c dt} |^2
 *   z_{j,c} = <chi | p_j(c dt) q_j(c dt)> e^{i (S_j(c dt) + phi_j(c dt))}                Eq. 11
 *
 * the Monte Carlo / rectangle-rule form of the time-averaged, separable-prefactor SC-IVR
 * spectral density (Eq. 10), T = nsteps dt.  Per trajectory j, started at
 * (p0, q0), the library integrates (p, q) with a symplectic composition step (
 * velocity-Verlet by default), together with the F x F monodromy blocks M_pp, M_pq, M_qp, M_qq
 * (PAPER.md:64), the classical action S, the Herman-Kluk prefactor phase phi = continuous
 * branch of arg sqrt(det K),
 *   K_ab = 1/2 [ M_qq,ab + (g_b/g_a) M_pp,ab ] + (i/2) [ M_pq,ab / g_a - g_b M_qp,ab ]   Eq. 5
 * (g = gamma, the coherent-state widths), the coherent-state overlap with the reference state
 * chi = |p_eq, q_eq> (Eq. 3), and the quality flag
 * good_j = all finite and |det M - 1| <= det_tol at every checked step.
 * DESIGN.md lists every reading taken where the paper is silent (R1..R21).
 *
 * Conventions
 *   - Atomic units, hbar = 1.  All floating point is IEEE double.
 *   - "DEVICE" pointers are CUDA device memory of the current device, owned by the caller
 *     (PyTorch tensors in the Python binding); "HOST" pointers are ordinary host memory.
 *   - No entry point throws or aborts.  Each returns an sc_ivr_status; a message is kept in
 *     the context (sc_ivr_last_error).  There is NO CPU fallback: without a CUDA device
 *     sc_ivr_create fails with SC_IVR_ECUDA.
 *   - The library never allocates device memory in run/propagate/eval_pes: the caller passes a
 *     workspace.  sc_ivr_create makes one small cudaMalloc for the packed PES coefficients.
 *   - All device work of a call is enqueued on `cuda_stream` (a cudaStream_t cast to void*, NULL =
 *     legacy default stream).  Calls are asynchronous unless stated otherwise.
 *
 * Layouts
 *   p0q0   [2F][ntraj]   struct-of-arrays: rows 0..F-1 = p_k, rows F..2F-1 = q_k
 *   chi    [2F]          p_eq[F] then q_eq[F]
 *   M_out  [4][F][F][n]  blocks pp, pq, qp, qq;  M_xy[a][b] = d x_a(t) / d y_b(0)
 *   pes_coeffs
 *     SC_IVR_PES_MORSE1D (F must be 1): { D, a, q_e, mass },  V = D (1 - exp(-a (q - q_e)))^2
 *     SC_IVR_PES_MORSE_UNCOUPLED:       { D, a, q_e, mass } per mode, F blocks
 *     SC_IVR_PES_QFF (mass-weighted normal coordinates, all masses 1):
 *        omega[F];  cubic Phi_ijk for i<=j<=k in lexicographic order (F(F+1)(F+2)/6 values, the entry
 *        of the fully symmetric tensor);  quartic Phi_iijj for i<=j lexicographic (F(F+1)/2 values,
 *        i=j is Phi_iiii);   V = 1/2 sum w_i^2 q_i^2 + 1/6 sum_ijk Phi_ijk q_i q_j q_k
 *        + 1/24 sum_ijkl Phi_ijkl q_i q_j q_k q_l  (unrestricted sums; only pair-type quartic entries non-zero)
 */
#ifndef SC_IVR_H
#define SC_IVR_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SC_IVR_MAX_F 12

typedef struct sc_ivr_ctx sc_ivr_ctx; /* opaque, owned by the library */

typedef enum {
  SC_IVR_OK = 0,
  SC_IVR_EINVAL = 1,       /* bad argument (NULL, size, non-finite coefficient, workspace too small) */
  SC_IVR_ENOMEM = 2,
  SC_IVR_ECUDA = 3,        /* CUDA runtime error or no device */
  SC_IVR_EUNSUPPORTED = 4, /* F outside 1..SC_IVR_MAX_F, unknown PES kind / integrator */
  SC_IVR_ENOGOOD = 5       /* every trajectory was rejected; I_out is zero-filled */
} sc_ivr_status;

typedef enum { SC_IVR_PES_MORSE1D = 0, SC_IVR_PES_QFF = 1, SC_IVR_PES_MORSE_UNCOUPLED = 2 } sc_ivr_pes_kind;

typedef struct {
  int det_stride;  /* check det M every det_stride steps and at the last step; default 1 */
  double det_tol;  /* default 1e-6 */
  int integrator;  /* 0 = velocity-Verlet (default), 1 = 4-stage 4th-order symplectic */
  double lu_growth_max; /* the two determinants are eliminated in a fixed pivot order while every multiplier of det K
                           stays below lu_growth_max and every multiplier of det M below lu_growth_max^2; a step that
                           exceeds them is repeated with pivoting, and so is the first step at
                           which the fixed order finds |det M - 1| > det_tol: a trajectory is only rejected by the pivoted
                           elimination.  0 = default 1e4; < 0 = always use the pivoted eliminations
                           (testing) */
  int fourier_mode;     /* 0 = automatic: an equally spaced energy grid with k <= 7169 and at most 16
                           blocks of 8193 - k time samples takes the chirp-z (FFT) evaluation of the sum of Eq. 11,
                           anything else the direct sum; 1 = always the direct sum */
} sc_ivr_options;

/*
 * Create a context for one potential-energy surface and one time grid.
 *   out        receives the context (NULL on failure).
 *   pes_coeffs HOST [n_coeffs], layout above, copied.
 *   gamma      HOST [F], coherent-state widths, all > 0, copied.
 *   dt > 0, nsteps >= 1.   opt may be NULL (defaults).
 * Synchronous (one small host-to-device copy).
 */
sc_ivr_status sc_ivr_create(sc_ivr_ctx **out, int F, sc_ivr_pes_kind kind, const double *pes_coeffs,
                            size_t n_coeffs, const double *gamma, double dt, int nsteps,
                            const sc_ivr_options *opt);

void sc_ivr_destroy(sc_ivr_ctx *ctx);

/* Library-owned, NUL-terminated; valid until the next call on ctx.  ctx == NULL gives the message of the
 * last failed sc_ivr_create on this thread. */
const char *sc_ivr_last_error(const sc_ivr_ctx *ctx);

/*
 * Bytes of DEVICE workspace sc_ivr_run wants for (ntraj, k) so that trajectories are processed in
 * batches of at most `max_batch` (0 = library default, 131072).  A smaller workspace is accepted as
 * long as it holds one batch of sc_ivr_min_batch(ctx) trajectories; run then uses more, smaller batches.
 */
size_t sc_ivr_workspace_bytes(const sc_ivr_ctx *ctx, long long ntraj, int k, long long max_batch);
long long sc_ivr_min_batch(const sc_ivr_ctx *ctx);

/*
 * The whole path, Eq. 11: I_out[i] = I(E[i]).
 *   p0q0      DEVICE [2F][ntraj]          weights  DEVICE [ntraj] or NULL (all 1)
 *   chi       HOST [2F]                   E        HOST [k], atomic units, any values
 *   I_out     DEVICE [k], overwritten     n_good_out HOST, may be NULL
 *   workspace DEVICE, >= the size described above, 256-byte aligned
 * Trajectories are reduced in a fixed order (no atomics): results are bitwise
 * reproducible for fixed (inputs, workspace size).  Asynchronous on cuda_stream when n_good_out is
 * NULL (then a batch with no good trajectory yields I_out = 0 and SC_IVR_OK); otherwise the stream
 * is synchronised once at the end and SC_IVR_ENOGOOD is returned when n_good == 0.
 * Lifetime in the asynchronous case: E is copied to the device with cudaMemcpyAsync on cuda_stream; if it is PINNED host
 * memory the caller keeps it alive and unmodified until the stream has passed this call (pageable memory is staged before
 * the call returns).  chi is consumed before the call returns.
 * Device: the call must be issued with the context's device current (the one that was current in sc_ivr_create);
 * otherwise SC_IVR_EINVAL.  The same holds for every other entry point that takes a stream.
 */
sc_ivr_status sc_ivr_run(sc_ivr_ctx *ctx, const double *p0q0, const double *weights, long long ntraj,
                         const double *chi, const double *E, int k, double *I_out, long long *n_good_out,
                         void *workspace, size_t workspace_bytes, void *cuda_stream);

/*
 * Same computation with HOST inputs and outputs: p0q0 [2F][ntraj], weights [ntraj] or NULL and
 * I_out [k] are HOST buffers (pinned memory makes the copies asynchronous).  The workspace (DEVICE)
 * must be sc_ivr_workspace_bytes(...) + sc_ivr_host_staging_bytes(...) large.  Synchronises the
 * stream before returning.
 */
size_t sc_ivr_host_staging_bytes(const sc_ivr_ctx *ctx, long long ntraj, int k);
sc_ivr_status sc_ivr_run_host(sc_ivr_ctx *ctx, const double *p0q0, const double *weights, long long ntraj,
                              const double *chi, const double *E, int k, double *I_out,
                              long long *n_good_out, void *workspace, size_t workspace_bytes,
                              void *cuda_stream);

/*
 * Several reference states per run, each a combination of coherent states (Fig. 4: the spectrum is
 * projected on irreducible representations with "different coherent state combinations"):
 *   |chi_n> = sum_m eps[n][m] |p_m, q_m>,   <chi_n|p q> = sum_m conj(eps[n][m]) <p_m q_m|p q>   (each overlap: Eq. 3),
 *   I_out[n][i] = I(E_i) of Eq. 11 with chi = chi_n.
 * The trajectories (a1-a5, a7) are propagated ONCE and shared by all nchi reference states; only the overlaps (a6) and the
 * Fourier / reduction stages (a8, a9) are repeated per state.
 *   chis  HOST [ncs][2F]  (p_m[F] then q_m[F])        eps  HOST [nchi][ncs][2]  (re, im)
 *   I_out DEVICE [nchi][k]                             E    HOST [k], equally spaced (chirp-z path only)
 *   workspace DEVICE, sc_ivr_multi_workspace_bytes(ctx, ntraj, k, ncs, max_batch); a smaller one (>= one batch of
 *   sc_ivr_min_batch) makes more, smaller batches.  1 <= ncs <= 16, 1 <= nchi <= 16.
 * Other arguments, ordering and error behaviour as sc_ivr_run, except that this call ALWAYS synchronises the stream before it
 * returns (with or without n_good_out); SC_IVR_EUNSUPPORTED when the grid is not equally spaced or too long for the chirp-z
 * stage.
 */
size_t sc_ivr_multi_workspace_bytes(const sc_ivr_ctx *ctx, long long ntraj, int k, int ncs, long long max_batch /*0 = 32768*/);
sc_ivr_status sc_ivr_run_multi(sc_ivr_ctx *ctx, const double *p0q0, const double *weights, long long ntraj, const double *chis,
                               int ncs, const double *eps, int nchi, const double *E, int k, double *I_out,
                               long long *n_good_out, void *workspace, size_t workspace_bytes, void *cuda_stream);

/*
 * Parity / debug entry: propagate only (steps a1-a7), return the state after nsteps_run steps
 * (0 <= nsteps_run; independent of the context's nsteps).  Any output may be NULL.
 *   pq_out    DEVICE [2F][ntraj]      S_out  DEVICE [ntraj]       M_out DEVICE [4][F][F][ntraj]
 *   theta_out DEVICE [ntraj], continuous (unwrapped) arg det K at the last step = 2 phi
 *   good_out  DEVICE [ntraj] bytes
 *   z_out     DEVICE [nsteps_run+1][ntraj][2], z_{j,c} of Eq. 11 (needs chi; chi NULL = zeros)
 *   workspace DEVICE, sc_ivr_propagate_workspace_bytes(ctx, ntraj, nsteps_run)
 */
size_t sc_ivr_propagate_workspace_bytes(const sc_ivr_ctx *ctx, long long ntraj, int nsteps_run);
sc_ivr_status sc_ivr_propagate(sc_ivr_ctx *ctx, const double *p0q0, long long ntraj, int nsteps_run,
                               const double *chi, double *pq_out, double *S_out, double *M_out,
                               double *theta_out, unsigned char *good_out, double *z_out,
                               void *workspace, size_t workspace_bytes, void *cuda_stream);

/*
 * Parity / debug entry for the z assembly alone (the branch rule of a5, a6 and the input of a8): from the per-step records that
 * the propagation kernel writes to the z_{j,c} of Eq. 11, by the kernel sc_ivr_propagate and the direct-sum
 * path of sc_ivr_run use.
 *   raw       DEVICE [nsteps_run+1][n][4]: (ln|<chi|pq>|, S + arg<chi|pq>, Re D, Im D), D = det 2K times ANY positive factor
 *             (only its phase is used; components from subnormal up to the largest finite double are handled)
 *   z_out     DEVICE [nsteps_run+1][n][2]:  exp(raw0) e^{i raw1} u_c,  u_c = the square root of D_c / |D_c| on the branch that is
 *             continuous in c, u_0 the principal one
 *   theta_out DEVICE [n] or NULL: the unwrapped arg D at the last step
 */
sc_ivr_status sc_ivr_assemble_z(sc_ivr_ctx *ctx, const double *raw, long long n, int nsteps_run, double *z_out,
                                double *theta_out, void *cuda_stream);

/*
 * Parity / debug entry for step a1: the potential, its gradient and Hessian, evaluated by the same
 * device code the propagation kernel inlines.   q DEVICE [F][n] -> V_out [n], g_out [F][n], H_out [F][F][n].
 */
sc_ivr_status sc_ivr_eval_pes(sc_ivr_ctx *ctx, const double *q, long long n, double *V_out, double *g_out,
                              double *H_out, void *cuda_stream);

/*
 * Parity / debug entry for step a8 alone: A_out[j][i] = sum_c z[c][j] e^{i E_i c dt} computed by the
 * production Fourier kernel.   z DEVICE [nsteps+1][n][2] (time-major), E HOST [k],
 * A_out DEVICE [n][k][2], workspace DEVICE sc_ivr_fourier_workspace_bytes(ctx, n, k).
 */
size_t sc_ivr_fourier_workspace_bytes(const sc_ivr_ctx *ctx, long long n, int k);
sc_ivr_status sc_ivr_fourier(sc_ivr_ctx *ctx, const double *z, long long n, const double *E, int k,
                             double *A_out, void *workspace, size_t workspace_bytes, void *cuda_stream);

/*
 * The same sum (Eq. 11; the kernels of sc_ivr_fourier) for callers that CANNOT ALLOCATE device memory and so
 * have no workspace to pass: a plug-in inside a program whose own pool took all of HBM at start-up (any later cudaMalloc
 * fails there), a step in a latency-bound loop (cudaMalloc / cudaFree lock the driver and synchronise the device for an
 * unbounded time), a process whose device-memory budget is fixed and spent.  The scratch (zero-padded copy of z + twiddle
 * table) is a static array of SC_IVR_STATIC_SCRATCH_BYTES inside the library's device image; every GPU that loads the
 * library's kernels holds it until the process exits.  The call needs no context, performs no cudaMalloc / cudaFree /
 * cudaMemcpy and calls nothing that allocates.
 *   z      DEVICE [nsteps+1][n][2] (time-major)      E      DEVICE [k] (not HOST: there is nowhere to stage a copy)
 *   A_out  DEVICE [n][k][2], overwritten              dt     any finite value; nsteps >= 0
 * Limit: sc_ivr_fourier_static_scratch_bytes(n, nsteps, k) = 16 ceil16(nsteps+1) (ceil128(n) + ceil64(k)) bytes (each term
 * rounded to 256) must be <= SC_IVR_STATIC_SCRATCH_BYTES, e.g. n <= 128 trajectories x 1001 time samples x 896 energies;
 * larger sizes are rejected with SC_IVR_EINVAL and a message that names both numbers (split the call over trajectories or
 * energies, the sum is independent in both).  The size query returns 0 for arguments that are out of range.
 * First call on a device: looks up the array's device address (cudaGetSymbolAddress, once per device, with that device
 * current; thread-safe).  Make this first call outside any stream capture.  Later calls only launch kernels on cuda_stream.
 * Sharing: there is ONE array per device.  Every call overwrites all of it that it reads (nothing has to be cleared by the
 * caller, the previous call's contents never leak into a result), and it is dead once the call's kernels have finished.
 * Two calls whose kernels can overlap on the GPU (different streams without an event between them, or two host threads
 * on different streams) RACE on it: serialise them.  Calls on one stream are ordered and safe.
 * Asynchronous; errors as everywhere (status + message), but the message is per host thread and read with
 * sc_ivr_fourier_static_last_error() because there is no context to keep it.
 */
#define SC_IVR_STATIC_SCRATCH_BYTES (16u << 20)
size_t sc_ivr_fourier_static_scratch_bytes(long long n, int nsteps, int k);
sc_ivr_status sc_ivr_fourier_static(const double *z, long long n, int nsteps, double dt, const double *E, int k, double *A_out,
                                    void *cuda_stream);
const char *sc_ivr_fourier_static_last_error(void);

/*
 * Parity / debug entry for step a8 through the chirp-z kernels that sc_ivr_run uses on equally spaced grids:
 * P_out[j][i] = | sum_c z[c][j] e^{i E_i c dt} |^2.   z DEVICE [nsteps+1][n][2] (time-major), E HOST [k] equally spaced,
 * P_out DEVICE [n][k], workspace DEVICE sc_ivr_fourier_power_workspace_bytes(ctx, n, k).
 * SC_IVR_EUNSUPPORTED when the grid is not equally spaced, k > 7169 or the series needs more than 16 blocks.
 */
size_t sc_ivr_fourier_power_workspace_bytes(const sc_ivr_ctx *ctx, long long n, int k);
sc_ivr_status sc_ivr_fourier_power(sc_ivr_ctx *ctx, const double *z, long long n, const double *E, int k, double *P_out,
                                   void *workspace, size_t workspace_bytes, void *cuda_stream);

/*
 * Measurement helpers (no method arithmetic).
 * sc_ivr_fp64_probe: runs a register-only DFMA loop (mode 0) or an mma.sync m8n8k4 f64 loop (mode 1)
 * on every SM and returns the achieved FLOP/s (2 flop per FMA) in *flops_out.  Synchronous.
 * Issue-budget probes, mode = kind + 10 * wps: kind 2 = the DFMA loop with a 64-bit warp shuffle after every 4 DFMAs, 3 = with
 * an LDS.64 after every 4, 4 = with an integer LOP3 / IADD3 pair after every DFMA (only the DFMAs count as flop: a rate equal to
 * kind 0's means the extra instruction issued in the FP64 pipe's shadow); wps 0 = 16 warps per scheduler, 1 or 2 = exactly that
 * many (one CTA of 128 or 256 threads per SM), which is the occupancy kernel A runs at.  Other modes: SC_IVR_EINVAL.
 * sc_ivr_last_timings: device times in ms (CUDA events on the run stream) of the stages of the most
 * recent sc_ivr_run on ctx, summed over batches: [0] propagate kernel, [1] z assembly, [2] twiddle / chirp tables,
 * [3] Fourier kernel (direct sum or chirp-z), [4] reduction kernels; [5] number of kernel launches.  Synchronises the stream's
 * last event.  Timing is recorded only after sc_ivr_set_timing(ctx, 1).
 */
sc_ivr_status sc_ivr_fp64_probe(int mode, int iters, double *flops_out, double *ms_out);
/* Number of trajectory-steps of the most recent sc_ivr_run with n_good_out != NULL (or sc_ivr_run_host) on ctx whose
 * determinants were repeated with the pivoted eliminations because a multiplier of the fixed-order elimination exceeded
 * lu_growth_max or because the fixed order was about to reject the trajectory; -1 when that run did not read it back.
 * Statistics only. */
long long sc_ivr_last_fallbacks(const sc_ivr_ctx *ctx);
void sc_ivr_set_timing(sc_ivr_ctx *ctx, int on);
sc_ivr_status sc_ivr_last_timings(sc_ivr_ctx *ctx, double out[6]);

#ifdef __cplusplus
}
#endif
#endif /* SC_IVR_H */
