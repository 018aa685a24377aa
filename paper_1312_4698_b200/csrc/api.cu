// C ABI of libsc_ivr (include/sc_ivr.h): argument validation, workspace carving, kernel sequencing.
// No method arithmetic lives here except the host-side constants (reduced-coordinate scaling, the
// normalisation of Eq. 11).
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <new>
#include <vector>

#include <stdlib.h>

#include "common.cuh"

namespace {

thread_local char g_create_err[512] = "";

sc_ivr_status fail(sc_ivr_ctx *ctx, sc_ivr_status st, const char *fmt, ...) {
  char *dst = ctx ? ctx->err : g_create_err;
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(dst, 512, fmt, ap);
  va_end(ap);
  return st;
}

// every entry point that launches work: the context's device (kernel attributes, coefficient buffers) must be current
sc_ivr_status check_device(sc_ivr_ctx *ctx) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return fail(ctx, SC_IVR_ECUDA, "cannot query the current device");
  if (dev != ctx->device)
    return fail(ctx, SC_IVR_EINVAL, "context belongs to device %d but device %d is current", ctx->device, dev);
  return SC_IVR_OK;
}

#define CU(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) return fail(ctx, SC_IVR_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline long long round_up_ll(long long x, long long a) { return (x + a - 1) / a * a; }

long n_coeffs_expected(int F, int kind) {
  if (kind == SC_IVR_PES_MORSE1D) return 4;
  if (kind == SC_IVR_PES_QFF) return F + (long)F * (F + 1) * (F + 2) / 6 + (long)F * (F + 1) / 2;
  if (kind == SC_IVR_PES_MORSE_UNCOUPLED) return 4L * F;
  return -1;
}

// Workspace layout for one run.  Everything 256-byte aligned.
struct Carve {
  long long nbatch;     // trajectories per batch
  long long nbp;        // nbatch rounded to the Fourier tile (z row stride)
  int rows, zrows, kp;  // nsteps+1, rows padded to KC, k padded to TI
  long long tiles_total;
  long long xstride;    // chirp path: row stride of x[j][c] (rows = nsteps+1 rounded up to 32)
  size_t off_raw, off_z, off_W, off_partial, off_good, off_wg, off_E, off_ngood, off_pc, off_hrow, off_HpT, off_yscr, total;
};

Carve carve(const sc_ivr_ctx *ctx, long long ntraj, int k, long long nbatch) {
  Carve c;
  c.nbatch = nbatch;
  c.nbp = round_up_ll(nbatch, SCI_TJ);
  c.rows = ctx->nsteps + 1;
  c.zrows = (int)round_up_ll(c.rows, SCI_KC);
  c.kp = (int)round_up_ll(k, SCI_TI);
  const long long nbatches = (ntraj + nbatch - 1) / nbatch;
  c.tiles_total = nbatches * (c.nbp / SCI_TJ);
  if (c.tiles_total < nbatches * ctx->sm_count) c.tiles_total = nbatches * ctx->sm_count;  // chirp path: one partial per CTA
  c.xstride = round_up_ll(c.rows, 32);
  size_t zbytes = sizeof(double2) * (size_t)c.zrows * (size_t)c.nbp;                   // direct path: z[c][j]
  const size_t xbytes = sizeof(double2) * (size_t)c.xstride * (size_t)nbatch;          // chirp path:  x[j][c]
  if (xbytes > zbytes) zbytes = xbytes;
  size_t o = 0;
  c.off_raw = o; o = align_up(o + sizeof(double4) * (size_t)c.rows * (size_t)nbatch, 256);
  c.off_z = o; o = align_up(o + zbytes, 256);
  c.off_W = o; o = align_up(o + sizeof(double2) * (size_t)c.zrows * (size_t)c.kp, 256);
  c.off_partial = o; o = align_up(o + sizeof(double) * (size_t)c.tiles_total * (size_t)c.kp, 256);
  c.off_good = o; o = align_up(o + (size_t)ntraj, 256);
  c.off_wg = o; o = align_up(o + sizeof(double) * (size_t)ntraj, 256);
  c.off_E = o; o = align_up(o + sizeof(double) * (size_t)k, 256);
  c.off_ngood = o; o = align_up(o + 64, 256);
  c.off_pc = o; o = align_up(o + sizeof(double2) * (size_t)c.rows, 256);
  c.off_hrow = o; o = align_up(o + sizeof(double2) * SCI_CHIRP_L * SCI_CHIRP_MAX_BLOCKS, 256);
  c.off_HpT = o; o = align_up(o + sizeof(double2) * SCI_CHIRP_L * SCI_CHIRP_MAX_BLOCKS, 256);
  c.off_yscr = o; o = align_up(o + sizeof(double2) * SCI_CHIRP_L * (size_t)ctx->sm_count, 256);
  c.total = o;
  return c;
}

long long default_batch(const sc_ivr_ctx *ctx, long long ntraj, long long max_batch) {
  if (max_batch <= 0) max_batch = 131072;
  long long nb = ntraj < max_batch ? ntraj : max_batch;
  if (nb < ntraj) {  // several batches: make each a whole number of kernel-A waves
    nb = nb / ctx->wave * ctx->wave;
    if (nb < ctx->wave) nb = ctx->wave;
  }
  return nb;
}

void fill_prop_params(const sc_ivr_ctx *ctx, PropParams &P, const double *chi) {
  memset(&P, 0, sizeof(P));
  const int F = ctx->F;
  P.nstages = ctx->nstages;
  for (int s = 0; s < ctx->nstages; s++) {
    P.kick[s] = ctx->sb[s] * ctx->dt;
    P.drift[s] = ctx->sa[s] * ctx->dt;
  }
  {  // evaluation points: every non-zero drift leaves one; kicks at the step's first point follow the snapshot, the
     // kicks after the last drift precede the next one
    int cur = 0, np = 0;
    for (int s = 0; s < ctx->nstages; s++)
      if (ctx->sa[s] != 0.0) np++;
    P.npoints = np;
    for (int s = 0; s < ctx->nstages; s++) {
      const double b = ctx->sb[s] * ctx->dt;
      if (cur == 0) P.pt_post[0] += b;
      else if (cur == np) P.pt_pre[0] += b;
      else P.pt_pre[cur] += b;
      if (ctx->sa[s] != 0.0) P.pt_drift[cur++] = ctx->sa[s] * ctx->dt;
    }
  }
  for (int a = 0; a < F; a++) {
    const double sg = sqrt(ctx->gamma[a]);
    P.sg[a] = sg;
    P.isg[a] = 1.0 / sg;
    P.mu[a] = ctx->gamma[a] / ctx->mass[a];
    P.Peq[a] = chi ? chi[a] / sg : 0.0;
    P.Qeq[a] = chi ? chi[F + a] * sg : 0.0;
  }
  P.coef = ctx->d_coef;
  P.det_tol = ctx->det_tol;
  P.det_stride = ctx->det_stride;
  // thresholds of the static-order eliminations as IEEE high words (the kernel compares exponents + top mantissa bits)
  auto hi_word = [](double x) {
    unsigned long long u;
    memcpy(&u, &x, sizeof(u));
    return (unsigned)(u >> 32);
  };
  if (ctx->lu_growth_max < 0.0) {
    P.grow_k_max = P.grow_m_max = 0u;
  } else {
    P.grow_k_max = hi_word(ctx->lu_growth_max);
    P.grow_m_max = hi_word(ctx->lu_growth_max * ctx->lu_growth_max);
  }
}

// Equally spaced grid?  E_i = E_0 + i dE to within a few ulp of the largest |E|.
bool uniform_grid(const double *E, int k, double *e0, double *de) {
  *e0 = E[0];
  *de = k > 1 ? (E[k - 1] - E[0]) / (double)(k - 1) : 0.0;
  double emax = 0.0;
  for (int i = 0; i < k; i++) {
    if (!isfinite(E[i])) return false;
    emax = fmax(emax, fabs(E[i]));
  }
  const double tol = 8.0 * 2.220446049250313e-16 * emax;
  for (int i = 0; i < k; i++)
    if (fabs(E[i] - (*e0 + (double)i * *de)) > tol) return false;
  return true;
}

// Chirp-z plan: blocks of bsz = L - k + 1 time samples.
bool chirp_plan(int nsteps, int k, int *nblocks, int *bsz) {
  const long long b = (long long)SCI_CHIRP_L - k + 1;
  if (b < SCI_CHIRP_MIN_BLOCK) return false;
  const long long nb = ((long long)nsteps + 1 + b - 1) / b;
  if (nb > SCI_CHIRP_MAX_BLOCKS) return false;
  *nblocks = (int)nb;
  *bsz = (int)b;
  return true;
}

bool chirp_applies(const sc_ivr_ctx *ctx, const double *E, int k, double *e0, double *de, int *nblocks, int *bsz) {
  if (ctx->fourier_mode == 1) return false;
  if (!chirp_plan(ctx->nsteps, k, nblocks, bsz)) return false;
  return uniform_grid(E, k, e0, de);
}

// kernel A: one thread per trajectory for F <= SCI_TPT_MAXF, C modes per lane (cml_table.h) above
cudaError_t launch_kernel_a(const sc_ivr_ctx *ctx, const PropParams &P, cudaStream_t st) {
  if (ctx->F <= SCI_TPT_MAXF) {
    TptParams TP;
    TP.P = P;
    memcpy(TP.coef, ctx->tpt_coef, sizeof(TP.coef));
    return sci_tpt_launch_propagate(ctx->F, ctx->kind, TP, st);
  }
  return sci_cml_launch_propagate(ctx->F, ctx->kind, P, st);
}

struct StageTimer {
  sc_ivr_ctx *ctx;
  cudaStream_t st;
  bool on;
  StageTimer(sc_ivr_ctx *c, cudaStream_t s) : ctx(c), st(s), on(c->timing != 0) {
    if (on) {
      ctx->ev_used = 0;
      ctx->ev_slot.clear();
    }
  }
  void begin() {
    if (!on) return;
    if (ctx->ev.size() < ctx->ev_used + 2) {
      cudaEvent_t a = nullptr, b = nullptr;
      if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) {  // timing is a measurement aid: switch it off
        if (a) cudaEventDestroy(a);
        on = false;
        ctx->timing = 0;
        return;
      }
      ctx->ev.push_back(a);
      ctx->ev.push_back(b);
    }
    cudaEventRecord(ctx->ev[ctx->ev_used], st);
  }
  void end(int slot) {
    if (!on) return;
    cudaEventRecord(ctx->ev[ctx->ev_used + 1], st);
    ctx->ev_used += 2;
    ctx->ev_slot.push_back(slot);
  }
};

}  // namespace

extern "C" {

const char *sc_ivr_last_error(const sc_ivr_ctx *ctx) { return ctx ? ctx->err : g_create_err; }

sc_ivr_status sc_ivr_create(sc_ivr_ctx **out, int F, sc_ivr_pes_kind kind, const double *pes_coeffs, size_t n_coeffs,
                            const double *gamma, double dt, int nsteps, const sc_ivr_options *opt) {
  sc_ivr_ctx *ctx = nullptr;  // errors before allocation go to the thread-local message
  if (!out) return fail(ctx, SC_IVR_EINVAL, "out is NULL");
  *out = nullptr;
  if (!pes_coeffs || !gamma) return fail(ctx, SC_IVR_EINVAL, "pes_coeffs/gamma is NULL");
  if (F < 1) return fail(ctx, SC_IVR_EINVAL, "F = %d < 1", F);
  if (F > SC_IVR_MAX_F) return fail(ctx, SC_IVR_EUNSUPPORTED, "F = %d > SC_IVR_MAX_F = %d", F, SC_IVR_MAX_F);
  if (kind != SC_IVR_PES_MORSE1D && kind != SC_IVR_PES_QFF && kind != SC_IVR_PES_MORSE_UNCOUPLED)
    return fail(ctx, SC_IVR_EUNSUPPORTED, "unknown PES kind %d", (int)kind);
  if (kind == SC_IVR_PES_MORSE1D && F != 1) return fail(ctx, SC_IVR_EINVAL, "MORSE1D needs F = 1");
  if ((long)n_coeffs != n_coeffs_expected(F, kind))
    return fail(ctx, SC_IVR_EINVAL, "n_coeffs = %zu, expected %ld", n_coeffs, n_coeffs_expected(F, kind));
  if (!(dt > 0.0) || !isfinite(dt)) return fail(ctx, SC_IVR_EINVAL, "dt must be > 0");
  if (nsteps < 1) return fail(ctx, SC_IVR_EINVAL, "nsteps must be >= 1");
  for (size_t i = 0; i < n_coeffs; i++)
    if (!isfinite(pes_coeffs[i])) return fail(ctx, SC_IVR_EINVAL, "pes_coeffs[%zu] is not finite", i);
  for (int a = 0; a < F; a++)
    if (!(gamma[a] > 0.0) || !isfinite(gamma[a])) return fail(ctx, SC_IVR_EINVAL, "gamma[%d] must be > 0", a);
  int integrator = opt ? opt->integrator : 0;
  int det_stride = opt ? opt->det_stride : 1;
  double det_tol = opt ? opt->det_tol : 1e-6;
  double lu_growth_max = opt ? opt->lu_growth_max : 0.0;
  if (lu_growth_max == 0.0) lu_growth_max = 1e4;
  if (!(lu_growth_max < 1e100)) return fail(ctx, SC_IVR_EINVAL, "bad lu_growth_max");
  if (det_stride == 0) det_stride = 1;
  if (det_tol == 0.0) det_tol = 1e-6;
  if (det_stride < 1 || !(det_tol > 0.0)) return fail(ctx, SC_IVR_EINVAL, "bad det_stride/det_tol");
  if (integrator != 0 && integrator != 1) return fail(ctx, SC_IVR_EUNSUPPORTED, "unknown integrator %d", integrator);
  const int fourier_mode = opt ? opt->fourier_mode : 0;
  if (fourier_mode != 0 && fourier_mode != 1) return fail(ctx, SC_IVR_EUNSUPPORTED, "unknown fourier_mode %d", fourier_mode);

  int ndev = 0;
  cudaError_t ce = cudaGetDeviceCount(&ndev);
  if (ce != cudaSuccess || ndev < 1)
    return fail(ctx, SC_IVR_ECUDA, "no CUDA device (%s): this library has no CPU fallback",
                ce == cudaSuccess ? "device count 0" : cudaGetErrorString(ce));

  ctx = new (std::nothrow) sc_ivr_ctx();
  if (!ctx) return fail(nullptr, SC_IVR_ENOMEM, "out of host memory");
  ctx->F = F;
  ctx->kind = (int)kind;
  ctx->nsteps = nsteps;
  ctx->dt = dt;
  ctx->det_stride = det_stride;
  ctx->det_tol = det_tol;
  ctx->lu_growth_max = lu_growth_max;
  ctx->integrator = integrator;
  ctx->fourier_mode = fourier_mode;
  for (int a = 0; a < F; a++) {
    ctx->gamma[a] = gamma[a];
    ctx->mass[a] = (kind == SC_IVR_PES_QFF) ? 1.0 : pes_coeffs[4 * a + 3];
    if (!(ctx->mass[a] > 0.0)) {
      delete ctx;
      return fail(nullptr, SC_IVR_EINVAL, "mass[%d] must be > 0", a);
    }
  }
  if (integrator == 0) {  // velocity-Verlet as "kick b then drift a" stages (R10)
    ctx->nstages = 2;
    ctx->sb[0] = 0.5; ctx->sa[0] = 1.0;
    ctx->sb[1] = 0.5; ctx->sa[1] = 0.0;
  } else {  // 4-stage 4th-order symplectic composition (table of McLachlan & Atela)
    ctx->nstages = 4;
    const double b[4] = {0.1344961992774310892, -0.2248198030794208058, 0.7563200005156682911, 0.3340036032863214255};
    const double a[4] = {0.5153528374311229364, -0.085782019412973646, 0.4415830236164665242, 0.1288461583653841854};
    for (int s = 0; s < 4; s++) { ctx->sb[s] = b[s]; ctx->sa[s] = a[s]; }
  }
  sc_ivr_status rc = SC_IVR_OK;
  do {
    if (cudaGetDevice(&ctx->device) != cudaSuccess ||
        cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, ctx->device) != cudaSuccess) {
      rc = fail(nullptr, SC_IVR_ECUDA, "cannot query the CUDA device");
      break;
    }
    const bool cml = F > SCI_TPT_MAXF;
    if (cml && sci_cml_lanes(F) == 0) {
      rc = fail(nullptr, SC_IVR_EINVAL, "F = %d has no kernel (cml_table.h)", F);
      break;
    }
    const size_t nc = cml ? sci_cml_pack_coeffs(F, (int)kind, pes_coeffs, gamma, nullptr) : 0;
    std::vector<double> packed(nc + F);  // sqrt(gamma) rides behind the coefficients (for sc_ivr_eval_pes)
    if (cml) sci_cml_pack_coeffs(F, (int)kind, pes_coeffs, gamma, packed.data());
    for (int a = 0; a < F; a++) packed[nc + a] = sqrt(gamma[a]);
    ctx->n_coef = nc;
    if ((ce = cudaMalloc(&ctx->d_coef, sizeof(double) * (nc + F))) != cudaSuccess ||
        (ce = cudaMemcpy(ctx->d_coef, packed.data(), sizeof(double) * (nc + F), cudaMemcpyHostToDevice)) != cudaSuccess) {
      rc = fail(nullptr, SC_IVR_ECUDA, "coefficient upload: %s", cudaGetErrorString(ce));
      break;
    }
    if (F <= SCI_TPT_MAXF) {  // one thread per trajectory
      memset(ctx->tpt_coef, 0, sizeof(ctx->tpt_coef));
      sci_tpt_pack_coeffs(F, (int)kind, pes_coeffs, gamma, ctx->tpt_coef);
      ctx->wave = (long long)ctx->sm_count * sci_tpt_blocks_per_sm(F, (int)kind) * sci_tpt_traj_per_block();
    } else {
      ctx->wave = (long long)ctx->sm_count * sci_cml_traj_per_block(F);  // one CTA per SM
    }
  } while (0);
  if (rc != SC_IVR_OK) {
    sc_ivr_destroy(ctx);
    return rc;
  }
  *out = ctx;
  return SC_IVR_OK;
}

void sc_ivr_destroy(sc_ivr_ctx *ctx) {
  if (!ctx) return;
  if (ctx->d_coef) cudaFree(ctx->d_coef);
  for (cudaEvent_t e : ctx->ev)
    if (e) cudaEventDestroy(e);
  delete ctx;
}

long long sc_ivr_min_batch(const sc_ivr_ctx *ctx) { return ctx ? ctx->wave : 0; }

size_t sc_ivr_workspace_bytes(const sc_ivr_ctx *ctx, long long ntraj, int k, long long max_batch) {
  if (!ctx || ntraj < 1 || k < 1) return 0;
  return carve(ctx, ntraj, k, default_batch(ctx, ntraj, max_batch)).total;
}

size_t sc_ivr_host_staging_bytes(const sc_ivr_ctx *ctx, long long ntraj, int k) {
  if (!ctx || ntraj < 1 || k < 1) return 0;
  return align_up(sizeof(double) * 2 * (size_t)ctx->F * (size_t)ntraj, 256) + align_up(sizeof(double) * (size_t)ntraj, 256) +
         align_up(sizeof(double) * (size_t)k, 256);
}

void sc_ivr_set_timing(sc_ivr_ctx *ctx, int on) {
  if (ctx) ctx->timing = on;
}

sc_ivr_status sc_ivr_last_timings(sc_ivr_ctx *ctx, double out[6]) {
  if (!ctx || !out) return SC_IVR_EINVAL;
  if (ctx->ev_used >= 2) CU(cudaEventSynchronize(ctx->ev[ctx->ev_used - 1]));
  for (int i = 0; i < 5; i++) ctx->tms[i] = 0.0;
  for (size_t p = 0; p < ctx->ev_slot.size(); p++) {
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, ctx->ev[2 * p], ctx->ev[2 * p + 1]));
    ctx->tms[ctx->ev_slot[p]] += ms;
  }
  for (int i = 0; i < 6; i++) out[i] = ctx->tms[i];
  return SC_IVR_OK;
}

sc_ivr_status sc_ivr_fp64_probe(int mode, int iters, double *flops_out, double *ms_out) {
  sc_ivr_ctx *ctx = nullptr;
  if (!flops_out || !ms_out || iters < 1 || mode < 0 || mode % 10 > 4 || mode / 10 > 2)
    return fail(ctx, SC_IVR_EINVAL, "bad probe arguments (mode = kind 0..4 + 10 x warps per scheduler 0..2)");
  CU(sci_fp64_probe(mode, iters, flops_out, ms_out));
  return SC_IVR_OK;
}

sc_ivr_status sc_ivr_run(sc_ivr_ctx *ctx, const double *p0q0, const double *weights, long long ntraj, const double *chi,
                         const double *E, int k, double *I_out, long long *n_good_out, void *workspace,
                         size_t workspace_bytes, void *cuda_stream) {
  if (!ctx) return SC_IVR_EINVAL;
  if (sc_ivr_status ds = check_device(ctx)) return ds;
  if (!p0q0 || !chi || !E || !I_out || !workspace) return fail(ctx, SC_IVR_EINVAL, "NULL argument");
  if (ntraj < 1 || k < 1) return fail(ctx, SC_IVR_EINVAL, "ntraj and k must be >= 1");
  if (((uintptr_t)workspace & 255) != 0) return fail(ctx, SC_IVR_EINVAL, "workspace must be 256-byte aligned");
  for (int a = 0; a < 2 * ctx->F; a++)
    if (!isfinite(chi[a])) return fail(ctx, SC_IVR_EINVAL, "chi[%d] is not finite", a);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int F = ctx->F;

  // largest batch (whole kernel-A waves) whose workspace fits
  long long nbatch = default_batch(ctx, ntraj, 0);
  Carve cv = carve(ctx, ntraj, k, nbatch);
  while (cv.total > workspace_bytes && nbatch > ctx->wave) {
    long long nx = nbatch / 2 / ctx->wave * ctx->wave;
    if (nx < ctx->wave) nx = ctx->wave;
    nbatch = nx;
    cv = carve(ctx, ntraj, k, nbatch);
  }
  if (cv.total > workspace_bytes)
    return fail(ctx, SC_IVR_EINVAL, "workspace too small: %zu bytes given, %zu needed for the minimum batch of %lld", workspace_bytes,
                cv.total, nbatch);

  char *ws = (char *)workspace;
  double4 *raw = (double4 *)(ws + cv.off_raw);
  double2 *z = (double2 *)(ws + cv.off_z);
  double2 *W = (double2 *)(ws + cv.off_W);
  double *partial = (double *)(ws + cv.off_partial);
  unsigned char *good = (unsigned char *)(ws + cv.off_good);
  double *wg = (double *)(ws + cv.off_wg);
  double *E_dev = (double *)(ws + cv.off_E);
  long long *ngood = (long long *)(ws + cv.off_ngood);

  for (int i = 0; i < 6; i++) ctx->tms[i] = 0.0;
  StageTimer tm(ctx, st);
  double launches = 0;

  double2 *pc = (double2 *)(ws + cv.off_pc);
  double2 *hrow = (double2 *)(ws + cv.off_hrow);
  double2 *HpT = (double2 *)(ws + cv.off_HpT);
  double2 *yscr = (double2 *)(ws + cv.off_yscr);
  double e0 = 0.0, de = 0.0;
  int cblocks = 1, cbsz = 0;
  const bool chirp = chirp_applies(ctx, E, k, &e0, &de, &cblocks, &cbsz);
  const int chirp_grid = ctx->sm_count;
  tm.begin();
  if (chirp) {  // inner chirp, filter rows, filter spectra (one FFT per block)
    CU(sci_launch_chirp_tables(e0 * ctx->dt, de * ctx->dt, cv.rows, k, cblocks, cbsz, pc, hrow, st));
    CU(sci_launch_chirp_fft(1, hrow, SCI_CHIRP_L, SCI_CHIRP_L, 1, nullptr, nullptr, k, cv.kp, nullptr, HpT, cblocks, cbsz, nullptr, 1, st));
    launches += 1 + cblocks;
  } else {
    CU(cudaMemcpyAsync(E_dev, E, sizeof(double) * k, cudaMemcpyHostToDevice, st));
    CU(sci_launch_twiddle(E_dev, k, cv.kp, cv.zrows, ctx->dt, W, st));
    launches += 1;
  }
  tm.end(2);

  PropParams P;
  fill_prop_params(ctx, P, chi);
  P.p0q0 = p0q0;
  P.stride = ntraj;
  P.nsteps = ctx->nsteps;
  P.raw = raw;
  P.raw_stride = cv.nbatch;
  P.fb_count = (unsigned long long *)(ngood + 1);
  CU(cudaMemsetAsync(ngood + 1, 0, sizeof(long long), st));
  ctx->last_fallbacks = -1;

  long long tile0 = 0;
  for (long long j0 = 0; j0 < ntraj; j0 += nbatch) {
    const long long nb = (ntraj - j0 < nbatch) ? ntraj - j0 : nbatch;
    const long long zcols = round_up_ll(nb, SCI_TJ);
    P.j0 = j0;
    P.nb = nb;
    P.good = good + j0;
    tm.begin();
    CU(launch_kernel_a(ctx, P, st));
    tm.end(0);
    tm.begin();
    if (chirp) CU(sci_launch_zassemble_rows(raw, cv.nbatch, nb, ctx->nsteps, pc, z, cv.xstride, st));
    else CU(sci_launch_zassemble(raw, cv.nbatch, nb, ctx->nsteps, z, cv.nbp, zcols, cv.zrows, nullptr, st));
    tm.end(1);
    tm.begin();
    CU(sci_launch_weights(weights ? weights + j0 : nullptr, good + j0, nb, wg + j0, st));
    tm.end(4);
    tm.begin();
    if (chirp) {
      const int grid = nb < chirp_grid ? (int)nb : chirp_grid;
      CU(sci_launch_chirp_fft(0, z, cv.xstride, cv.rows, nb, HpT, wg + j0, k, cv.kp, partial + tile0 * cv.kp, nullptr, cblocks, cbsz, yscr, grid,
                              st));
      tile0 += grid;
    } else {
      CU(sci_launch_fourier(z, cv.nbp, zcols, cv.zrows, W, cv.kp, nb, wg + j0, partial + tile0 * cv.kp, nullptr, k, st));
      tile0 += zcols / SCI_TJ;
    }
    tm.end(3);
    launches += 4;
  }
  tm.begin();
  CU(sci_launch_count_good(good, ntraj, ngood, 0, st));
  const double T = (double)ctx->nsteps * ctx->dt;
  const double norm = ctx->dt * ctx->dt / (pow(2.0 * M_PI, F + 1) * T);  // Eq. 11 with R4's dt^2; 1/n_good on the device
  CU(sci_launch_final(partial, tile0, cv.kp, k, ngood, norm, I_out, st));
  tm.end(4);
  launches += 2;
  ctx->tms[5] = launches;

  if (n_good_out) {
    long long ng[2] = {0, 0};
    CU(cudaMemcpyAsync(ng, ngood, 2 * sizeof(long long), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    *n_good_out = ng[0];
    ctx->last_fallbacks = ng[1];
    if (ng[0] == 0) return fail(ctx, SC_IVR_ENOGOOD, "every trajectory was rejected");
  }
  return SC_IVR_OK;
}

long long sc_ivr_last_fallbacks(const sc_ivr_ctx *ctx) { return ctx ? ctx->last_fallbacks : -1; }

sc_ivr_status sc_ivr_run_host(sc_ivr_ctx *ctx, const double *p0q0, const double *weights, long long ntraj, const double *chi,
                              const double *E, int k, double *I_out, long long *n_good_out, void *workspace,
                              size_t workspace_bytes, void *cuda_stream) {
  if (!ctx) return SC_IVR_EINVAL;
  if (sc_ivr_status ds = check_device(ctx)) return ds;
  if (!p0q0 || !I_out || !workspace) return fail(ctx, SC_IVR_EINVAL, "NULL argument");
  if (ntraj < 1 || k < 1) return fail(ctx, SC_IVR_EINVAL, "ntraj and k must be >= 1");
  const size_t stg = sc_ivr_host_staging_bytes(ctx, ntraj, k);
  if (workspace_bytes < stg) return fail(ctx, SC_IVR_EINVAL, "workspace smaller than the host staging area");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  char *ws = (char *)workspace;
  const size_t n_pq = sizeof(double) * 2 * (size_t)ctx->F * (size_t)ntraj;
  double *d_pq = (double *)ws;
  double *d_w = (double *)(ws + align_up(n_pq, 256));
  double *d_I = (double *)((char *)d_w + align_up(sizeof(double) * (size_t)ntraj, 256));
  CU(cudaMemcpyAsync(d_pq, p0q0, n_pq, cudaMemcpyHostToDevice, st));
  if (weights) {
    const cudaError_t ce = cudaMemcpyAsync(d_w, weights, sizeof(double) * (size_t)ntraj, cudaMemcpyHostToDevice, st);
    if (ce != cudaSuccess) {
      cudaStreamSynchronize(st);  // the copy of p0q0 may still read the caller's pinned buffer
      return fail(ctx, SC_IVR_ECUDA, "copy of the weights: %s", cudaGetErrorString(ce));
    }
  }
  long long ng = 0;
  sc_ivr_status rc = sc_ivr_run(ctx, d_pq, weights ? d_w : nullptr, ntraj, chi, E, k, d_I, &ng, ws + stg, workspace_bytes - stg, st);
  if (n_good_out) *n_good_out = ng;
  if (rc != SC_IVR_OK && rc != SC_IVR_ENOGOOD) {
    cudaStreamSynchronize(st);  // no copy from the caller's host buffers is left in flight when an error is returned
    return rc;
  }
  CU(cudaMemcpyAsync(I_out, d_I, sizeof(double) * (size_t)k, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  return rc;
}

size_t sc_ivr_propagate_workspace_bytes(const sc_ivr_ctx *ctx, long long ntraj, int nsteps_run) {
  if (!ctx || ntraj < 1 || nsteps_run < 0) return 0;
  return align_up(sizeof(double4) * (size_t)(nsteps_run + 1) * (size_t)ntraj, 256);
}

sc_ivr_status sc_ivr_propagate(sc_ivr_ctx *ctx, const double *p0q0, long long ntraj, int nsteps_run, const double *chi,
                               double *pq_out, double *S_out, double *M_out, double *theta_out, unsigned char *good_out,
                               double *z_out, void *workspace, size_t workspace_bytes, void *cuda_stream) {
  if (!ctx) return SC_IVR_EINVAL;
  if (sc_ivr_status ds = check_device(ctx)) return ds;
  if (!p0q0) return fail(ctx, SC_IVR_EINVAL, "p0q0 is NULL");
  if (ntraj < 1 || nsteps_run < 0) return fail(ctx, SC_IVR_EINVAL, "ntraj must be >= 1 and nsteps_run >= 0");
  const bool need_raw = theta_out || z_out;
  if (need_raw && (!workspace || workspace_bytes < sc_ivr_propagate_workspace_bytes(ctx, ntraj, nsteps_run)))
    return fail(ctx, SC_IVR_EINVAL, "workspace too small for theta_out/z_out");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  PropParams P;
  fill_prop_params(ctx, P, chi);
  P.p0q0 = p0q0;
  P.stride = ntraj;
  P.j0 = 0;
  P.nb = ntraj;
  P.nsteps = nsteps_run;
  P.raw = need_raw ? (double4 *)workspace : nullptr;
  P.raw_stride = ntraj;
  P.good = good_out;
  P.pq_out = pq_out;
  P.S_out = S_out;
  P.M_out = M_out;
  CU(launch_kernel_a(ctx, P, st));
  if (need_raw)
    CU(sci_launch_zassemble((const double4 *)workspace, ntraj, ntraj, nsteps_run, (double2 *)z_out, ntraj, ntraj, nsteps_run + 1,
                            theta_out, st));
  return SC_IVR_OK;
}

sc_ivr_status sc_ivr_assemble_z(sc_ivr_ctx *ctx, const double *raw, long long n, int nsteps_run, double *z_out, double *theta_out,
                                void *cuda_stream) {
  if (!ctx) return SC_IVR_EINVAL;
  if (sc_ivr_status ds = check_device(ctx)) return ds;
  if (!raw || !z_out) return fail(ctx, SC_IVR_EINVAL, "NULL argument");
  if (n < 1 || nsteps_run < 0) return fail(ctx, SC_IVR_EINVAL, "n must be >= 1 and nsteps_run >= 0");
  CU(sci_launch_zassemble((const double4 *)raw, n, n, nsteps_run, (double2 *)z_out, n, n, nsteps_run + 1, theta_out,
                          (cudaStream_t)cuda_stream));
  return SC_IVR_OK;
}

sc_ivr_status sc_ivr_eval_pes(sc_ivr_ctx *ctx, const double *q, long long n, double *V_out, double *g_out, double *H_out,
                              void *cuda_stream) {
  if (!ctx) return SC_IVR_EINVAL;
  if (sc_ivr_status ds = check_device(ctx)) return ds;
  if (!q || !V_out || !g_out || !H_out) return fail(ctx, SC_IVR_EINVAL, "NULL argument");
  if (n < 1) return fail(ctx, SC_IVR_EINVAL, "n must be >= 1");
  if (ctx->F <= SCI_TPT_MAXF) {
    TptParams TP;
    fill_prop_params(ctx, TP.P, nullptr);
    memcpy(TP.coef, ctx->tpt_coef, sizeof(TP.coef));
    CU(sci_tpt_launch_eval_pes(ctx->F, ctx->kind, TP, q, n, V_out, g_out, H_out, (cudaStream_t)cuda_stream));
    return SC_IVR_OK;
  }
  CU(sci_cml_launch_eval_pes(ctx->F, ctx->kind, ctx->d_coef, ctx->d_coef + ctx->n_coef, q, n, V_out, g_out, H_out,
                             (cudaStream_t)cuda_stream));
  return SC_IVR_OK;
}

size_t sc_ivr_fourier_workspace_bytes(const sc_ivr_ctx *ctx, long long n, int k) {
  if (!ctx || n < 1 || k < 1) return 0;
  const size_t zrows = (size_t)round_up_ll(ctx->nsteps + 1, SCI_KC), ncp = (size_t)round_up_ll(n, SCI_TJ);
  const size_t kp = (size_t)round_up_ll(k, SCI_TI);
  return align_up(sizeof(double2) * zrows * ncp, 256) + align_up(sizeof(double2) * zrows * kp, 256) + align_up(sizeof(double) * k, 256);
}

sc_ivr_status sc_ivr_fourier(sc_ivr_ctx *ctx, const double *zin, long long n, const double *E, int k, double *A_out,
                             void *workspace, size_t workspace_bytes, void *cuda_stream) {
  if (!ctx) return SC_IVR_EINVAL;
  if (sc_ivr_status ds = check_device(ctx)) return ds;
  if (!zin || !E || !A_out || !workspace) return fail(ctx, SC_IVR_EINVAL, "NULL argument");
  if (n < 1 || k < 1) return fail(ctx, SC_IVR_EINVAL, "n and k must be >= 1");
  if (workspace_bytes < sc_ivr_fourier_workspace_bytes(ctx, n, k)) return fail(ctx, SC_IVR_EINVAL, "workspace too small");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int rows = ctx->nsteps + 1;
  const int zrows = (int)round_up_ll(rows, SCI_KC), kp = (int)round_up_ll(k, SCI_TI);
  const long long ncp = round_up_ll(n, SCI_TJ);
  char *ws = (char *)workspace;
  double2 *z = (double2 *)ws;
  double2 *W = (double2 *)(ws + align_up(sizeof(double2) * (size_t)zrows * (size_t)ncp, 256));
  double *E_dev = (double *)((char *)W + align_up(sizeof(double2) * (size_t)zrows * (size_t)kp, 256));
  CU(cudaMemsetAsync(z, 0, sizeof(double2) * (size_t)zrows * (size_t)ncp, st));
  CU(cudaMemcpy2DAsync(z, sizeof(double2) * ncp, zin, sizeof(double2) * n, sizeof(double2) * n, rows, cudaMemcpyDeviceToDevice, st));
  CU(cudaMemcpyAsync(E_dev, E, sizeof(double) * k, cudaMemcpyHostToDevice, st));
  CU(sci_launch_twiddle(E_dev, k, kp, zrows, ctx->dt, W, st));
  CU(sci_launch_fourier(z, ncp, ncp, zrows, W, kp, n, nullptr, nullptr, (double2 *)A_out, k, st));
  return SC_IVR_OK;
}

size_t sc_ivr_fourier_power_workspace_bytes(const sc_ivr_ctx *ctx, long long n, int k) {
  if (!ctx || n < 1 || k < 1) return 0;
  const size_t rows = (size_t)ctx->nsteps + 1, xstride = (size_t)round_up_ll((long long)rows, 32);
  return align_up(sizeof(double2) * xstride * (size_t)n, 256) + align_up(sizeof(double2) * rows, 256) +
         2 * align_up(sizeof(double2) * SCI_CHIRP_L * SCI_CHIRP_MAX_BLOCKS, 256) +
         align_up(sizeof(double2) * SCI_CHIRP_L * (size_t)ctx->sm_count, 256);
}

sc_ivr_status sc_ivr_fourier_power(sc_ivr_ctx *ctx, const double *zin, long long n, const double *E, int k, double *P_out,
                                   void *workspace, size_t workspace_bytes, void *cuda_stream) {
  if (!ctx) return SC_IVR_EINVAL;
  if (sc_ivr_status ds = check_device(ctx)) return ds;
  if (!zin || !E || !P_out || !workspace) return fail(ctx, SC_IVR_EINVAL, "NULL argument");
  if (n < 1 || k < 1) return fail(ctx, SC_IVR_EINVAL, "n and k must be >= 1");
  if (workspace_bytes < sc_ivr_fourier_power_workspace_bytes(ctx, n, k)) return fail(ctx, SC_IVR_EINVAL, "workspace too small");
  double e0 = 0.0, de = 0.0;
  int cblocks = 1, cbsz = 0;
  if (!chirp_plan(ctx->nsteps, k, &cblocks, &cbsz) || !uniform_grid(E, k, &e0, &de))
    return fail(ctx, SC_IVR_EUNSUPPORTED, "chirp-z needs an equally spaced grid, k <= %d and at most %d blocks of %d - k + 1 samples",
                SCI_CHIRP_L - SCI_CHIRP_MIN_BLOCK + 1, SCI_CHIRP_MAX_BLOCKS, SCI_CHIRP_L);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int rows = ctx->nsteps + 1;
  const long long xstride = round_up_ll(rows, 32);
  char *ws = (char *)workspace;
  double2 *x = (double2 *)ws;
  double2 *pc = (double2 *)(ws + align_up(sizeof(double2) * (size_t)xstride * (size_t)n, 256));
  double2 *hrow = (double2 *)((char *)pc + align_up(sizeof(double2) * (size_t)rows, 256));
  double2 *HpT = (double2 *)((char *)hrow + align_up(sizeof(double2) * SCI_CHIRP_L * SCI_CHIRP_MAX_BLOCKS, 256));
  double2 *yscr = (double2 *)((char *)HpT + align_up(sizeof(double2) * SCI_CHIRP_L * SCI_CHIRP_MAX_BLOCKS, 256));
  CU(sci_launch_chirp_tables(e0 * ctx->dt, de * ctx->dt, rows, k, cblocks, cbsz, pc, hrow, st));
  CU(sci_launch_chirp_fft(1, hrow, SCI_CHIRP_L, SCI_CHIRP_L, 1, nullptr, nullptr, k, k, nullptr, HpT, cblocks, cbsz, nullptr, 1, st));
  CU(sci_launch_rows_from_z((const double2 *)zin, n, rows, pc, x, xstride, st));
  const int grid = n < ctx->sm_count ? (int)n : ctx->sm_count;
  CU(sci_launch_chirp_fft(2, x, xstride, rows, n, HpT, nullptr, k, k, P_out, nullptr, cblocks, cbsz, yscr, grid, st));
  return SC_IVR_OK;
}

}  // extern "C"

namespace {
struct CarveMulti {
  long long nbatch, xstride;
  int rows, kp;
  long long tiles_per_chi;  // partial rows per reference state
  size_t off_raw, off_pq, off_ov, off_x, off_partial, off_good, off_wg, off_ngood, off_pc, off_hrow, off_HpT, off_yscr, off_chis, off_eps, total;
};
CarveMulti carve_multi(const sc_ivr_ctx *ctx, long long ntraj, int k, int ncs, long long nbatch) {
  CarveMulti c;
  c.nbatch = nbatch;
  c.rows = ctx->nsteps + 1;
  c.xstride = round_up_ll(c.rows, 32);
  c.kp = (int)round_up_ll(k, SCI_TI);
  const long long nbatches = (ntraj + nbatch - 1) / nbatch;
  c.tiles_per_chi = nbatches * ctx->sm_count;
  size_t o = 0;
  c.off_raw = o; o = align_up(o + sizeof(double4) * (size_t)c.rows * (size_t)nbatch, 256);
  c.off_pq = o; o = align_up(o + sizeof(double2) * (size_t)c.rows * (size_t)ctx->F * (size_t)nbatch, 256);
  c.off_ov = o; o = align_up(o + sizeof(double2) * (size_t)c.rows * (size_t)(ncs + 1) * (size_t)nbatch, 256);
  c.off_x = o; o = align_up(o + sizeof(double2) * (size_t)c.xstride * (size_t)nbatch, 256);
  c.off_partial = o; o = align_up(o + sizeof(double) * 16 * (size_t)c.tiles_per_chi * (size_t)c.kp, 256);
  c.off_good = o; o = align_up(o + (size_t)ntraj, 256);
  c.off_wg = o; o = align_up(o + sizeof(double) * (size_t)ntraj, 256);
  c.off_ngood = o; o = align_up(o + 64, 256);
  c.off_pc = o; o = align_up(o + sizeof(double2) * (size_t)c.rows, 256);
  c.off_hrow = o; o = align_up(o + sizeof(double2) * SCI_CHIRP_L * SCI_CHIRP_MAX_BLOCKS, 256);
  c.off_HpT = o; o = align_up(o + sizeof(double2) * SCI_CHIRP_L * SCI_CHIRP_MAX_BLOCKS, 256);
  c.off_yscr = o; o = align_up(o + sizeof(double2) * SCI_CHIRP_L * (size_t)ctx->sm_count, 256);
  c.off_chis = o; o = align_up(o + sizeof(double) * 16 * 2 * SCI_MAXF, 256);
  c.off_eps = o; o = align_up(o + sizeof(double) * 16 * 16 * 2, 256);
  c.total = o;
  return c;
}
}  // namespace

extern "C" {

size_t sc_ivr_multi_workspace_bytes(const sc_ivr_ctx *ctx, long long ntraj, int k, int ncs, long long max_batch) {
  if (!ctx || ntraj < 1 || k < 1 || ncs < 1 || ncs > 16) return 0;
  return carve_multi(ctx, ntraj, k, ncs, default_batch(ctx, ntraj, max_batch > 0 ? max_batch : 32768)).total;
}

sc_ivr_status sc_ivr_run_multi(sc_ivr_ctx *ctx, const double *p0q0, const double *weights, long long ntraj, const double *chis,
                               int ncs, const double *eps, int nchi, const double *E, int k, double *I_out,
                               long long *n_good_out, void *workspace, size_t workspace_bytes, void *cuda_stream) {
  if (!ctx) return SC_IVR_EINVAL;
  if (sc_ivr_status ds = check_device(ctx)) return ds;
  if (!p0q0 || !chis || !eps || !E || !I_out || !workspace) return fail(ctx, SC_IVR_EINVAL, "NULL argument");
  if (ntraj < 1 || k < 1) return fail(ctx, SC_IVR_EINVAL, "ntraj and k must be >= 1");
  if (ncs < 1 || ncs > 16 || nchi < 1 || nchi > 16) return fail(ctx, SC_IVR_EINVAL, "ncs and nchi must be in 1..16");
  if (((uintptr_t)workspace & 255) != 0) return fail(ctx, SC_IVR_EINVAL, "workspace must be 256-byte aligned");
  const int F = ctx->F;
  for (int i = 0; i < ncs * 2 * F; i++)
    if (!isfinite(chis[i])) return fail(ctx, SC_IVR_EINVAL, "chis[%d] is not finite", i);
  for (int i = 0; i < nchi * ncs * 2; i++)
    if (!isfinite(eps[i])) return fail(ctx, SC_IVR_EINVAL, "eps[%d] is not finite", i);
  double e0 = 0.0, de = 0.0;
  int cblocks = 1, cbsz = 0;
  if (!chirp_plan(ctx->nsteps, k, &cblocks, &cbsz) || !uniform_grid(E, k, &e0, &de))
    return fail(ctx, SC_IVR_EUNSUPPORTED, "sc_ivr_run_multi needs an equally spaced grid within the chirp-z limits");
  cudaStream_t st = (cudaStream_t)cuda_stream;

  long long nbatch = default_batch(ctx, ntraj, 32768);
  CarveMulti cv = carve_multi(ctx, ntraj, k, ncs, nbatch);
  while (cv.total > workspace_bytes && nbatch > ctx->wave) {
    long long nx = nbatch / 2 / ctx->wave * ctx->wave;
    if (nx < ctx->wave) nx = ctx->wave;
    nbatch = nx;
    cv = carve_multi(ctx, ntraj, k, ncs, nbatch);
  }
  if (cv.total > workspace_bytes)
    return fail(ctx, SC_IVR_EINVAL, "workspace too small: %zu bytes given, %zu needed for the minimum batch of %lld", workspace_bytes,
                cv.total, nbatch);
  char *ws = (char *)workspace;
  double4 *raw = (double4 *)(ws + cv.off_raw);
  double2 *ovph = (double2 *)(ws + cv.off_ov);
  double2 *pqs = (double2 *)(ws + cv.off_pq);
  double2 *x = (double2 *)(ws + cv.off_x);
  double *partial = (double *)(ws + cv.off_partial);
  unsigned char *good = (unsigned char *)(ws + cv.off_good);
  double *wg = (double *)(ws + cv.off_wg);
  long long *ngood = (long long *)(ws + cv.off_ngood);
  double2 *pc = (double2 *)(ws + cv.off_pc);
  double2 *hrow = (double2 *)(ws + cv.off_hrow);
  double2 *HpT = (double2 *)(ws + cv.off_HpT);
  double2 *yscr = (double2 *)(ws + cv.off_yscr);
  double *chis_dev = (double *)(ws + cv.off_chis);
  double *eps_dev = (double *)(ws + cv.off_eps);

  // reference coherent states in reduced coordinates (P_eq then Q_eq per state); the copies are synchronous-safe
  // because the host arrays below live until the stream is synchronised at the end of this call
  std::vector<double> chr((size_t)ncs * 2 * F);
  for (int m = 0; m < ncs; m++)
    for (int a = 0; a < F; a++) {
      const double sg = sqrt(ctx->gamma[a]);
      chr[(size_t)(2 * m) * F + a] = chis[(size_t)m * 2 * F + a] / sg;
      chr[(size_t)(2 * m + 1) * F + a] = chis[(size_t)m * 2 * F + F + a] * sg;
    }
  CU(cudaMemcpyAsync(chis_dev, chr.data(), sizeof(double) * chr.size(), cudaMemcpyHostToDevice, st));
  CU(cudaMemcpyAsync(eps_dev, eps, sizeof(double) * (size_t)nchi * ncs * 2, cudaMemcpyHostToDevice, st));
  CU(sci_launch_chirp_tables(e0 * ctx->dt, de * ctx->dt, cv.rows, k, cblocks, cbsz, pc, hrow, st));
  CU(sci_launch_chirp_fft(1, hrow, SCI_CHIRP_L, SCI_CHIRP_L, 1, nullptr, nullptr, k, cv.kp, nullptr, HpT, cblocks, cbsz, nullptr, 1, st));

  PropParams P;
  fill_prop_params(ctx, P, nullptr);
  P.p0q0 = p0q0;
  P.stride = ntraj;
  P.nsteps = ctx->nsteps;
  P.raw = raw;
  P.raw_stride = cv.nbatch;
  P.pq_steps = pqs;
  P.raw_plain = 1;

  long long tile0 = 0;
  for (long long j0 = 0; j0 < ntraj; j0 += nbatch) {
    const long long nb = (ntraj - j0 < nbatch) ? ntraj - j0 : nbatch;
    P.j0 = j0;
    P.nb = nb;
    P.good = good + j0;
    CU(launch_kernel_a(ctx, P, st));
    CU(sci_launch_weights(weights ? weights + j0 : nullptr, good + j0, nb, wg + j0, st));
    const int grid = nb < ctx->sm_count ? (int)nb : ctx->sm_count;
    CU(sci_launch_overlap_phase(raw, pqs, cv.nbatch, nb, ctx->nsteps, F, chis_dev, ncs, pc, ovph, st));
    for (int n = 0; n < nchi; n++) {
      CU(sci_launch_combine_rows(ovph, cv.nbatch, nb, ctx->nsteps, eps_dev + (size_t)n * ncs * 2, ncs, x, cv.xstride, st));
      CU(sci_launch_chirp_fft(0, x, cv.xstride, cv.rows, nb, HpT, wg + j0, k, cv.kp,
                              partial + ((size_t)n * cv.tiles_per_chi + tile0) * cv.kp, nullptr, cblocks, cbsz, yscr, grid, st));
    }
    tile0 += grid;
  }
  CU(sci_launch_count_good(good, ntraj, ngood, 0, st));
  const double T = (double)ctx->nsteps * ctx->dt;
  const double norm = ctx->dt * ctx->dt / (pow(2.0 * M_PI, F + 1) * T);
  for (int n = 0; n < nchi; n++)
    CU(sci_launch_final(partial + (size_t)n * cv.tiles_per_chi * cv.kp, tile0, cv.kp, k, ngood, norm, I_out + (size_t)n * k, st));
  long long ng = 0;
  CU(cudaMemcpyAsync(&ng, ngood, sizeof(long long), cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  if (n_good_out) *n_good_out = ng;
  if (ng == 0) return fail(ctx, SC_IVR_ENOGOOD, "every trajectory was rejected");
  return SC_IVR_OK;
}

}  // extern "C"
