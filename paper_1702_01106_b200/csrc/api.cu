// api.cu -- the C ABI of include/grim.h: context, argument checking, stage sequencing.  Host code only; every
// step of the hot path runs in the kernels of kernels_*.cu.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <string>
#include <vector>

#include "../../include/grim.h"
#include "grim_internal.h"

using namespace grim;

// grim_invert_primitives: Newton iterations per sweep over the compacted active set (first sweep, later sweeps)
static constexpr int SWEEP_FIRST = 4, SWEEP_REST = 4;

struct KernelSpan {
  int kclass, launches;
  cudaEvent_t e0, e1;
};

struct grim_ctx {
  grim_grid_desc d;
  GridView gv;
  cudaStream_t stream;
  int metric_set;
  // geometry tables
  double *geomC, *geomF[3], *conn;
  // scratch
  double *C, *G;               // stage constant, EMHD gradient terms
  double *Fface, *cface;       // face fluxes (3 x N x Zg), face speeds (3 x Zg)
  double *emf;                 // edge fields (3 x Zg), flux-CT only
  double *Ph, *Pnew;           // stage buffers
  double *resnorm;
  int32_t *status, *iters;
  Counters *cnt;               // device
  StatsDev *stats;             // device, 2 stages
  double *probe_sink;
  long long *list[2];          // inversion active lists
  long long list_cap[2];   // capacity, in zones, of list[0] (stage sweeps and inversion) and list[1] (inversion only)
  double *hostP;               // staging for the *_host entry points
  cudaStream_t s_in, s_out;    // copy streams of the pipelined grim_timestep_host
  cudaStream_t s_st2;          // its second compute stream (stage 2 of a slab beside stage 1 of a later one)
  std::vector<cudaEvent_t> ev_in, ev_done, ev_s1;
  double *invbuf;              // U, P, resnorm, iters, status of grim_invert_primitives_host
  long long invbuf_nz;
  int64_t launches;
  int last_host_mode;          // what the last grim_timestep_host call did: GRIM_HOST_MODE_*
  int no_pipeline;             // GRIM_HOST_PIPELINE in the environment: 1 = "0" (never), -1 = "1" (always), 0 = unset
  // sweep policy of solve_stage: the deferred-zone counts of the recent sweep-mode solves arrive asynchronously in
  // pinned host memory; a run whose solves never defer a zone (smooth data) goes back to single launches and probes again
  // every SWEEP_PROBE solves
  unsigned long long *sweep_counts;  // pinned, SWEEP_RING entries
  cudaEvent_t sweep_ev[4];
  int sweep_pending[4];
  int sweep_slot, sweep_quiet, sweep_skip;
  // optional per-kernel-class timing (grim_set_timing): event pairs recorded around the launches
  int timing;
  std::vector<KernelSpan> spans;
  double class_ms[GRIM_NKCLASS];
  int64_t class_n[GRIM_NKCLASS];
  std::string err;
};

// records an event pair around the launches enqueued by `body` when timing is on
template <class F>
static int timed(grim_ctx *c, int kclass, F body, cudaStream_t on = nullptr) {
  if (!c->timing) return body();
  if (!on) on = c->stream;
  KernelSpan sp;
  sp.kclass = kclass;
  cudaEventCreate(&sp.e0);
  cudaEventCreate(&sp.e1);
  cudaEventRecord(sp.e0, on);
  int n = body();
  cudaEventRecord(sp.e1, on);
  sp.launches = n;
  c->spans.push_back(sp);
  return n;
}

static void drain_spans(grim_ctx *c) {
  for (auto &sp : c->spans) {
    cudaEventSynchronize(sp.e1);
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, sp.e0, sp.e1) == cudaSuccess) {
      c->class_ms[sp.kclass] += ms;
      c->class_n[sp.kclass] += sp.launches;
    }
    cudaEventDestroy(sp.e0);
    cudaEventDestroy(sp.e1);
  }
  c->spans.clear();
}

static std::string g_init_error;

// the context-free entry point (kernels_newton.cu) reports through grim_last_error(NULL) too
namespace grim {
void set_global_error(const char *msg) { g_init_error = msg ? msg : ""; }
}  // namespace grim

static int fail(grim_ctx *c, int code, const std::string &msg) {
  if (c) c->err = msg;
  else g_init_error = msg;
  return code;
}

#define CU(call)                                                                                       \
  do {                                                                                                 \
    cudaError_t e_ = (call);                                                                           \
    if (e_ != cudaSuccess)                                                                             \
      return fail(c, e_ == cudaErrorMemoryAllocation ? GRIM_ENOMEM : GRIM_ECUDA,                       \
                  std::string(#call) + ": " + cudaGetErrorString(e_));                                 \
  } while (0)

static int check_launch(grim_ctx *c, const char *what) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(c, GRIM_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
  return GRIM_OK;
}

extern "C" int grim_version(void) { return GRIM_VERSION; }

extern "C" const char *grim_last_error(const grim_ctx *c) { return c ? c->err.c_str() : g_init_error.c_str(); }

extern "C" int64_t grim_launch_count(const grim_ctx *c) { return c ? c->launches : 0; }

extern "C" int grim_set_timing(grim_ctx *c, int32_t on) {
  if (!c) return GRIM_EINVAL;
  cudaSetDevice(c->d.device);
  drain_spans(c);
  c->timing = on ? 1 : 0;
  if (on)
    for (int k = 0; k < GRIM_NKCLASS; k++) { c->class_ms[k] = 0.0; c->class_n[k] = 0; }
  return GRIM_OK;
}

extern "C" int grim_get_timing(grim_ctx *c, double *ms, int64_t *launches) {
  if (!c) return GRIM_EINVAL;
  cudaSetDevice(c->d.device);
  drain_spans(c);
  for (int k = 0; k < GRIM_NKCLASS; k++) {
    if (ms) ms[k] = c->class_ms[k];
    if (launches) launches[k] = c->class_n[k];
  }
  return GRIM_OK;
}

extern "C" int64_t grim_zones_padded(const grim_ctx *c, int32_t extents[3]) {
  if (!c) return 0;
  if (extents)
    for (int a = 0; a < 3; a++) extents[a] = c->gv.sz[a];
  return c->gv.zg;
}

extern "C" void grim_free(grim_ctx *c) {
  if (!c) return;
  cudaSetDevice(c->d.device);
  cudaStreamSynchronize(c->stream);
  drain_spans(c);
  void *ptrs[] = {c->geomC, c->geomF[0], c->geomF[1], c->geomF[2], c->conn, c->C, c->G, c->Fface, c->cface,
                  c->emf, c->Ph, c->Pnew, c->resnorm, c->status, c->iters, c->cnt, c->stats, c->probe_sink,
                  c->list[0], c->list[1], c->hostP, c->invbuf};
  for (void *p : ptrs)
    if (p) cudaFree(p);
  for (auto e : c->ev_in) cudaEventDestroy(e);
  for (auto e : c->ev_done) cudaEventDestroy(e);
  for (auto e : c->ev_s1) cudaEventDestroy(e);
  if (c->s_st2) cudaStreamDestroy(c->s_st2);
  if (c->sweep_counts) {
    cudaFreeHost(c->sweep_counts);
    for (int q = 0; q < 4; q++) cudaEventDestroy(c->sweep_ev[q]);
  }
  if (c->s_in) cudaStreamDestroy(c->s_in);
  if (c->s_out) cudaStreamDestroy(c->s_out);
  delete c;
}

extern "C" int grim_init_grid(grim_ctx **out, const grim_grid_desc *d) {
  grim_ctx *c = nullptr;
  if (!out || !d) return fail(c, GRIM_EINVAL, "grim_init_grid: null argument");
  *out = nullptr;
  if (d->dim < 1 || d->dim > 3) return fail(c, GRIM_EINVAL, "dim must be 1, 2 or 3");
  if (d->model != GRIM_IDEAL && d->model != GRIM_EMHD) return fail(c, GRIM_EINVAL, "model must be 8 or 10");
  if (d->recon != GRIM_MINMOD && d->recon != GRIM_MP5) return fail(c, GRIM_EINVAL, "unknown reconstruction");
  if (d->riemann != GRIM_LLF && d->riemann != GRIM_HLLE)
    return fail(c, GRIM_EINVAL, "riemann must be GRIM_LLF (eq 17) or GRIM_HLLE (eq 18)");
  const int nn[3] = {d->n1, d->n2, d->n3};
  const int need = d->recon == GRIM_MP5 ? 3 : 2;
  if (d->ng < need) return fail(c, GRIM_EINVAL, "ghost depth too small for the reconstruction");
  for (int a = 0; a < 3; a++) {
    if (nn[a] < 1) return fail(c, GRIM_EINVAL, "zone counts must be positive");
    if (a >= d->dim && nn[a] != 1) return fail(c, GRIM_EINVAL, "inactive directions must have one zone");
    if (a < d->dim && nn[a] < d->ng) return fail(c, GRIM_EINVAL, "active directions need at least ng zones");
    if (a < d->dim && !(d->xend[a] > d->xstart[a])) return fail(c, GRIM_EINVAL, "empty coordinate extent");
    for (int s = 0; s < 2; s++)
      if (d->bc[a][s] < 0 || d->bc[a][s] > 3) return fail(c, GRIM_EINVAL, "unknown boundary condition");
  }
  if (!(d->gamma > 1.0)) return fail(c, GRIM_EINVAL, "adiabatic index must exceed 1");
  if (!(d->limiter_theta >= 1.0 && d->limiter_theta <= 2.0)) return fail(c, GRIM_EINVAL, "limiter_theta outside [1,2]");
  if (!(d->fd_eps > 0.0) || d->kmax < 0 || d->lsmax < 0) return fail(c, GRIM_EINVAL, "bad solver parameters");
  if (d->closure != GRIM_CLOSURE_CS2TAU && d->closure != GRIM_CLOSURE_CONST)
    return fail(c, GRIM_EINVAL, "unknown closure");
  if (d->model == GRIM_EMHD && !(d->tau_mode == GRIM_TAU_R32 || d->tau > 0.0))
    return fail(c, GRIM_EINVAL, "tau_R must be positive");

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
    return fail(c, GRIM_ECUDA, "no CUDA device: this library has no CPU fallback");
  if (d->device < 0 || d->device >= ndev) return fail(c, GRIM_EINVAL, "device ordinal out of range");
  if (cudaSetDevice(d->device) != cudaSuccess) return fail(c, GRIM_ECUDA, "cudaSetDevice failed");
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, d->device) != cudaSuccess) return fail(c, GRIM_ECUDA, "no device properties");
  if (prop.major != 10) return fail(c, GRIM_ECUDA, "kernels are built for sm_100a only");

  c = new grim_ctx();
  c->d = *d;
  c->stream = (cudaStream_t)d->stream;
  c->metric_set = 0;
  c->launches = 0;
  c->s_in = c->s_out = c->s_st2 = nullptr;
  {
    const char *e = getenv("GRIM_HOST_PIPELINE");  // 0: never; 1: whenever the grid allows; unset: large grids only
    c->no_pipeline = (e && e[0] == '0') ? 1 : (e && e[0] == '1') ? -1 : 0;
  }
  c->timing = 0;
  for (int k = 0; k < GRIM_NKCLASS; k++) { c->class_ms[k] = 0.0; c->class_n[k] = 0; }
  GridView &gv = c->gv;
  memset(&gv, 0, sizeof(gv));
  gv.dim = d->dim;
  gv.nvar = d->model;
  gv.recon = d->recon;
  gv.riemann = d->riemann;
  gv.metric = -1;
  gv.nint = 1;
  gv.zg = 1;
  for (int a = 0; a < 3; a++) {
    gv.n[a] = nn[a];
    gv.ngd[a] = (a < d->dim) ? d->ng : 0;
    gv.sz[a] = gv.n[a] + 2 * gv.ngd[a];
    gv.dx[a] = (d->xend[a] - d->xstart[a]) / gv.n[a];  // L70
    gv.idx[a] = 1.0 / gv.dx[a];
    gv.xstart[a] = d->xstart[a];
    gv.nint *= gv.n[a];
    gv.zg *= gv.sz[a];
  }
  gv.n2d = (long long)gv.sz[0] * gv.sz[1];
  gv.theta = d->limiter_theta;
  gv.m.gam = d->gamma;
  gv.m.gm1 = d->gamma - 1.0;
  gv.m.phi = d->phi;
  gv.m.psi = d->psi;
  gv.m.closure = d->closure ? 1 : 0;
  gv.tau_const = d->tau;
  gv.sp.fd_eps = d->fd_eps;
  gv.sp.eps_bt = d->eps_bt;
  gv.sp.atol = d->atol;
  gv.sp.rtol = d->rtol;
  gv.sp.kmax = d->kmax;
  gv.sp.lsmax = d->lsmax;

  const size_t N = (size_t)gv.nvar, zg = (size_t)gv.zg, n2d = (size_t)gv.n2d;
  auto alloc = [&](void **p, size_t bytes) { return cudaMalloc(p, bytes ? bytes : 8); };
  cudaError_t e = cudaSuccess;
#define A_(ptr, bytes) if (e == cudaSuccess) e = alloc((void **)&(ptr), (bytes))
  A_(c->geomC, GT_NCOMP * n2d * 8);
  for (int a = 0; a < 3; a++) A_(c->geomF[a], GT_NCOMP * n2d * 8);
  A_(c->conn, CONN_NCOMP * n2d * 8);
  A_(c->C, N * zg * 8);
  A_(c->G, 3 * zg * 8);
  A_(c->Fface, 3 * N * zg * 8);
  A_(c->cface, 3 * zg * 8);
  if (d->flux_ct) A_(c->emf, 3 * zg * 8);
  A_(c->Ph, N * zg * 8);
  A_(c->Pnew, N * zg * 8);
  A_(c->resnorm, zg * 8);
  A_(c->status, zg * 4);
  A_(c->iters, zg * 4);
  A_(c->cnt, sizeof(Counters));
  A_(c->stats, 2 * sizeof(StatsDev));
  A_(c->probe_sink, 64);
#undef A_
  if (e != cudaSuccess) {
    std::string msg = std::string("cudaMalloc: ") + cudaGetErrorString(e);
    grim_free(c);
    return fail(nullptr, GRIM_ENOMEM, msg);
  }
  gv.geomC = c->geomC;
  for (int a = 0; a < 3; a++) gv.geomF[a] = c->geomF[a];
  gv.conn = c->conn;
  gv.flux_ct = d->flux_ct ? 1 : 0;
  gv.reduced = d->reduced_solve ? 1 : 0;
  gv.emf = c->emf;
  gv.nsm = prop.multiProcessorCount;
  cudaMemsetAsync(c->G, 0, 3 * zg * 8, c->stream);
  cudaMemsetAsync(c->C, 0, N * zg * 8, c->stream);
  *out = c;
  return GRIM_OK;
}

extern "C" int grim_set_metric(grim_ctx *c, int32_t kind, const double *params, int32_t nparams) {
  if (!c) return GRIM_EINVAL;
  CU(cudaSetDevice(c->d.device));
  if (kind == GRIM_MINKOWSKI) {
    c->launches += timed(c, GRIM_K_OTHER, [&] { return launch_metric_flat(c->gv, c->geomC, c->geomF[0], c->geomF[1], c->geomF[2], c->conn, c->stream); });
  } else if (kind == GRIM_KERR_MKS) {
    if (!params || nparams < 2) return fail(c, GRIM_EINVAL, "Kerr needs params = {a, h}");
    if (c->d.dim < 2) return fail(c, GRIM_EINVAL, "Kerr needs at least the X1, X2 directions");
    c->launches += timed(c, GRIM_K_OTHER, [&] { return launch_metric_kerr(c->gv, params[0], params[1], c->d.tau_mode, c->geomC, c->geomF[0],
                                      c->geomF[1], c->geomF[2], c->conn, c->stream); });
  } else {
    return fail(c, GRIM_EINVAL, "unknown metric");
  }
  int rc = check_launch(c, "metric kernel");
  if (rc) return rc;
  c->gv.metric = kind;
  c->metric_set = 1;
  return GRIM_OK;
}

extern "C" int grim_set_metric_tables(grim_ctx *c, const double *tab, const double *conn) {
  if (!c) return GRIM_EINVAL;
  if (!tab || !conn) return fail(c, GRIM_EINVAL, "grim_set_metric_tables: null argument");
  if (c->d.dim < 2) return fail(c, GRIM_EINVAL, "a general metric needs at least the X1, X2 directions");
  CU(cudaSetDevice(c->d.device));
  const size_t n2d = (size_t)c->gv.n2d;
  std::vector<double> h((size_t)GT_NCOMP * n2d);
  for (int loc = 0; loc < 4; loc++) {
    const double *t = tab + (size_t)loc * 23 * n2d;
    memcpy(&h[(size_t)GT_GCOV * n2d], t, 20 * n2d * sizeof(double));  // g_mu_nu, g^mu^nu
    memcpy(&h[(size_t)GT_SQRTMG * n2d], t + 20 * n2d, n2d * sizeof(double));
    memcpy(&h[(size_t)GT_ALPHA * n2d], t + 21 * n2d, n2d * sizeof(double));
    for (size_t id = 0; id < n2d; id++) {
      h[(size_t)GT_TAU * n2d + id] = (c->d.tau_mode == GRIM_TAU_R32) ? t[22 * n2d + id] : c->d.tau;
      for (int i = 1; i < 4; i++)  // alpha g^{ti} = beta^i/alpha (C-9)
        h[(size_t)(GT_BFAC + i - 1) * n2d + id] = t[21 * n2d + id] * t[(size_t)(GT_GCON + sym4(0, i)) * n2d + id];
    }
    double *dst = loc == 0 ? c->geomC : c->geomF[loc - 1];
    CU(cudaMemcpyAsync(dst, h.data(), h.size() * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    CU(cudaStreamSynchronize(c->stream));
  }
  CU(cudaMemcpyAsync(c->conn, conn, (size_t)CONN_NCOMP * n2d * sizeof(double), cudaMemcpyHostToDevice, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  c->gv.metric = GRIM_KERR_MKS;
  c->metric_set = 1;
  return GRIM_OK;
}

static int need_metric(grim_ctx *c) {
  if (!c) return GRIM_EINVAL;
  if (!c->metric_set) return fail(c, GRIM_ESTATE, "grim_set_metric has not been called");
  return GRIM_OK;
}

extern "C" int grim_fill_ghosts(grim_ctx *c, double *P) {
  if (!c || !P) return fail(c, GRIM_EINVAL, "grim_fill_ghosts: null argument");
  CU(cudaSetDevice(c->d.device));
  c->launches += timed(c, GRIM_K_GHOSTS, [&] { return launch_fill_ghosts(c->gv, c->d.bc, P, c->stream); });
  return check_launch(c, "fill_ghosts kernel");
}

extern "C" int grim_compute_fluxes(grim_ctx *c, const double *P_E, const double *P_n, double dt_stage,
                                   double *C_out, double *G_out, double *speeds_out) {
  int rc = need_metric(c);
  if (rc) return rc;
  if (!P_E || !P_n) return fail(c, GRIM_EINVAL, "grim_compute_fluxes: null P_E or P_n");
  if (!(dt_stage > 0.0)) return fail(c, GRIM_EINVAL, "dt_stage must be positive");
  CU(cudaSetDevice(c->d.device));
  Counters *cnt = nullptr;
  if (speeds_out) {
    CU(cudaMemsetAsync(c->cnt, 0, sizeof(Counters), c->stream));
    cnt = c->cnt;
  }
  c->launches += timed(c, GRIM_K_FLUX, [&] { return launch_fluxes(c->gv, P_E, P_n, dt_stage, C_out ? C_out : c->C, G_out ? G_out : c->G, c->Fface,
                               c->cface, cnt, c->stream); });
  rc = check_launch(c, "flux kernels");
  if (rc) return rc;
  if (speeds_out)
    CU(cudaMemcpyAsync(speeds_out, c->cnt->speeds, 4 * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
  return GRIM_OK;
}

extern "C" int grim_newton_step(grim_ctx *c, const double *P_n, const double *P_E, const double *C, const double *G,
                                double dt_stage, int32_t max_iters, double *P_iter, double *resnorm,
                                int32_t *status, int32_t *iters, int64_t *n_active_out) {
  int rc = need_metric(c);
  if (rc) return rc;
  if (!P_n || !P_E || !P_iter || !resnorm || !status || !iters)
    return fail(c, GRIM_EINVAL, "grim_newton_step: null array argument");
  if (!(dt_stage > 0.0)) return fail(c, GRIM_EINVAL, "dt_stage must be positive");
  CU(cudaSetDevice(c->d.device));
  CU(cudaMemsetAsync(c->cnt, 0, sizeof(Counters), c->stream));
  c->launches += timed(c, GRIM_K_NEWTON, [&] { return launch_newton_stage(c->gv, P_n, P_E, C ? C : c->C, G ? G : c->G, P_iter, 0, dt_stage, max_iters, P_iter,
                                     resnorm, status, iters, c->cnt, c->stream); });
  rc = check_launch(c, "newton_stage kernel");
  if (rc) return rc;
  if (n_active_out) {
    unsigned long long na = 0;
    CU(cudaMemcpyAsync(&na, &c->cnt->n_active, sizeof(na), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    *n_active_out = (int64_t)na;
  }
  return GRIM_OK;
}

// Grows active-zone list a to hold n zone indices (never shrinks).
static int ensure_list(grim_ctx *c, int a, long long n) {
  if (c->list_cap[a] >= n) return GRIM_OK;
  if (c->list[a]) cudaFree(c->list[a]);
  c->list[a] = nullptr;
  c->list_cap[a] = 0;
  CU(cudaMalloc((void **)&c->list[a], (size_t)n * sizeof(long long)));
  c->list_cap[a] = n;
  return GRIM_OK;
}

// A fresh solve of every interior zone to a terminal status (steps a4-a7), in sweeps: the first launch gives every zone
// STAGE_SWEEP iterations; the zones that need more -- a few per cent in a run whose iteration counts spread (the
// torus: 2-8), none in a smooth run -- are collected and solved afresh, to the end, by a second launch over that list
// only, so that a warp does not idle through the long solves of a few of its lanes.  The per-zone results are those of
// one uninterrupted solve (it IS one, for every zone); the list length stays on the device.
static constexpr int STAGE_SWEEP = 4;   // iterations of the first launch (3 and 5 measured slower on the torus)
static constexpr int SWEEP_PROBE = 64;  // single-launch solves between two probes of the sweep mode
static int solve_stage(grim_ctx *c, const GridView &gv, const double *Pn, const double *PE, const double *C,
                       const double *G, const double *Pguess, double dt_stage, double *Pout, double *resnorm,
                       int32_t *status, int32_t *iters) {
  cudaStream_t s = c->stream;
  bool sweeps = STAGE_SWEEP > 0 && gv.sp.kmax > STAGE_SWEEP;
  // While the stream is being captured into a CUDA graph the policy below (event queries, a pinned read-back) must not
  // run: a captured step always takes the two-launch form, whose list length stays on the device.
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(s, &cap);
  const bool capturing = cap != cudaStreamCaptureStatusNone;
  if (sweeps && !capturing) {
    // Both modes give the same results zone for zone; the policy only decides which is faster.  Collect the counts of
    // earlier sweep-mode solves that have landed: 4 in a row without a deferred zone -> single launches for a while.
    if (!c->sweep_counts) {
      CU(cudaMallocHost((void **)&c->sweep_counts, 4 * sizeof(unsigned long long)));
      for (int q = 0; q < 4; q++) {
        CU(cudaEventCreateWithFlags(&c->sweep_ev[q], cudaEventDisableTiming));
        c->sweep_pending[q] = 0;
      }
    }
    for (int q = 0; q < 4; q++) {
      if (!c->sweep_pending[q]) continue;
      if (cudaEventQuery(c->sweep_ev[q]) == cudaSuccess) {
        c->sweep_pending[q] = 0;
        if (c->sweep_counts[q] == 0) c->sweep_quiet++;
        else c->sweep_quiet = 0;
      } else {
        (void)cudaGetLastError();  // cudaErrorNotReady is an answer, not a failure: keep it out of check_launch()
      }
    }
    if (c->sweep_quiet >= 4) {
      c->sweep_quiet = 0;
      c->sweep_skip = SWEEP_PROBE;
    }
    if (c->sweep_skip > 0) {
      c->sweep_skip--;
      sweeps = false;
    }
  }
  if (sweeps) {
    int rcl = ensure_list(c, 0, gv.nint);  // the stage solve compacts once: one list
    if (rcl) return rcl;
  }
  CU(cudaMemsetAsync(c->cnt, 0, sizeof(Counters), s));
  GridView g1 = gv;
  if (sweeps) g1.sp.kmax = STAGE_SWEEP;
  c->launches += timed(c, GRIM_K_NEWTON, [&] {
    return launch_newton_stage(g1, Pn, PE, C, G, Pguess, 1, dt_stage, 0, Pout, resnorm, status, iters, c->cnt, s, nullptr, 0,
                               sweeps ? c->list[0] : nullptr);
  });
  int rc = check_launch(c, "newton_stage kernel");
  if (rc || !sweeps) return rc;
  // the second sweep reads the list length from the device: no synchronisation; the length also goes to the host,
  // asynchronously, for the sweep policy
  if (!capturing) {
    const int q = c->sweep_slot;
    if (!c->sweep_pending[q]) {
      CU(cudaMemcpyAsync(&c->sweep_counts[q], &c->cnt->list_count, sizeof(unsigned long long), cudaMemcpyDeviceToHost, s));
      CU(cudaEventRecord(c->sweep_ev[q], s));
      c->sweep_pending[q] = 1;
      c->sweep_slot = (q + 1) % 4;
    }
  }
  c->launches += timed(c, GRIM_K_NEWTON, [&] {
    return launch_newton_stage(gv, Pn, PE, C, G, Pguess, 1, dt_stage, 0, Pout, resnorm, status, iters, c->cnt, s,
                               c->list[0], 0, nullptr);
  });
  return check_launch(c, "newton_stage kernel (second sweep)");
}

extern "C" int grim_newton_solve(grim_ctx *c, const double *P_n, const double *P_E, const double *C, const double *G,
                                 double dt_stage, const double *P_guess, double *P_out, double *resnorm,
                                 int32_t *status, int32_t *iters) {
  int rc = need_metric(c);
  if (rc) return rc;
  if (!P_n || !P_E || !P_guess || !P_out) return fail(c, GRIM_EINVAL, "grim_newton_solve: null array argument");
  if (!(dt_stage > 0.0)) return fail(c, GRIM_EINVAL, "dt_stage must be positive");
  CU(cudaSetDevice(c->d.device));
  return solve_stage(c, c->gv, P_n, P_E, C ? C : c->C, G ? G : c->G, P_guess, dt_stage, P_out,
                     resnorm ? resnorm : c->resnorm, status ? status : c->status, iters ? iters : c->iters);
}

extern "C" int grim_prim_to_conserved(grim_ctx *c, int64_t nz, const double *P, double *U) {
  if (!c || !P || !U || nz < 0) return fail(c, GRIM_EINVAL, "grim_prim_to_conserved: bad argument");
  CU(cudaSetDevice(c->d.device));
  c->launches += timed(c, GRIM_K_OTHER, [&] { return launch_prim_to_conserved(c->gv, nz, P, U, c->stream); });
  return check_launch(c, "prim_to_conserved kernel");
}

extern "C" int grim_invert_primitives(grim_ctx *c, int64_t nz, const double *U_target, const double *geom,
                                      double *P_inout, int32_t *iters, int32_t *status, double *resnorm) {
  if (!c) return GRIM_EINVAL;
  if (nz < 0 || (nz > 0 && (!U_target || !P_inout || !iters || !status || !resnorm)))
    return fail(c, GRIM_EINVAL, "grim_invert_primitives: bad argument");
  if (nz == 0) return GRIM_OK;
  CU(cudaSetDevice(c->d.device));
  for (int a = 0; a < 2; a++) {  // the inversion ping-pongs between two lists
    int rcl = ensure_list(c, a, nz);
    if (rcl) return rcl;
  }
  // sweeps of a few iterations each over the compacted set of zones that are still iterating
  const int kmax = c->gv.sp.kmax;
  long long nlist = nz;
  int first = 1, cur = 0, done_iters = 0;
  while (nlist > 0) {
    const int sweep = first ? SWEEP_FIRST : SWEEP_REST;
    CU(cudaMemsetAsync(c->cnt, 0, sizeof(Counters), c->stream));
    c->launches += timed(c, GRIM_K_INVERT, [&] { return launch_invert(c->gv, nz, nlist, c->list[cur], U_target, geom, P_inout, iters, status, resnorm, sweep,
                                 first, c->list[cur ^ 1], c->cnt, c->stream); });
    int rc = check_launch(c, "invert kernel");
    if (rc) return rc;
    unsigned long long cntn = 0;
    CU(cudaMemcpyAsync(&cntn, &c->cnt->list_count, sizeof(cntn), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    nlist = (long long)cntn;
    cur ^= 1;
    first = 0;
    done_iters += sweep;
    if (done_iters > kmax + 8) break;  // cannot happen: every zone reaches kmax
  }
  return GRIM_OK;
}

static void stats_to_host(const StatsDev *h, int stage, grim_step_stats *st) {
  for (int b = 0; b < 16; b++) st->iters_hist[stage][b] = (int64_t)h->hist[b];
  st->unconverged[stage] = (int64_t)h->unconverged;
  double v;
  memcpy(&v, &h->max_rel, sizeof(v));
  st->max_resnorm[stage] = v;
}

extern "C" int grim_timestep(grim_ctx *c, double *P, double dt, double *dt_used, grim_step_stats *stats) {
  int rc = need_metric(c);
  if (rc) return rc;
  if (!P) return fail(c, GRIM_EINVAL, "grim_timestep: null P");
  CU(cudaSetDevice(c->d.device));
  const GridView &gv = c->gv;
  const size_t pbytes = (size_t)gv.nvar * gv.zg * 8;
  cudaStream_t s = c->stream;
  unsigned long long bt[2] = {0, 0};

  c->launches += timed(c, GRIM_K_GHOSTS, [&] { return launch_fill_ghosts(gv, c->d.bc, P, s); });
  bool have_faces = false;
  if (!(dt > 0.0)) {
    // C-15: dt = cfl / max_z sum_d c^d/dX^d.  The face fluxes and speeds of stage 1 (P_E = P_n) do not depend on dt:
    // compute them now, reduce the speeds, and let stage 1 below form its stage constant from the same face arrays.
    CU(cudaMemsetAsync(c->cnt, 0, sizeof(Counters), s));
    c->launches += timed(c, GRIM_K_FLUX, [&] {
      int n = launch_fluxes(gv, P, P, 1.0, c->C, c->G, c->Fface, c->cface, nullptr, s, 1);
      return n + launch_speeds(gv, c->cface, c->cnt, s);
    });
    double sp3 = 0.0;
    CU(cudaMemcpyAsync(&sp3, &c->cnt->speeds[3], sizeof(double), cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    if (!(sp3 > 0.0)) return fail(c, GRIM_ESTATE, "maximum wave speed is not positive");
    dt = c->d.cfl / sp3;
    have_faces = true;
  }
  if (stats) CU(cudaMemsetAsync(c->stats, 0, 2 * sizeof(StatsDev), s));

  // Ghost zones of a direction whose boundary condition is GRIM_BC_NONE are the caller's: the stage buffer then
  // starts as a copy of P so that it carries them.  Otherwise each stage reads its guess from P_E and writes the
  // interior of its output, and nothing is copied.
  bool caller_ghosts = false;
  for (int a = 0; a < 3; a++)
    for (int sd = 0; sd < 2; sd++)
      if (gv.ngd[a] > 0 && c->d.bc[a][sd] == GRIM_BC_NONE) caller_ghosts = true;

  // stage 1: P_E = P_n, dt' = dt/2, guess P_n (eq 19; C-7)
  const double dt1 = 0.5 * dt;
  c->launches += timed(c, GRIM_K_FLUX, [&] { return launch_fluxes(gv, P, P, dt1, c->C, c->G, c->Fface, c->cface, nullptr, s, have_faces ? 2 : 3); });
  if (caller_ghosts) CU(cudaMemcpyAsync(c->Ph, P, pbytes, cudaMemcpyDeviceToDevice, s));
  rc = solve_stage(c, gv, P, P, c->C, c->G, P, dt1, c->Ph, c->resnorm, c->status, c->iters);
  if (rc) return rc;
  if (stats) {
    c->launches += timed(c, GRIM_K_OTHER, [&] { return launch_stats(gv, P, dt1, c->resnorm, c->status, c->iters, &c->stats[0], s); });
    CU(cudaMemcpyAsync(&bt[0], &c->cnt->backtracks, 8, cudaMemcpyDeviceToHost, s));
  }
  // stage 2: P_E = P_{n+1/2}, dt' = dt, guess P_{n+1/2} (eq 13).  The Newton kernel reads P_n zone by zone
  // before it writes that zone, so P_{n+1} goes straight into P -- unless the statistics still need P_n.
  c->launches += timed(c, GRIM_K_GHOSTS, [&] { return launch_fill_ghosts(gv, c->d.bc, c->Ph, s); });
  c->launches += timed(c, GRIM_K_FLUX, [&] { return launch_fluxes(gv, c->Ph, P, dt, c->C, c->G, c->Fface, c->cface, nullptr, s); });
  if (stats) CU(cudaStreamSynchronize(s));  // bt[0] must land before the counters are cleared
  double *out2 = stats ? c->Pnew : P;
  rc = solve_stage(c, gv, P, c->Ph, c->C, c->G, c->Ph, dt, out2, c->resnorm, c->status, c->iters);
  if (rc) return rc;
  if (stats) {
    c->launches += timed(c, GRIM_K_OTHER, [&] { return launch_stats(gv, P, dt, c->resnorm, c->status, c->iters, &c->stats[1], s); });
    CU(cudaMemcpyAsync(&bt[1], &c->cnt->backtracks, 8, cudaMemcpyDeviceToHost, s));
    c->launches += timed(c, GRIM_K_OTHER, [&] { return launch_copy_interior(gv, c->Pnew, P, s); });
  }
  rc = check_launch(c, "timestep kernels");
  if (rc) return rc;
  if (stats) {
    StatsDev h[2];
    CU(cudaMemcpyAsync(h, c->stats, sizeof(h), cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    memset(stats, 0, sizeof(*stats));
    stats->zones = gv.nint;
    stats_to_host(&h[0], 0, stats);
    stats_to_host(&h[1], 1, stats);
    stats->backtracks[0] = (int64_t)bt[0];
    stats->backtracks[1] = (int64_t)bt[1];
  }
  if (dt_used) {
    CU(cudaStreamSynchronize(s));
    *dt_used = dt;
  }
  return GRIM_OK;
}

extern "C" int grim_get_geometry(grim_ctx *c, int32_t loc, int64_t idx2d, double *gcov, double *gcon,
                                 double *sqrtmg, double *alpha, double *tau, double *conn) {
  int rc = need_metric(c);
  if (rc) return rc;
  if (loc < 0 || loc > 3 || idx2d < 0 || idx2d >= c->gv.n2d) return fail(c, GRIM_EINVAL, "bad location");
  CU(cudaSetDevice(c->d.device));
  const double *tab = loc == 0 ? c->geomC : c->geomF[loc - 1];
  double comp[GT_NCOMP];
  CU(cudaStreamSynchronize(c->stream));
  CU(cudaMemcpy2D(comp, 8, tab + idx2d, (size_t)c->gv.n2d * 8, 8, GT_NCOMP, cudaMemcpyDeviceToHost));
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < 4; n++) {
      if (gcov) gcov[m * 4 + n] = comp[GT_GCOV + sym4(m, n)];
      if (gcon) gcon[m * 4 + n] = comp[GT_GCON + sym4(m, n)];
    }
  if (sqrtmg) *sqrtmg = comp[GT_SQRTMG];
  if (alpha) *alpha = comp[GT_ALPHA];
  if (tau) *tau = comp[GT_TAU];
  if (conn) CU(cudaMemcpy2D(conn, 8, c->conn + idx2d, (size_t)c->gv.n2d * 8, 8, CONN_NCOMP, cudaMemcpyDeviceToHost));
  return GRIM_OK;
}

extern "C" int grim_fp64_probe(grim_ctx *c, int32_t fma, int32_t iters, double *inst_per_s) {
  if (!c || !inst_per_s || iters <= 0) return fail(c, GRIM_EINVAL, "grim_fp64_probe: bad argument");
  CU(cudaSetDevice(c->d.device));
  cudaDeviceProp prop;
  CU(cudaGetDeviceProperties(&prop, c->d.device));
  const int threads = 256, blocks = prop.multiProcessorCount * 8;
  cudaEvent_t e0, e1;
  CU(cudaEventCreate(&e0));
  CU(cudaEventCreate(&e1));
  launch_fp64_probe(fma, iters, c->probe_sink, blocks, threads, c->stream);  // warm-up
  CU(cudaEventRecord(e0, c->stream));
  launch_fp64_probe(fma, iters, c->probe_sink, blocks, threads, c->stream);
  CU(cudaEventRecord(e1, c->stream));
  CU(cudaEventSynchronize(e1));
  c->launches += 2;
  float ms = 0.f;
  CU(cudaEventElapsedTime(&ms, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *inst_per_s = (double)blocks * threads * (double)iters * 8.0 / (ms * 1e-3);
  return check_launch(c, "fp64 probe");
}

extern "C" int grim_arith_selftest(grim_ctx *c, int64_t n, int64_t seed, int32_t wide, int64_t *out6) {
  if (!c || !out6 || n < 0) return fail(c, GRIM_EINVAL, "grim_arith_selftest: bad argument");
  CU(cudaSetDevice(c->d.device));
  unsigned long long *d = nullptr;
  CU(cudaMalloc((void **)&d, 6 * sizeof(unsigned long long)));
  CU(cudaMemsetAsync(d, 0, 6 * sizeof(unsigned long long), c->stream));
  c->launches += launch_arith_selftest((unsigned long long)n, (unsigned long long)seed, wide, d, c->stream);
  unsigned long long h[6];
  cudaError_t e = cudaMemcpyAsync(h, d, sizeof(h), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  cudaFree(d);
  if (e != cudaSuccess) return fail(c, GRIM_ECUDA, cudaGetErrorString(e));
  for (int k = 0; k < 6; k++) out6[k] = (int64_t)h[k];
  return check_launch(c, "arith selftest");
}

// One time step with HOST buffers, pipelined over K slabs of X^3 planes: the host -> device copy of slab c + 1, the
// kernels of slab c (stage 1) and c - 1 (stage 2) and the device -> host copy of slab c - 2 run at the same time on three
// streams.  A slab's stage 1 needs P_n of the neighbouring slabs (stencil of the flux step, 3 + 1 planes), its stage 2
// P_{n+1/2} of the neighbouring slabs; the X^3 boundary (periodic wrap or a physical boundary) couples the first and
// the last slab, which therefore arrive first and finish last.  Stage 1 of every slab runs on the context's stream, stage 2
// on a second compute stream (s_st2), ordered by events so that every read stays ahead of the write that would overwrite
// it (stage 2 writes P_{n+1} over P_n in place); the results are those of grim_timestep bit for bit.  Ghost zones of P_host are neither read nor written.
static constexpr int HOST_SLABS = 16;  // slabs of the pipelined host step
static constexpr int HOST_EDGE = 4;    // planes of its first and last slab
static int pipelined_enqueue(grim_ctx *c, double *P_host, double dt) {
  const GridView &gv = c->gv;
  cudaStream_t s = c->stream;
  const int K = HOST_SLABS, ng = gv.ngd[2], n3 = gv.n[2];
  const size_t plane = (size_t)gv.sz[0] * gv.sz[1], pitch = (size_t)gv.zg * 8;
  if (!c->s_in) CU(cudaStreamCreateWithFlags(&c->s_in, cudaStreamNonBlocking));
  if (!c->s_out) CU(cudaStreamCreateWithFlags(&c->s_out, cudaStreamNonBlocking));
  if (!c->s_st2) CU(cudaStreamCreateWithFlags(&c->s_st2, cudaStreamNonBlocking));
  while ((int)c->ev_in.size() < K + 1) {
    cudaEvent_t e;
    CU(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    c->ev_in.push_back(e);
    CU(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    c->ev_done.push_back(e);
    CU(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    c->ev_s1.push_back(e);
  }
  cudaStream_t s2 = c->s_st2;
  int k0[HOST_SLABS + 1];
  // Slab boundaries, multiples of the 4-plane flux tiles.  The first and the last slab are coupled through the X^3
  // boundary: they arrive first and finish last, nothing overlaps their copies -- so they are thin (HOST_EDGE
  // planes) and the K - 2 slabs between them share the rest.
  {
    const int e = (n3 >= 16 * HOST_EDGE) ? HOST_EDGE : 0;
    if (e) {
      k0[0] = 0;
      k0[1] = e;
      for (int q = 2; q < K - 1; q++) k0[q] = e + (int)((long long)(n3 - 2 * e) * (q - 1) / (K - 2) / 4 * 4);
      k0[K - 1] = n3 - e;
      k0[K] = n3;
    } else {
      for (int q = 0; q <= K; q++) k0[q] = (int)((long long)n3 * q / K / 4 * 4);
      k0[K] = n3;
    }
  }
  double *d = c->hostP;
  // the copy streams start after whatever the caller enqueued on the context's stream
  CU(cudaEventRecord(c->ev_in[K], s));
  CU(cudaStreamWaitEvent(c->s_in, c->ev_in[K], 0));
  CU(cudaStreamWaitEvent(c->s_out, c->ev_in[K], 0));
  CU(cudaStreamWaitEvent(s2, c->ev_in[K], 0));
  // the lambdas cannot return through CU(): they keep the first failing return code, checked at the end
  cudaError_t bad = cudaSuccess;
  auto keep = [&](cudaError_t e) {
    if (e != cudaSuccess && bad == cudaSuccess) bad = e;
  };
  auto h2d = [&](int q) {
    const size_t off = (size_t)(ng + k0[q]) * plane;
    keep(cudaMemcpy2DAsync(d + off, pitch, P_host + off, pitch, (size_t)(k0[q + 1] - k0[q]) * plane * 8, (size_t)gv.nvar,
                           cudaMemcpyHostToDevice, c->s_in));
    keep(cudaEventRecord(c->ev_in[q], c->s_in));
  };
  h2d(K - 1);
  for (int q = 0; q < K - 1; q++) h2d(q);
  auto slab = [&](int q) {
    GridView g = gv;
    g.koff = k0[q];
    g.n[2] = k0[q + 1] - k0[q];
    g.nint = (long long)g.n[0] * g.n[1] * g.n[2];
    return g;
  };
  auto ghosts01 = [&](double *P, int q) {  // X^1, X^2 ghosts of the slab's planes
    c->launches += timed(c, GRIM_K_GHOSTS, [&] { return launch_fill_ghosts(gv, c->d.bc, P, s, 3, ng + k0[q], k0[q + 1] - k0[q]); });
  };
  auto ghosts2 = [&](double *P) {
    c->launches += timed(c, GRIM_K_GHOSTS, [&] { return launch_fill_ghosts(gv, c->d.bc, P, s, 4); });
  };
  const double dt1 = 0.5 * dt;
  auto stage1 = [&](int q) {
    const GridView g = slab(q);
    c->launches += timed(c, GRIM_K_FLUX, [&] { return launch_fluxes(g, d, d, dt1, c->C, c->G, c->Fface, c->cface, nullptr, s); });
    c->launches += timed(c, GRIM_K_NEWTON, [&] { return launch_newton_stage(g, d, d, c->C, c->G, d, 1, dt1, 0, c->Ph, c->resnorm, c->status, c->iters, c->cnt, s); });
  };
  // Stage 2 runs on a second stream: stage 2 of slab q needs stage 1 of slabs q - 1, q, q + 1 (event ev_s1[q + 1]) and
  // is independent of stage 1 of the later slabs, which the first stream goes on with -- the two streams' kernels touch
  // disjoint plane ranges of every scratch array (slab q against slabs >= q + 2), and the ramps and tails of the small
  // slab-wise launches overlap instead of adding up.
  auto stage2 = [&](int q, cudaEvent_t after) {
    const GridView g = slab(q);
    keep(cudaStreamWaitEvent(s2, after, 0));
    c->launches += timed(c, GRIM_K_FLUX, [&] { return launch_fluxes(g, c->Ph, d, dt, c->C, c->G, c->Fface, c->cface, nullptr, s2); }, s2);
    c->launches += timed(c, GRIM_K_NEWTON, [&] { return launch_newton_stage(g, d, c->Ph, c->C, c->G, c->Ph, 1, dt, 0, d, c->resnorm, c->status, c->iters, c->cnt, s2); }, s2);
    keep(cudaEventRecord(c->ev_done[q], s2));
    keep(cudaStreamWaitEvent(c->s_out, c->ev_done[q], 0));
    const size_t off = (size_t)(ng + k0[q]) * plane;
    keep(cudaMemcpy2DAsync(P_host + off, pitch, d + off, pitch, (size_t)(k0[q + 1] - k0[q]) * plane * 8, (size_t)gv.nvar,
                           cudaMemcpyDeviceToHost, c->s_out));
  };
  CU(cudaMemsetAsync(c->cnt, 0, sizeof(Counters), s));
  CU(cudaStreamWaitEvent(s, c->ev_in[K - 1], 0));
  CU(cudaStreamWaitEvent(s, c->ev_in[0], 0));
  ghosts01(d, K - 1);
  ghosts01(d, 0);
  ghosts2(d);
  for (int q = 0; q < K; q++) {
    if (q + 1 <= K - 2) {
      CU(cudaStreamWaitEvent(s, c->ev_in[q + 1], 0));
      ghosts01(d, q + 1);
    }
    stage1(q);
    ghosts01(c->Ph, q);
    CU(cudaEventRecord(c->ev_s1[q], s));
    if (q >= 2) stage2(q - 1, c->ev_s1[q]);
  }
  ghosts2(c->Ph);
  CU(cudaEventRecord(c->ev_s1[K], s));
  stage2(K - 1, c->ev_s1[K]);
  stage2(0, c->ev_s1[K]);
  if (bad != cudaSuccess) return fail(c, GRIM_ECUDA, std::string("pipelined timestep: ") + cudaGetErrorString(bad));
  return check_launch(c, "pipelined timestep");
}

// Enqueues the pipelined step and waits for it.  Whatever pipelined_enqueue returns -- also an early error return with
// copies into the caller's P_host still in flight -- all four streams are drained before the caller gets control back.
static int timestep_host_pipelined(grim_ctx *c, double *P_host, double dt) {
  int rc = pipelined_enqueue(c, P_host, dt);
  cudaStream_t side[3] = {c->s_in, c->s_st2, c->s_out};
  for (int q = 0; q < 4; q++) {
    if (q < 3 && side[q] == nullptr) continue;  // a side stream that was never created
    cudaError_t e = cudaStreamSynchronize(q < 3 ? side[q] : c->stream);
    if (e != cudaSuccess && rc == GRIM_OK) rc = fail(c, GRIM_ECUDA, std::string("pipelined timestep: ") + cudaGetErrorString(e));
  }
  return rc;
}

extern "C" int grim_timestep_host(grim_ctx *c, double *P_host, int32_t nsteps, double dt, double *dt_used) {
  int rc = need_metric(c);
  if (rc) return rc;
  if (!P_host || nsteps < 0) return fail(c, GRIM_EINVAL, "grim_timestep_host: bad argument");
  CU(cudaSetDevice(c->d.device));
  const size_t pbytes = (size_t)c->gv.nvar * c->gv.zg * 8;
  if (!c->hostP) CU(cudaMalloc((void **)&c->hostP, pbytes));
  {
    bool caller_ghosts = false;
    for (int a = 0; a < 3; a++)
      for (int sd = 0; sd < 2; sd++)
        if (c->gv.ngd[a] > 0 && c->d.bc[a][sd] == GRIM_BC_NONE) caller_ghosts = true;
    // slab-wise launches pay off from about 1.5 M zones (measured: 64^3 and 96^3 are faster copied whole)
    const bool big = c->gv.nint >= 1500000 || c->no_pipeline < 0;
    if (nsteps == 1 && dt > 0.0 && c->gv.dim == 3 && c->gv.n[2] >= 4 * HOST_SLABS && !c->gv.flux_ct && !caller_ghosts &&
        big && c->no_pipeline <= 0) {
      c->last_host_mode = GRIM_HOST_MODE_PIPELINED;
      rc = timestep_host_pipelined(c, P_host, dt);
      if (rc == GRIM_OK && dt_used) *dt_used = dt;
      return rc;
    }
  }
  c->last_host_mode = GRIM_HOST_MODE_WHOLE;
  CU(cudaMemcpyAsync(c->hostP, P_host, pbytes, cudaMemcpyHostToDevice, c->stream));
  for (int s = 0; s < nsteps; s++) {
    rc = grim_timestep(c, c->hostP, dt, dt_used, nullptr);
    if (rc) return rc;
  }
  CU(cudaMemcpyAsync(P_host, c->hostP, pbytes, cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  return GRIM_OK;
}

extern "C" int grim_last_host_mode(const grim_ctx *c) { return c ? c->last_host_mode : GRIM_HOST_MODE_NONE; }

extern "C" int grim_invert_primitives_host(grim_ctx *c, int64_t nz, const double *U_host, double *P_host,
                                           int32_t *iters_host, int32_t *status_host, double *resnorm_host) {
  if (!c) return GRIM_EINVAL;
  if (nz < 0 || (nz > 0 && (!U_host || !P_host))) return fail(c, GRIM_EINVAL, "grim_invert_primitives_host: bad argument");
  if (nz == 0) return GRIM_OK;
  CU(cudaSetDevice(c->d.device));
  const size_t N = (size_t)c->gv.nvar;
  if (c->invbuf_nz < nz) {
    if (c->invbuf) cudaFree(c->invbuf);
    c->invbuf = nullptr;
    CU(cudaMalloc((void **)&c->invbuf, (2 * N + 2) * (size_t)nz * 8));
    c->invbuf_nz = nz;
  }
  double *dU = c->invbuf, *dP = dU + N * nz, *dres = dP + N * nz;
  int32_t *dit = (int32_t *)(dres + nz), *dst = dit + nz;
  CU(cudaMemcpyAsync(dU, U_host, N * nz * 8, cudaMemcpyHostToDevice, c->stream));
  CU(cudaMemcpyAsync(dP, P_host, N * nz * 8, cudaMemcpyHostToDevice, c->stream));
  int rc = grim_invert_primitives(c, nz, dU, nullptr, dP, dit, dst, dres);
  if (rc) return rc;
  CU(cudaMemcpyAsync(P_host, dP, N * nz * 8, cudaMemcpyDeviceToHost, c->stream));
  if (iters_host) CU(cudaMemcpyAsync(iters_host, dit, (size_t)nz * 4, cudaMemcpyDeviceToHost, c->stream));
  if (status_host) CU(cudaMemcpyAsync(status_host, dst, (size_t)nz * 4, cudaMemcpyDeviceToHost, c->stream));
  if (resnorm_host) CU(cudaMemcpyAsync(resnorm_host, dres, (size_t)nz * 8, cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  return GRIM_OK;
}
