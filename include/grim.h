/*
 * grim.h -- C ABI of the B200-native hot path of grim (arXiv 1702.01106).
 *
 * The library advances the primitive variables P of an ideal-GRMHD (N = 8) or extended-GRMHD (N = 10)
 * fluid by the paper's combined time step + primitive-variable inversion: in every zone, independently,
 *
 *     R(P) = [U(P) - U(P_n)]/dt' + div F(P_E) - S = 0                          (eq 19; eq 13)
 *
 * is solved by Newton-Raphson (L190-194, eq 20) with a finite-difference Jacobian (L196-216, eqs 21-23), a
 * dense LU solve with partial pivoting (L198-200, eq 21; L434) and a quadratic backtracking line search
 * (L218-235, eqs 24-25).  div F comes from slope-limited reconstruction (L154-160) and local Lax-Friedrichs
 * fluxes (L164-166, eq 17); geometry from eqs 5-8 (L68-89).  "Lnnn" = line of /root/reference/PAPER.md;
 * "C-n", "G-n" = readings of the paper listed in DESIGN.md.
 *
 * Conventions
 *   - Every array argument is a DEVICE pointer owned by the caller unless its comment says "host".  The library
 *     never allocates, frees or copies caller arrays to the host.  The context owns geometry tables and scratch.
 *   - Grid arrays are SoA, fp64: P[v][k][j][i], i (X^1) fastest, ghosts included in every active dimension:
 *     extent s_d = n_d + 2 ng for d < dim, else n_d (= 1, no ghosts).  Zg = s1*s2*s3 zones per variable.
 *     Primitive order (L297): rho, u, u~^1, u~^2, u~^3, B^1, B^2, B^3 [, q, dP]   (u~: reading C-9).
 *   - Flat arrays (grim_invert_primitives, grim_prim_to_conserved) are [v][z], z fastest.
 *   - All work is enqueued on the stream given at grim_init_grid; calls that return a host scalar
 *     (n_active_out, dt_used, stats, speeds on host) synchronise that stream, the others are asynchronous.
 *   - Return value: 0 on success, a negative GRIM_E* code otherwise; grim_last_error() gives the text.  Nothing
 *     throws across the ABI.  Non-convergence of a zone is NOT an error: it is reported in the per-zone status
 *     word and in the counts.
 *   - Arithmetic: fp64, round-to-nearest, no FMA contraction: every + - * / sqrt is a separately rounded IEEE
 *     operation in a documented order, so results do not depend on launch geometry.
 *   - There is no CPU fallback: every entry point fails with GRIM_ECUDA if no sm_100 device is usable.
 */
#ifndef GRIM_H
#define GRIM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GRIM_VERSION 101   /* 101: grim_grid_desc gained `closure`; binding.py refuses a library of another version */

/* error codes */
enum { GRIM_OK = 0, GRIM_EINVAL = -1, GRIM_ECUDA = -2, GRIM_ENOMEM = -3, GRIM_ESTATE = -4 };

/* physics model: number of primitives per zone (L297; BASELINE north_star; reading C-1) */
enum { GRIM_IDEAL = 8, GRIM_EMHD = 10 };
/* metric (L68-89; C-10) */
enum { GRIM_MINKOWSKI = 0, GRIM_KERR_MKS = 1 };
/* reconstruction (L154-160, L115; MP5: C-6) */
enum { GRIM_MINMOD = 0, GRIM_MP5 = 1 };
/* Riemann solver (eq 17) */
enum { GRIM_LLF = 0, GRIM_HLLE = 1 };
/* boundary conditions per direction and side (C-11) */
enum { GRIM_BC_PERIODIC = 0, GRIM_BC_OUTFLOW = 1, GRIM_BC_REFLECT_POLAR = 2, GRIM_BC_NONE = 3 };
/* damping time scale tau_R: constant, or r^{3/2} (C-11) */
enum { GRIM_TAU_CONST = 0, GRIM_TAU_R32 = 1 };
enum { GRIM_CLOSURE_CS2TAU = 0, GRIM_CLOSURE_CONST = 1 };

/* per-zone status word */
enum {
  GRIM_ST_CONVERGED = 1,     /* ||R||_2 < tol_z                                              (L194) */
  GRIM_ST_KMAX = 2,          /* stopped at kmax iterations without converging                (L194) */
  GRIM_ST_LS_EXHAUSTED = 4,  /* some line search used all lsmax+1 trials; last trial taken   (C-14) */
  GRIM_ST_SINGULAR = 8,      /* zero / non-finite pivot or zero FD step; zone left unchanged (C-17, C-19) */
  GRIM_ST_NONFINITE = 16     /* non-finite residual norm                                     (C-12) */
};
#define GRIM_ST_TERMINAL (GRIM_ST_CONVERGED | GRIM_ST_KMAX | GRIM_ST_SINGULAR | GRIM_ST_NONFINITE)

typedef struct grim_ctx grim_ctx; /* opaque */

typedef struct {
  int32_t n1, n2, n3;       /* interior zones per direction (unused directions: 1)                 (L406)   */
  int32_t ng;               /* ghost depth in active directions: >= 2 for minmod, >= 3 for MP5     (G-9)    */
  int32_t dim;              /* 1, 2 or 3 active directions                                                  */
  double xstart[3], xend[3];/* extent of the interior in X^i; dX^i = (xend-xstart)/n_i             (L70-72) */
  int32_t bc[3][2];         /* GRIM_BC_* for [direction][lower, upper]                             (C-11)   */
  int32_t model;            /* GRIM_IDEAL | GRIM_EMHD                                                       */
  int32_t recon;            /* GRIM_MINMOD | GRIM_MP5                                                       */
  double limiter_theta;     /* generalised-minmod theta in [1,2] (L115, L651); also limits EMHD gradients   */
  int32_t riemann;          /* GRIM_LLF (eq 17) | GRIM_HLLE (eq 18)                                (L162-172) */
  double gamma;             /* adiabatic index                                                     (L248)   */
  double phi, psi;          /* closure chi = phi cs^2 tau_R, nu = psi cs^2 tau_R                   (L299)   */
  int32_t tau_mode;         /* GRIM_TAU_CONST | GRIM_TAU_R32                                                */
  double tau;               /* tau_R when tau_mode == GRIM_TAU_CONST                                        */
  double fd_eps;            /* epsilon of eq 23 (L202-214; C-16)                                            */
  double eps_bt;            /* epsilon_BT of the sufficient-decrease test (L223), paper: 1e-4               */
  double atol, rtol;        /* stop when ||R||_2 < atol + rtol*scale_z (L194; C-2)                          */
  int32_t kmax, lsmax;      /* Newton-iteration and line-search caps (L194; C-14)                           */
  double cfl;               /* Courant factor (L651; C-15)                                                  */
  int32_t device;           /* CUDA device ordinal                                                          */
  void *stream;             /* cudaStream_t; NULL = the legacy default stream                               */
  int32_t flux_ct;          /* != 0: flux-CT averaging of the B-field face fluxes between a2 and a3 (L327-335):
                               face -> edge -> face simple averages (Toth 2000 as in harm), F^d(B^d) = 0; keeps the
                               cell-corner-centred div B at round-off.  Needs ghost zones filled in the corners.    */
  int32_t reduced_solve;    /* != 0: the paper's own split (L148, L643): B^i is advanced explicitly,
                               sqrt(-g) B^i_new = sqrt(-g) B^i_n - dt' [div F]_{B^i}, and the Newton iteration of
                               grim_newton_step / grim_newton_solve / grim_timestep runs on the other N - 3 primitives
                               (5 x 5 / 7 x 7 Jacobian); ||R||, the tolerance and the status refer to those rows.
                               0 (default): all N primitives are unknowns (BASELINE.json).                           */
  int32_t closure;          /* GRIM_CLOSURE_CS2TAU (0, default): chi = phi cs^2 tau_R, nu = psi cs^2 tau_R (L299).
                               GRIM_CLOSURE_CONST: phi and psi ARE the thermal diffusivity chi and the kinematic
                               viscosity nu, constants, as the anisotropic-conduction test prescribes (L566:
                               "the thermal diffusivity chi = 0.01").                                                */
} grim_grid_desc;

typedef struct {
  int64_t zones;              /* interior zones                                                  */
  int64_t iters_hist[2][16];  /* [stage][min(iterations,15)] number of zones                     */
  int64_t backtracks[2];      /* rejected line-search trials per stage                           */
  int64_t unconverged[2];     /* zones without GRIM_ST_CONVERGED per stage                       */
  double max_resnorm[2];      /* max over zones of ||R||_2 / scale_z per stage                   */
} grim_step_stats;

/* ---- the six entry points named by the north star ------------------------------------------------------- */

/* Creates a context for one grid (L400-408).  `out` host.  Validates the descriptor (GRIM_EINVAL), selects the
 * device, allocates scratch: C (N*Zg), G (3*Zg), two P-sized stage buffers, per-zone resnorm/status/iters. */
int grim_init_grid(grim_ctx **out, const grim_grid_desc *d);

/* Geometry precompute (a0: L68-89 eqs 5-8; L339; C-10): fills the context's tables of g_mu_nu, g^mu^nu,
 * sqrt(-g), lapse at zone centres and lower face centres, and the connection at centres, on the device.
 * GRIM_MINKOWSKI: params ignored (geometry is compile-time constant in the kernels).
 * GRIM_KERR_MKS : params (host) = {a, h}, M = 1; Kerr-Schild transformed by eqs 5-8; X^1 = ln r, X^2 in [0,1].
 * Must be called before any compute call (GRIM_ESTATE otherwise). */
int grim_set_metric(grim_ctx *c, int32_t kind, const double *params, int32_t nparams);

/* Steps a1-a3 (L150-173 eqs 17; L99 eq 10; L438): reconstructs P_E to faces, forms LLF fluxes with face-centre
 * geometry (C-8), and writes the stage constant
 *     C = -U(P_n)/dt' + div F(P_E) - S^E(P_E)                                  (eq 19 / eq 13; C-5)
 * and, for EMHD, the three spatial-gradient terms G = (Xq, Xd, divx) of the relaxation targets (eqs 37-38; O-8).
 * Ghost zones of P_E must be filled (grim_fill_ghosts).  Only interior zones of C, G are written.
 *   P_E, P_n : N*Zg   C_out : N*Zg or NULL (context scratch)   G_out : 3*Zg or NULL (scratch; ignored for N=8)
 *   speeds_out : device double[4] or NULL: max over zones of c^d/dX^d (d=1..3) and of sum_d c^d/dX^d (C-15). */
int grim_compute_fluxes(grim_ctx *c, const double *P_E, const double *P_n, double dt_stage, double *C_out,
                        double *G_out, double *speeds_out);

/* Steps a4-a7 (L190-235 eqs 20-25): advances the Newton iteration of every interior zone whose status has no
 * terminal bit by at most `max_iters` iterations (<= 0: until terminal), in place.
 *   P_n, P_E : N*Zg   C : N*Zg or NULL (scratch of the last grim_compute_fluxes)   G : 3*Zg or NULL (same)
 *   P_iter : N*Zg, in: P^k, out: P^{k'}     resnorm : Zg, out: ||R(P^{k'})||_2
 *   status, iters : Zg int32 each, in/out (zero them to start a solve)
 *   n_active_out : host int64 or NULL: zones still without a terminal bit after the call (synchronises). */
int grim_newton_step(grim_ctx *c, const double *P_n, const double *P_E, const double *C, const double *G,
                     double dt_stage, int32_t max_iters, double *P_iter, double *resnorm, int32_t *status,
                     int32_t *iters, int64_t *n_active_out);

/* Steps a4-a7 as one fresh solve (what grim_timestep enqueues per stage): every interior zone starts from
 * P_guess with status = iters = 0 and iterates to a terminal status; the result goes to P_out (interior zones only;
 * ghost zones of P_out are not touched).  P_out may be P_guess, and it may be P_n: a zone's inputs are read before
 * its result is written and no other zone reads them.  resnorm, status, iters : Zg each or NULL (context scratch).
 * Other arguments as grim_newton_step.  Does not synchronise. */
int grim_newton_solve(grim_ctx *c, const double *P_n, const double *P_E, const double *C, const double *G,
                      double dt_stage, const double *P_guess, double *P_out, double *resnorm, int32_t *status,
                      int32_t *iters);

/* Standalone primitive recovery (O-10; BASELINE config 2): for each of nz zones solves
 * R(P) = (U(P) - U*)/||U*||_2 = 0 by the same Newton iteration, tol = rtol.
 *   U_target : N*nz flat
 *   geom : NULL (Minkowski), or the geometry of each zone, device double[15*nz], component-major [c*nz + z]:
 *          c = 0..9 g_mu_nu in the order 00 01 02 03 11 12 13 22 23 33, c = 10..12 g^{t1} g^{t2} g^{t3},
 *          c = 13 sqrt(-g), c = 14 the lapse alpha = 1/sqrt(-g^{tt}) (L248; C-9: beta^i/alpha = alpha g^{ti});
 *          tau_R is the descriptor's constant tau
 *   P_inout : N*nz, guess -> result   iters, status : nz int32, out   resnorm : nz, out
 * Zones are solved to a terminal status; the active set is compacted between iteration sweeps. */
int grim_invert_primitives(grim_ctx *c, int64_t nz, const double *U_target, const double *geom, double *P_inout,
                           int32_t *iters, int32_t *status, double *resnorm);

/* One time step (a8: L113-148, eq 19 then eq 13; O-11): ghost fill, stage 1 (P_E = P_n, dt' = dt/2, guess P_n),
 * ghost fill, stage 2 (P_E = P_{n+1/2}, dt' = dt, guess P_{n+1/2}); P_inout interior is overwritten by P_{n+1}.
 * Ghost zones of P_inout on return are those the first ghost fill gave P_n (every call refills them; ghosts of a
 * GRIM_BC_NONE side are the caller's and are used unchanged for both stages).
 *   dt <= 0: dt = cfl / max_z sum_d c^d/dX^d (C-15).   dt_used : host or NULL.   stats : host or NULL
 * (requesting dt_used or stats synchronises the stream). 
 * With dt > 0, dt_used == NULL and stats == NULL the call only enqueues work on the context's stream (no
 * synchronisation, no allocation once the context has run a step): it may be captured into a CUDA graph on that
 * stream and replayed (tests/test_gpu_host_pipeline.py). */
int grim_timestep(grim_ctx *c, double *P_inout, double dt, double *dt_used, grim_step_stats *stats);

/* ---- helpers beyond the six ------------------------------------------------------------------------------ */

void grim_free(grim_ctx *c);
const char *grim_last_error(const grim_ctx *c); /* NULL ctx: error of the last failed grim_init_grid or
                                                    grim_invert_primitives_static */
int grim_version(void);

/* Padded zone count Zg and padded extents (host out, may be NULL). */
int64_t grim_zones_padded(const grim_ctx *c, int32_t extents[3]);

/* Ghost fill in place (C-11): direction 1, then 2 (covering direction-1 ghosts), then 3. */
int grim_fill_ghosts(grim_ctx *c, double *P);

/* U(P) for nz flat zones, Minkowski (eqs 30-32, 39-42); used to build inversion workloads on the device. */
int grim_prim_to_conserved(grim_ctx *c, int64_t nz, const double *P, double *U);

/* Caller-supplied stationary metric independent of X^3 (the paper keeps geometry in a separate library, L339):
 * replaces the tables grim_set_metric would compute.  Both arguments HOST, SoA over the padded 2-D plane
 * idx2d = j*s1 + i (n2d = s1*s2 entries per component):
 *   tab  : [loc][comp][idx2d], loc = 0 centre, 1..3 lower face in direction loc; comp 0..9 = g_mu_nu in the
 *          order 00 01 02 03 11 12 13 22 23 33, 10..19 = g^mu^nu (same order), 20 = sqrt(-g), 21 = lapse,
 *          22 = tau_R (used when tau_mode == GRIM_TAU_R32; otherwise the descriptor's tau)      (4*23*n2d doubles)
 *   conn : [l*16 + m*4 + n][idx2d] = Gamma^l_{mn} at zone centres                                (64*n2d doubles)
 *          symmetric in (m, n): the kernels read the m <= n entries and use them for both orders
 * The library derives alpha g^{ti} (one multiplication per entry) and copies the rest unchanged.  Afterwards the
 * context behaves as after grim_set_metric(GRIM_KERR_MKS): general-metric kernels.  Synchronises. */
int grim_set_metric_tables(grim_ctx *c, const double *tab, const double *conn);

/* Copies the geometry of padded 2-D zone (j,i) -> idx2d = j*s1 + i to the HOST (parity tests of a0):
 * loc = 0 centre, 1..3 lower face in direction loc.  gcov, gcon: 16 doubles row-major; conn: 64 doubles
 * [l][m][n] = Gamma^l_{mn} (centre only; may be NULL).  Synchronises. */
int grim_get_geometry(grim_ctx *c, int32_t loc, int64_t idx2d, double *gcov, double *gcon, double *sqrtmg,
                      double *alpha, double *tau, double *conn);

/* ---- diagnostic entry points (measurement and self-test hooks; not steps of the path) ------------------------
 * grim_fp64_probe, grim_arith_selftest here, grim_launch_count / grim_set_timing / grim_get_timing at the end of
 * this header. */

/* fp64 pipe probe: runs `iters` dependent-chain-free DFMA (fma=1) or DMUL+DADD (fma=0) instructions per thread
 * on a full grid and returns fp64 instructions per second (host out).  Used for the ALU roofline denominator. */
int grim_fp64_probe(grim_ctx *c, int32_t fma, int32_t iters, double *inst_per_s);

/* Arithmetic self-test: the kernels form every fp64 quotient, reciprocal and square root
 * speculatively as straight-line code that is IEEE-754 correctly rounded for operands of magnitude in
 * [2^-480, 2^480), guarded by an exponent test, and replay a zone with the plain operators when a guard fails.
 * This call compares the speculative operations with the plain operators bit for bit on n pseudo-random operand
 * pairs on the device (wide = 0: exponents within +-400 of 1; wide = 1: the whole fp64 range with zeros, negative
 * numbers, subnormals, infinities and NaNs, where the guard must reject what the straight-line code gets wrong).
 * out6 (HOST): mismatches of [0] a/b, [1] 1/b, [2] sqrt(a), [3] a/60, [4] the zero-tolerant variants -- all must be
 * 0 -- and [5] the number of a/b samples the guard accepted.  Synchronises. */
int grim_arith_selftest(grim_ctx *c, int64_t n, int64_t seed, int32_t wide, int64_t *out6);

/* End-to-end variants taking HOST buffers (pinned or pageable): copy in, run on the device, copy out, on the
 * context's stream; they return after the stream is synchronised.  Device staging buffers belong to the context.
 *   grim_timestep_host          : P_host N*Zg in/out; runs nsteps time steps (dt <= 0: chosen per step from cfl).
 *                                 nsteps == 1 with dt > 0 on a 3-D grid of >= 64 X^3 planes and >= 1.5 M zones (no flux-CT, no
 *                                 GRIM_BC_NONE side): pipelined over slabs of X^3 planes -- copies of other slabs run
 *                                 on two more streams while a slab's kernels run; same bits as grim_timestep.  In
 *                                 that mode the ghost zones of P_host are neither read nor written (the boundary
 *                                 conditions fill them on the device); otherwise the whole padded array is copied.
 *                                 Environment GRIM_HOST_PIPELINE=0 / 1 (read at grim_init_grid): never / whenever the
 *                                 grid allows it, regardless of size.
 *   grim_invert_primitives_host : U_host, P_host N*nz; iters/status/resnorm host outputs (may be NULL). */
int grim_timestep_host(grim_ctx *c, double *P_host, int32_t nsteps, double dt, double *dt_used);
/* Which of the two forms the context's last grim_timestep_host call took (it depends on the grid, on the arguments and
 * on GRIM_HOST_PIPELINE, see above): callers that account for the bytes copied, or that rely on the ghost zones of
 * P_host having been copied, read it here instead of re-deriving the rule.  Host bookkeeping, no device work. */
enum { GRIM_HOST_MODE_NONE = 0, GRIM_HOST_MODE_WHOLE = 1, GRIM_HOST_MODE_PIPELINED = 2 };
int grim_last_host_mode(const grim_ctx *c);
int grim_invert_primitives_host(grim_ctx *c, int64_t nz, const double *U_host, double *P_host, int32_t *iters_host,
                                int32_t *status_host, double *resnorm_host);

/* ---- for callers that must not allocate device memory -------------------------------------------------------
 *
 * Every call above needs a grim_ctx, and grim_init_grid buys the context's scratch with cudaMalloc (so do
 * grim_invert_primitives and the *_host variants when their lists or staging buffers grow).  Some users of this
 * library cannot do that: a plug-in of a host application (a simulation code, a PyTorch process) whose own memory pool
 * has already claimed the device's memory at start-up, so that a cudaMalloc from a library either fails or takes
 * memory the pool has promised elsewhere; and a caller inside a time-critical loop, because cudaMalloc and cudaFree
 * wait for the whole device and stall the application's other streams.  Such a caller owns device buffers for its
 * inputs and outputs (carved from its pool) but can give the library nothing else.
 *
 * grim_invert_primitives_static is grim_invert_primitives (O-10, BASELINE config 2; same kernels' arithmetic, same
 * result bit for bit, zone for zone) for them: it takes no context and calls no cudaMalloc, cudaFree or any other
 * allocating routine, in any call, the first included.  The two active-zone lists and the counters that the sweeps
 * need live in a fixed array inside the library's device image (a file-scope `static __device__` array in
 * kernels_newton.cu) of 256 + 8 * GRIM_STATIC_MAX_ZONES bytes = 8 MiB + 256 B.  Every GPU on which this library is
 * loaded holds that array from the moment the CUDA module loads until the process exits, whether or not this entry
 * point is ever called.
 *
 *   d  : HOST.  Read: model, gamma, phi, psi, closure, tau, fd_eps, eps_bt, rtol, kmax, lsmax (validated as in
 *        grim_init_grid), device, stream.  The grid fields (n1.., ng, dim, extents, bc, recon, ...) are ignored.
 *   nz : zones, 0 <= nz <= GRIM_STATIC_MAX_ZONES; a larger nz is refused with GRIM_EINVAL and a message that states
 *        the limit (split the batch, or use grim_invert_primitives).  nz == 0 returns GRIM_OK and does nothing.
 *   U_target, geom, P_inout, iters, status, resnorm : DEVICE, the caller's, exactly as for grim_invert_primitives.
 *
 * Behaviour the caller must know:
 *   - The first call on each device looks up the device address of the array (cudaGetSymbolAddress) and raises the
 *     kernels' shared-memory limit, once, and remembers both per device.  Make that first call during set-up, before
 *     starting any stream capture on that device.
 *   - All calls in the process share the one array per device, and it keeps whatever the previous call left in it.  The
 *     entry point zeroes its counters itself before every sweep; the lists need no clearing (only the entries a sweep
 *     has just written are read).  Because the array is shared, two calls whose kernels overlap on the same GPU
 *     (different streams, or different host threads) race on it and corrupt each other's lists: serialise them.
 *   - d->device becomes the calling thread's current device.  The call enqueues on d->stream and returns after
 *     synchronising it (each sweep reads the number of zones still iterating back to the host).
 *   - Errors: GRIM_EINVAL / GRIM_ECUDA as elsewhere; the text is at grim_last_error(NULL).  No CPU fallback. */
#define GRIM_STATIC_MAX_ZONES (1 << 20)
int grim_invert_primitives_static(const grim_grid_desc *d, int64_t nz, const double *U_target, const double *geom,
                                  double *P_inout, int32_t *iters, int32_t *status, double *resnorm);

/* Diagnostic: number of kernels the library has launched on this context since creation (host bookkeeping). */
int64_t grim_launch_count(const grim_ctx *c);

/* Diagnostic: per-kernel-class device timing for the roofline report (bench.py): while on, every launch group is bracketed by
 * a CUDA event pair on the context's stream.  grim_set_timing(on != 0) clears the accumulators; grim_get_timing
 * waits for the recorded events and returns, per class, the summed device milliseconds and the launch count
 * (host out, GRIM_NKCLASS entries each, may be NULL).  Classes: */
enum { GRIM_K_GHOSTS = 0, GRIM_K_FLUX = 1, GRIM_K_NEWTON = 2, GRIM_K_INVERT = 3, GRIM_K_OTHER = 4, GRIM_NKCLASS = 5 };
int grim_set_timing(grim_ctx *c, int32_t on);
int grim_get_timing(grim_ctx *c, double *ms, int64_t *launches);

#ifdef __cplusplus
}
#endif
#endif /* GRIM_H */
