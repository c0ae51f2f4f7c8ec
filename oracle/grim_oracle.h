/*
 * grim_oracle.h -- ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT).
 *
 * A plain, slow, fp64 CPU statement of the hot path of grim (arXiv 1702.01106):
 * the combined time step + primitive-variable inversion solved per zone by
 * Newton-Raphson (PAPER.md sections 2-4).  Written from the paper alone; shares
 * no code with the CUDA library in paper_1702_01106_b200/csrc.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load it.  Citations "Lnnn" are line numbers of /root/reference/PAPER.md.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"):
 *   Table 1 null vector + eigenvalue (L484-499), Table 1 evolution at 2nd order
 *   (L499-507), ideal-MHD magnetosonic/Alfven closed forms, shock-table flux
 *   equality (L517-528), line-search closed form (eq 25), psi_max (L325),
 *   conservation, round trip, LU vs LAPACK, MP5/minmod exactness, Newton
 *   behaviour, geometry identities; flux-CT (og_flux_ct, L327-335): corner-centred
 *   div B at round-off in 2-D / 3-D, conservation, 1-D and uniform reductions
 *   (tests/test_oracle_fluxct.py); reduced solve (L148, L643): same root as the full
 *   solve, conservation, explicit induction step (tests/test_oracle_reduced.py).
 *   Curved space (tests/test_oracle_curved.py): og_geometric_source against (1/2) T^{kl} d_nu g_kl; the connection
 *   terms of the EMHD targets against brute-force covariant derivatives; og_stage_prepare + og_zone_residual on Kerr
 *   grids (2-D and 3-D, all rows, face-centre geometry, tau_R = r^{3/2}, the terms (1/2) q~ div u, (1/2) dP~ div u)
 *   by a manufactured solution converging at second order to the continuum equations; an exact static Tolman
 *   atmosphere with a monopole field in Schwarzschild staying stationary at second order; polar reflection against the
 *   analytic field at the mirrored coordinates.
 * Parity unpinned (no printed number or invariant separates the alternatives;
 * listed in DESIGN.md "Readings"): C-3 beyond 2nd-order agreement, C-4 same-state
 * closure, C-7, C-9 inside the ergosphere, C-11 (choice of boundary conditions and floors), C-15, C-16.
 */
#ifndef GRIM_ORACLE_H
#define GRIM_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* primitive ordering (L297): rho, u, u~^1..3, B^1..3, q, dP */
enum { OG_RHO = 0, OG_UU = 1, OG_U1 = 2, OG_U2 = 3, OG_U3 = 4,
       OG_B1 = 5, OG_B2 = 6, OG_B3 = 7, OG_Q = 8, OG_DP = 9, OG_NMAX = 10 };

enum { OG_MINKOWSKI = 0, OG_KERR_MKS = 1 };
enum { OG_MINMOD = 0, OG_MP5 = 1 };
enum { OG_LLF = 0, OG_HLLE = 1 };
enum { OG_BC_PERIODIC = 0, OG_BC_OUTFLOW = 1, OG_BC_REFLECT_POLAR = 2, OG_BC_NONE = 3 };
enum { OG_TAU_CONST = 0, OG_TAU_R32 = 1 };
enum { OG_CLOSURE_CS2TAU = 0, OG_CLOSURE_CONST = 1 };

/* status word per zone */
enum { OG_ST_CONVERGED = 1, OG_ST_KMAX = 2, OG_ST_LS_EXHAUSTED = 4,
       OG_ST_SINGULAR = 8, OG_ST_NONFINITE = 16 };
#define OG_ST_TERMINAL (OG_ST_CONVERGED | OG_ST_KMAX | OG_ST_SINGULAR | OG_ST_NONFINITE)

/* geometry of one evaluation point (zone centre or face centre) */
typedef struct {
  double gcov[4][4];
  double gcon[4][4];
  double sqrtmg;      /* sqrt(-g) */
  double alpha;       /* lapse 1/sqrt(-g^tt) */
} og_geom;

/* physics parameters */
typedef struct {
  int32_t nvar;       /* 8 ideal GRMHD, 10 EMHD */
  double  gam;        /* adiabatic index (L248) */
  double  phi, psi;   /* closure chi = phi cs^2 tau_R, nu = psi cs^2 tau_R (L299) */
  int32_t closure;    /* OG_CLOSURE_CS2TAU (L299) | OG_CLOSURE_CONST: chi = phi, nu = psi constants (L566) */
} og_model;

/* solver parameters (eqs 20-25; C-2, C-14, C-16) */
typedef struct {
  double  fd_eps;     /* eq 23 epsilon */
  double  eps_bt;     /* L223, 1e-4 */
  double  atol, rtol; /* stop when ||R||_2 < atol + rtol*scale */
  int32_t kmax, lsmax;
} og_solver;

typedef struct og_grid og_grid;

typedef struct {
  int32_t n1, n2, n3, ng, dim;
  double  xstart[3], xend[3];
  int32_t bc[3][2];
  int32_t nvar;
  int32_t recon; double limiter_theta;
  int32_t riemann;
  double  gam, phi, psi;
  int32_t tau_mode; double tau;
  double  fd_eps, eps_bt, atol, rtol;
  int32_t kmax, lsmax;
  double  cfl;
  int32_t flux_ct;    /* != 0: flux-CT averaging of the magnetic-field fluxes (PAPER.md 4.2, L327-335) */
  int32_t closure;    /* OG_CLOSURE_* */
  int32_t reduced;    /* != 0: the paper's own split (L148 "equations without implicitly coupled source terms are
                         treated explicitly", L643 "5 x 5 ... as opposed to a 7 x 7 Jacobian"): B^i advanced
                         explicitly, Newton on the nvar-3 other primitives */
} og_grid_desc;

typedef struct {
  int64_t zones;
  int64_t iters_hist[2][16];   /* [stage][min(iters,15)] */
  int64_t backtracks[2];
  int64_t unconverged[2];
  double  max_resnorm[2];      /* max over zones of ||R||_2 / scale */
} og_step_stats;

/* ---- point functions (each cites the passage it follows in grim_oracle.c) ---- */
void   og_geom_minkowski(og_geom *g);
void   og_geom_kerr_mks(double a, double h, double X1, double X2, og_geom *g);
void   og_conn_kerr_mks(double a, double h, double X1, double X2, double conn[4][4][4]);
void   og_prim_to_U(const og_model *m, const og_geom *g, double tau, const double *P, double *U);
void   og_prim_to_F(const og_model *m, const og_geom *g, double tau, int dir, const double *P, double *F);
double og_vmax2(const og_model *m, const og_geom *g, double tau, const double *P);
void   og_wave_speeds(const og_model *m, const og_geom *g, double tau, int dir, const double *P,
                      double *vplus, double *vminus);
double og_cmax(const og_model *m, const og_geom *g, double tau, int dir, const double *P);
void   og_derived(const og_model *m, const og_geom *g, const double *P,
                  double *Theta, double ucon[4], double ucov[4]);
void   og_emhd_targets(const og_model *m, const og_geom *g, const double conn[4][4][4], double tau,
                       const double *PE, const double dTheta[4], const double ducov[4][4],
                       double divu, double *q0, double *dP0);
void   og_rescale_factors(const og_model *m, double tau, const double *P, double *fq, double *fdp);
/* geometric source S_nu = sqrt(-g) T^kappa_lambda Gamma^lambda_{nu kappa}, nu = 0..3 (eq 31), the routine
   og_stage_prepare calls per zone; and T^mu_nu itself (eq 27 lowered, eqs 33-34) */
void   og_geometric_source(const og_model *m, const og_geom *g, const double conn[4][4][4], const double *P,
                           double S[4]);
void   og_stress_tensor(const og_model *m, const og_geom *g, const double *P, double T[4][4]);
double og_minmod3(double a, double b, double c);
double og_slope(double theta, double vm, double v0, double vp);
void   og_reconstruct(int recon, double theta, const double v[5], double *left_of_upper, double *right_of_lower);
double og_mp5_face(double vm2, double vm1, double v0, double vp1, double vp2);
int    og_lu_solve(int n, double *A /* n*n row-major, overwritten */, double *b /* rhs -> x */, int32_t *piv);
double og_linesearch_lambda(double f0, double flam, double lam);
void   og_llf(int n, const double *Fm, const double *Fp, const double *Um, const double *Up, double c, double *F);

/* ---- grid-level ---- */
og_grid *og_grid_create(const og_grid_desc *d);
void     og_grid_free(og_grid *g);
int      og_grid_set_metric(og_grid *g, int kind, const double *params, int nparams);
int64_t  og_grid_zones_padded(const og_grid *g);
void     og_fill_ghosts(const og_grid *g, double *P);
/* geometry tables as the oracle holds them (for the geometry parity test): padded 2-D [j][i] */
void     og_grid_get_geom(const og_grid *g, int loc /*0 centre,1..3 lower faces*/, int64_t idx2d, og_geom *out);
void     og_grid_get_conn(const og_grid *g, int64_t idx2d, double conn[4][4][4]);
double   og_grid_get_tau(const og_grid *g, int loc, int64_t idx2d);   /* tau_R of that evaluation point (C-11) */
/* Flux-CT (PAPER.md 4.2 L327-335: Toth 2000 as used in harm): face-centred electric fields F^j(B^i) -> simple
   average to the edges -> average back to the faces; F^d(B^d) = 0.  Fface[a]: nvar*zg face fluxes of direction a
   (NULL for an inactive direction), valid on faces whose index along a is in [ng, ng+n] and whose transverse
   indices are in [ng-1, ng+n]; on return the B^i entries hold the averaged fluxes on the faces of the interior
   zones.  The cell-corner-centred div B of Toth's scheme is then unchanged by the update to round-off. */
/* HLLE flux (eq 18): cR >= max(c, 0), cL >= max(-c, 0) over the speeds of both states;
   F = [cR F^- + cL F^+ - cR cL (U^+ - U^-)] / (cL + cR) */
void     og_hlle(int n, const double *Fm, const double *Fp, const double *Um, const double *Up, double cR, double cL,
                 double *F);
void     og_flux_ct(const og_grid *g, double *const Fface[3]);
/* stage constant C (nvar x Zg) and explicit EMHD gradient terms G (3 x Zg: Xq, Xd, divx) (L438).
   speeds[0..2] = max_z c^d/dX^d, speeds[3] = max_z sum_d c^d/dX^d */
void     og_stage_prepare(const og_grid *g, const double *Pn, const double *PE, double dt_stage,
                          double *C, double *G, double speeds[4]);
/* residual of one zone at trial state P (eq 19 / eq 13) */
void     og_zone_residual(const og_grid *g, int64_t z, const double *Pn, const double *PE,
                          const double *C, const double *G, double dt_stage, const double *P, double *R);
/* Newton iterations on all interior zones; max_iters_this_call <= 0 means run to completion */
int64_t  og_newton(const og_grid *g, const double *Pn, const double *PE, const double *C, const double *G,
                   double dt_stage, double *P_iter, int max_iters_this_call,
                   double *resnorm, int32_t *status, int32_t *iters, int64_t *backtracks);
double   og_choose_dt(const og_grid *g, const double *P);
void     og_timestep(const og_grid *g, double *P, double dt, og_step_stats *stats);
/* standalone inversion (O-10): flat SoA [v][z]; geom may be NULL (Minkowski) */
void     og_invert(const og_model *m, const og_solver *s, double tau, int64_t nz, const double *Ustar,
                   const og_geom *geom_or_null, double *P, int32_t *iters, int32_t *status,
                   double *resnorm, int64_t *backtracks);
/* one zone of Newton on a user residual with a linear model R = A P - b (pin P-11) is done in tests via og_lu_solve */
int      og_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
