/*
 * grim_oracle.c -- ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT).  See grim_oracle.h.
 *
 * Plain fp64, one zone at a time, in the paper's order and notation.  No blocking, no
 * fusion, no vectorisation tricks; OpenMP only over independent zones / faces.
 * Build: gcc -O2 -ffp-contract=off -fopenmp -fPIC -shared (oracle/build.py).
 * "Lnnn" = line of /root/reference/PAPER.md.  "C-n", "G-n", "O-n" = readings listed in
 * DESIGN.md (section "Readings of the paper").
 */
#include "grim_oracle.h"

#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int og_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ===================================================================================
 * Geometry (L68-89 eqs 5-8; C-10)
 * =================================================================================== */

static void invert4(const double a[4][4], double inv[4][4]) {
  /* Gauss-Jordan with partial pivoting on a 4x4 */
  double w[4][8];
  for (int i = 0; i < 4; i++)
    for (int j = 0; j < 4; j++) { w[i][j] = a[i][j]; w[i][4 + j] = (i == j) ? 1.0 : 0.0; }
  for (int c = 0; c < 4; c++) {
    int p = c;
    for (int r = c + 1; r < 4; r++) if (fabs(w[r][c]) > fabs(w[p][c])) p = r;
    if (p != c) for (int j = 0; j < 8; j++) { double t = w[c][j]; w[c][j] = w[p][j]; w[p][j] = t; }
    double d = w[c][c];
    for (int j = 0; j < 8; j++) w[c][j] /= d;
    for (int r = 0; r < 4; r++) if (r != c) {
      double f = w[r][c];
      for (int j = 0; j < 8; j++) w[r][j] -= f * w[c][j];
    }
  }
  for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) inv[i][j] = w[i][4 + j];
}

void og_geom_minkowski(og_geom *g) {
  memset(g, 0, sizeof(*g));
  g->gcov[0][0] = -1.0; g->gcon[0][0] = -1.0;
  for (int i = 1; i < 4; i++) { g->gcov[i][i] = 1.0; g->gcon[i][i] = 1.0; }
  g->sqrtmg = 1.0;
  g->alpha = 1.0;
}

/* Kerr-Schild metric (t,r,theta,phi), M=1, transformed to X^i by eqs 5-8: g_X = L^T g L with
 * L = diag(1, r, pi(1+(1-h)cos(2 pi X2)), 1).  Complex arguments so that the connection can be
 * taken by complex-step differentiation (exact to rounding; independent of the CUDA path's
 * dual numbers). */
static void kerr_mks_gcov_c(double a, double h, double complex X1, double complex X2,
                            double complex gc[4][4], double complex *sqrtmg) {
  double complex r = cexp(X1);                                            /* eq 5 */
  double complex th = M_PI * X2 + 0.5 * (1.0 - h) * csin(2.0 * M_PI * X2); /* eq 6 */
  double complex sth = csin(th), cth = ccos(th);
  /* C-21: faces on the polar axis (theta = 0, pi) have sin(theta) = 0 and a singular metric; floor |sin(theta)|
   * at 1e-20 there, so that g^{mu nu} stays finite while sqrt(-g) ~ 1e-20 shuts the flux through the axis off */
  if (cabs(sth) < 1e-20) sth = 1e-20;
  double complex s2 = sth * sth;
  double complex Sig = r * r + a * a * cth * cth;
  double complex f = 2.0 * r / Sig;
  double complex L[4] = {1.0, r, M_PI * (1.0 + (1.0 - h) * ccos(2.0 * M_PI * X2)), 1.0}; /* eq 8 */
  double complex k[4][4];
  memset(k, 0, sizeof(k));
  k[0][0] = -(1.0 - f);
  k[0][1] = k[1][0] = f;
  k[0][3] = k[3][0] = -a * f * s2;
  k[1][1] = 1.0 + f;
  k[1][3] = k[3][1] = -a * s2 * (1.0 + f);
  k[2][2] = Sig;
  k[3][3] = s2 * (Sig + a * a * s2 * (1.0 + f));
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) gc[m][n] = k[m][n] * L[m] * L[n];
  if (sqrtmg) *sqrtmg = Sig * sth * L[1] * L[2];   /* sqrt(-g) = Sigma sin(theta) |det L| */
}

void og_geom_kerr_mks(double a, double h, double X1, double X2, og_geom *g) {
  double complex gc[4][4], sg;
  kerr_mks_gcov_c(a, h, X1, X2, gc, &sg);
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) g->gcov[m][n] = creal(gc[m][n]);
  invert4(g->gcov, g->gcon);
  g->sqrtmg = fabs(creal(sg));
  g->alpha = 1.0 / sqrt(-g->gcon[0][0]);
}

/* Gamma^l_{mn} = 1/2 g^{lk} (d_m g_{kn} + d_n g_{km} - d_k g_{mn}); metric independent of t, X3 */
void og_conn_kerr_mks(double a, double h, double X1, double X2, double conn[4][4][4]) {
  const double hs = 1e-30;
  double dg[4][4][4]; /* dg[k][m][n] = d_k g_mn */
  memset(dg, 0, sizeof(dg));
  double complex gc[4][4];
  kerr_mks_gcov_c(a, h, X1 + I * hs, X2, gc, NULL);
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) dg[1][m][n] = cimag(gc[m][n]) / hs;
  kerr_mks_gcov_c(a, h, X1, X2 + I * hs, gc, NULL);
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) dg[2][m][n] = cimag(gc[m][n]) / hs;
  og_geom g;
  og_geom_kerr_mks(a, h, X1, X2, &g);
  for (int l = 0; l < 4; l++)
    for (int m = 0; m < 4; m++)
      for (int n = 0; n < 4; n++) {
        double s = 0.0;
        for (int k = 0; k < 4; k++) s += g.gcon[l][k] * (dg[m][k][n] + dg[n][k][m] - dg[k][m][n]);
        conn[l][m][n] = 0.5 * s;
      }
}

/* ===================================================================================
 * O-1  State from primitives (L41, L248, L297; C-9)
 * =================================================================================== */

typedef struct {
  double ucon[4], ucov[4], bcon[4], bcov[4], bsq;
} og_state;

static void get_state(const double *P, const og_geom *g, og_state *s) {
  const double *ut = &P[OG_U1];
  const double *B = &P[OG_B1];
  /* W = sqrt(1 + g_ij u~^i u~^j); u^t = W/alpha; u^i = u~^i - W beta^i/alpha, beta^i/alpha = alpha g^{ti} (C-9) */
  double usq = 0.0;
  for (int i = 1; i < 4; i++)
    for (int j = 1; j < 4; j++) usq += g->gcov[i][j] * ut[i - 1] * ut[j - 1];
  double W = sqrt(1.0 + usq);
  s->ucon[0] = W / g->alpha;
  for (int i = 1; i < 4; i++) s->ucon[i] = ut[i - 1] - W * (g->alpha * g->gcon[0][i]);
  for (int m = 0; m < 4; m++) {
    double v = 0.0;
    for (int n = 0; n < 4; n++) v += g->gcov[m][n] * s->ucon[n];
    s->ucov[m] = v;
  }
  /* b^t = B^i u^mu g_{i mu} = B^i u_i ; b^i = (B^i + b^t u^i)/u^t (L248) */
  double bt = 0.0;
  for (int i = 1; i < 4; i++) bt += B[i - 1] * s->ucov[i];
  s->bcon[0] = bt;
  double iut = 1.0 / s->ucon[0];
  for (int i = 1; i < 4; i++) s->bcon[i] = (B[i - 1] + bt * s->ucon[i]) * iut;
  for (int m = 0; m < 4; m++) {
    double v = 0.0;
    for (int n = 0; n < 4; n++) v += g->gcov[m][n] * s->bcon[n];
    s->bcov[m] = v;
  }
  double bsq = 0.0;
  for (int m = 0; m < 4; m++) bsq += s->bcon[m] * s->bcov[m];
  s->bsq = bsq;
}

/* thermodynamics and closure (L248, L283, eq 45 L311 / L501, L299) */
static double pressure(const og_model *m, const double *P) { return (m->gam - 1.0) * P[OG_UU]; }
static double temperature(const og_model *m, const double *P) { return pressure(m, P) / P[OG_RHO]; }
static double sound_speed2(const og_model *m, const double *P) {
  return m->gam * pressure(m, P) / (P[OG_RHO] + m->gam * P[OG_UU]);
}

/* Closure: thermal diffusivity chi and kinematic viscosity nu of state P.  OG_CLOSURE_CS2TAU: chi = phi cs^2 tau_R,
 * nu = psi cs^2 tau_R (L299).  OG_CLOSURE_CONST: constants chi = phi, nu = psi, as the anisotropic-conduction test
 * prescribes ("the thermal diffusivity chi = 0.01", L566). */
static void closure(const og_model *m, double tau, double cs2, double *chi, double *nu) {
  if (m->closure == OG_CLOSURE_CONST) { *chi = m->phi; *nu = m->psi; return; }
  *chi = m->phi * cs2 * tau;
  *nu = m->psi * cs2 * tau;
}

/* eqs 41-42 (L291-293): q~ = q sqrt(tau/(chi rho Theta^2)), dP~ = dP sqrt(tau/(nu rho Theta)); closure of
 * the same state P (C-4) */
void og_rescale_factors(const og_model *m, double tau, const double *P, double *fq, double *fdp) {
  double cs2 = sound_speed2(m, P);
  double chi, nu;
  closure(m, tau, cs2, &chi, &nu);
  double Th = temperature(m, P);
  *fq = sqrt(tau / (chi * P[OG_RHO] * Th * Th));
  *fdp = sqrt(tau / (nu * P[OG_RHO] * Th));
}

void og_derived(const og_model *m, const og_geom *g, const double *P, double *Theta, double ucon[4],
                double ucov[4]) {
  double Pf[OG_NMAX] = {0};
  memcpy(Pf, P, sizeof(double) * (size_t)m->nvar);
  og_state s;
  get_state(Pf, g, &s);
  *Theta = temperature(m, P);
  for (int i = 0; i < 4; i++) { ucon[i] = s.ucon[i]; ucov[i] = s.ucov[i]; }
}

/* ===================================================================================
 * O-2, O-3  Stress tensor, conserved variables, fluxes (eq 27, eqs 30-34, 39-42; G-3, G-7, C-18)
 * =================================================================================== */

/* row `mu` of T^mu_nu */
static void stress_row(const og_model *m, const double *P, const og_state *s, int mu, double T[4]) {
  double rho = P[OG_RHO], u = P[OG_UU];
  double Pg = pressure(m, P);
  double w = rho + u + Pg + s->bsq;
  double ptot = Pg + 0.5 * s->bsq;
  double bhcon[4], bhcov[4], q = 0.0, dP = 0.0;
  if (m->nvar == 10) {
    double ibn = 1.0 / sqrt(s->bsq);
    for (int i = 0; i < 4; i++) { bhcon[i] = s->bcon[i] * ibn; bhcov[i] = s->bcov[i] * ibn; }
    q = P[OG_Q]; dP = P[OG_DP];
  }
  for (int nu = 0; nu < 4; nu++) {
    double d = (mu == nu) ? 1.0 : 0.0;
    double t = w * s->ucon[mu] * s->ucov[nu] + ptot * d - s->bcon[mu] * s->bcov[nu];
    if (m->nvar == 10) {
      /* + q^mu u_nu + u^mu q_nu + Pi^mu_nu, q^mu = q bhat^mu, Pi = -dP (bhat bhat - h/3) (eqs 33-34) */
      t = t + q * (bhcon[mu] * s->ucov[nu] + s->ucon[mu] * bhcov[nu]);
      t = t - dP * (bhcon[mu] * bhcov[nu] - (1.0 / 3.0) * (d + s->ucon[mu] * s->ucov[nu]));
    }
    T[nu] = t;
  }
}

/* mu = 0: U(P); mu = 1..3: F^mu(P).  All multiplied by sqrt(-g). */
static void flux_vector(const og_model *m, const og_geom *g, double tau, int mu, const double *P,
                        const og_state *s, double *out) {
  double T[4];
  stress_row(m, P, s, mu, T);
  out[0] = g->sqrtmg * (P[OG_RHO] * s->ucon[mu]);                   /* eq 30 */
  for (int nu = 0; nu < 4; nu++) out[1 + nu] = g->sqrtmg * T[nu];   /* eq 31 */
  for (int i = 1; i < 4; i++) {                                     /* eq 32 with G-3's sign */
    if (mu == 0) out[4 + i] = g->sqrtmg * P[OG_B1 + i - 1];
    else out[4 + i] = g->sqrtmg * (s->bcon[i] * s->ucon[mu] - s->bcon[mu] * s->ucon[i]);
  }
  if (m->nvar == 10) {                                              /* eqs 39-42 */
    double fq, fdp;
    og_rescale_factors(m, tau, P, &fq, &fdp);
    out[8] = g->sqrtmg * ((P[OG_Q] * fq) * s->ucon[mu]);
    out[9] = g->sqrtmg * ((P[OG_DP] * fdp) * s->ucon[mu]);
  }
}

static void pad_prims(const og_model *m, const double *P, double *Pf) {
  for (int v = 0; v < OG_NMAX; v++) Pf[v] = (v < m->nvar) ? P[v] : 0.0;
}

void og_prim_to_U(const og_model *m, const og_geom *g, double tau, const double *P, double *U) {
  double Pf[OG_NMAX]; pad_prims(m, P, Pf);
  og_state s; get_state(Pf, g, &s);
  flux_vector(m, g, tau, 0, Pf, &s, U);
}

void og_prim_to_F(const og_model *m, const og_geom *g, double tau, int dir, const double *P, double *F) {
  double Pf[OG_NMAX]; pad_prims(m, P, Pf);
  og_state s; get_state(Pf, g, &s);
  flux_vector(m, g, tau, dir, Pf, &s, F);
}

/* ===================================================================================
 * O-4  Wave-speed bound (eqs 43-48; prose L303)
 * =================================================================================== */

static double vmax2_state(const og_model *m, double tau, const double *P, const og_state *s) {
  double rho = P[OG_RHO], u = P[OG_UU];
  double cs2 = sound_speed2(m, P);                         /* eq 45 */
  double va2 = s->bsq / (rho + m->gam * u + s->bsq);       /* eq 44 */
  double cst2 = cs2;
  if (m->nvar == 10) {
    double chi, nu;
    closure(m, tau, cs2, &chi, &nu);
    double vq2 = (m->gam - 1.0) * chi / tau;               /* eq 47 */
    double vdp2 = 4.0 * nu / (3.0 * tau);                  /* eq 48 */
    cst2 = 0.5 * (cs2 + vq2 + sqrt(cs2 * cs2 + vq2 * vq2)) + vdp2;  /* eq 46 */
  }
  return cst2 + va2 - cst2 * va2;                          /* eq 43 */
}

double og_vmax2(const og_model *m, const og_geom *g, double tau, const double *P) {
  double Pf[OG_NMAX]; pad_prims(m, P, Pf);
  og_state s; get_state(Pf, g, &s);
  return vmax2_state(m, tau, Pf, &s);
}

/* grid-frame speeds of waves moving at +-vmax in the fluid frame along direction dir (L303):
 * (k.u)^2 = vmax^2 (g^{mn} + u^m u^n) k_m k_n with k = (-v, delta^dir) */
static void wave_speeds_state(const og_model *m, const og_geom *g, double tau, int dir, const double *P,
                              const og_state *s, double *vplus, double *vminus) {
  double vm2 = vmax2_state(m, tau, P, s);
  double ut = s->ucon[0], ud = s->ucon[dir];
  double A = ut * ut - (g->gcon[0][0] + ut * ut) * vm2;
  double B = 2.0 * (ud * ut - (g->gcon[0][dir] + ud * ut) * vm2);
  double C = ud * ud - (g->gcon[dir][dir] + ud * ud) * vm2;
  double disc = sqrt(fmax(B * B - 4.0 * A * C, 0.0));
  double i2A = 1.0 / (2.0 * A);
  *vplus = (B + disc) * i2A;
  *vminus = (B - disc) * i2A;
}

void og_wave_speeds(const og_model *m, const og_geom *g, double tau, int dir, const double *P,
                    double *vplus, double *vminus) {
  double Pf[OG_NMAX]; pad_prims(m, P, Pf);
  og_state s; get_state(Pf, g, &s);
  wave_speeds_state(m, g, tau, dir, Pf, &s, vplus, vminus);
}

double og_cmax(const og_model *m, const og_geom *g, double tau, int dir, const double *P) {
  double vp, vm;
  og_wave_speeds(m, g, tau, dir, P, &vp, &vm);
  return fmax(fabs(vp), fabs(vm));
}

/* ===================================================================================
 * O-5  Reconstruction (L154-160, L115, L651; MP5: C-6)
 * =================================================================================== */

double og_minmod3(double a, double b, double c) {
  if (a > 0.0 && b > 0.0 && c > 0.0) return fmin(a, fmin(b, c));
  if (a < 0.0 && b < 0.0 && c < 0.0) return fmax(a, fmax(b, c));
  return 0.0;
}

/* generalised minmod slope on the 3-point stencil (L115) */
double og_slope(double theta, double vm, double v0, double vp) {
  return og_minmod3(theta * (v0 - vm), 0.5 * (vp - vm), theta * (vp - v0));
}

static double minmod2(double a, double b) {
  if (a > 0.0 && b > 0.0) return fmin(a, b);
  if (a < 0.0 && b < 0.0) return fmax(a, b);
  return 0.0;
}
static double minmod4(double a, double b, double c, double d) {
  if (a > 0.0 && b > 0.0 && c > 0.0 && d > 0.0) return fmin(fmin(a, b), fmin(c, d));
  if (a < 0.0 && b < 0.0 && c < 0.0 && d < 0.0) return fmax(fmax(a, b), fmax(c, d));
  return 0.0;
}

/* Suresh & Huynh 1997 MP5 value at the i+1/2 face from v_{i-2..i+2}, alpha = 4, eps = 1e-10 (C-6) */
double og_mp5_face(double vm2, double vm1, double v0, double vp1, double vp2) {
  const double alpha = 4.0, eps = 1e-10;
  double vor = (2.0 * vm2 - 13.0 * vm1 + 47.0 * v0 + 27.0 * vp1 - 3.0 * vp2) / 60.0;
  double vmp = v0 + minmod2(vp1 - v0, alpha * (v0 - vm1));
  if ((vor - v0) * (vor - vmp) <= eps) return vor;
  double dm1 = vm2 - 2.0 * vm1 + v0;
  double d0 = vm1 - 2.0 * v0 + vp1;
  double dp1 = v0 - 2.0 * vp1 + vp2;
  double dM4p = minmod4(4.0 * d0 - dp1, 4.0 * dp1 - d0, d0, dp1);    /* at i+1/2 */
  double dM4m = minmod4(4.0 * dm1 - d0, 4.0 * d0 - dm1, dm1, d0);    /* at i-1/2 */
  double vul = v0 + alpha * (v0 - vm1);
  double vav = 0.5 * (v0 + vp1);
  double vmd = vav - 0.5 * dM4p;
  double vlc = v0 + 0.5 * (v0 - vm1) + (4.0 / 3.0) * dM4m;
  double vmin = fmax(fmin(fmin(v0, vp1), vmd), fmin(fmin(v0, vul), vlc));
  double vmax = fmin(fmax(fmax(v0, vp1), vmd), fmax(fmax(v0, vul), vlc));
  return vor + minmod2(vmin - vor, vmax - vor);
}

/* v[0..4] = P_{i-2..i+2}.  left_of_upper = P^-_{i+1/2}, right_of_lower = P^+_{i-1/2} (L158) */
void og_reconstruct(int recon, double theta, const double v[5], double *left_of_upper, double *right_of_lower) {
  if (recon == OG_MP5) {
    *left_of_upper = og_mp5_face(v[0], v[1], v[2], v[3], v[4]);
    *right_of_lower = og_mp5_face(v[4], v[3], v[2], v[1], v[0]);
  } else {
    double s = og_slope(theta, v[1], v[2], v[3]);
    *left_of_upper = v[2] + 0.5 * s;
    *right_of_lower = v[2] - 0.5 * s;
  }
}

/* ===================================================================================
 * O-6  LLF flux (eq 17)
 * =================================================================================== */
void og_llf(int n, const double *Fm, const double *Fp, const double *Um, const double *Up, double c, double *F) {
  for (int v = 0; v < n; v++) F[v] = 0.5 * (Fp[v] + Fm[v]) - 0.5 * c * (Up[v] - Um[v]);
}

/* eq 18 (L170) */
void og_hlle(int n, const double *Fm, const double *Fp, const double *Um, const double *Up, double cR, double cL,
             double *F) {
  for (int v = 0; v < n; v++) F[v] = (cR * Fm[v] + cL * Fp[v] - cR * cL * (Up[v] - Um[v])) / (cL + cR);
}

/* ===================================================================================
 * O-9 pieces: dense LU with partial pivoting (eq 21; L434 "LAPACK" -> dgesv semantics; C-19),
 * line-search update (eq 25)
 * =================================================================================== */

/* Solves A x = b in place.  Row-major A.  pivot = first row of max |a_ik|, i >= k; multipliers formed with the
 * reciprocal of the pivot (as LAPACK's dgetf2 does); returns 0, or k+1 if pivot k is zero or non-finite. */
int og_lu_solve(int n, double *A, double *b, int32_t *piv) {
  double rinv[OG_NMAX > 16 ? OG_NMAX : 16];
  for (int k = 0; k < n; k++) {
    int p = k;
    double amax = fabs(A[k * n + k]);
    for (int i = k + 1; i < n; i++) {
      double v = fabs(A[i * n + k]);
      if (v > amax) { amax = v; p = i; }
    }
    if (piv) piv[k] = p;
    if (!(amax > 0.0) || !isfinite(amax)) return k + 1;
    if (p != k) {
      for (int j = 0; j < n; j++) { double t = A[k * n + j]; A[k * n + j] = A[p * n + j]; A[p * n + j] = t; }
      double t = b[k]; b[k] = b[p]; b[p] = t;
    }
    double r = 1.0 / A[k * n + k];
    rinv[k] = r;
    for (int i = k + 1; i < n; i++) {
      double l = A[i * n + k] * r;
      A[i * n + k] = l;
      for (int j = k + 1; j < n; j++) A[i * n + j] = A[i * n + j] - l * A[k * n + j];
      b[i] = b[i] - l * b[k];
    }
  }
  for (int i = n - 1; i >= 0; i--) {
    double s = b[i];
    for (int j = i + 1; j < n; j++) s = s - A[i * n + j] * b[j];
    b[i] = s * rinv[i];
  }
  return 0;
}

/* eq 25 (L230): minimiser of the quadratic through f(0), f'(0) = -2 f(0), f(lam) */
double og_linesearch_lambda(double f0, double flam, double lam) {
  return f0 / (flam + (2.0 * lam - 1.0) * f0) * lam * lam;
}

/* ===================================================================================
 * EMHD relaxation targets (eqs 37-38; G-5) split into the part carrying time derivatives and
 * the part carrying spatial derivatives and connection terms (O-8).  All coefficients at P_E.
 * =================================================================================== */

/* Tq = bhat^t D_t Theta + Theta u^t bhat^mu D_t u_mu ;  Td = bhat^t bhat^nu D_t u_nu */
static void emhd_time_part(const double bh[4], double ThE, double utE, double dtTheta, const double dtucov[4],
                           double *Tq, double *Td) {
  double bdu = 0.0;
  for (int mu = 0; mu < 4; mu++) bdu += bh[mu] * dtucov[mu];
  *Tq = bh[0] * dtTheta + ThE * (utE * bdu);
  *Td = bh[0] * bdu;
}

/* Xq = bhat^i d_i Theta + Theta bhat^mu (u^i d_i u_mu - Gamma^l_{nu mu} u^nu u_l)
 * Xd = bhat^i bhat^nu d_i u_nu - Gamma^l_{mu nu} bhat^mu bhat^nu u_l
 * dTheta[i], ducov[i][nu] for i = 1..3 (index 0 unused) */
static void emhd_space_part(const double bh[4], double ThE, const double ucon[4], const double ucov[4],
                            const double conn[4][4][4], const double dTheta[4], const double ducov[4][4],
                            double *Xq, double *Xd) {
  double bgradTh = 0.0;
  for (int i = 1; i < 4; i++) bgradTh += bh[i] * dTheta[i];
  double ba = 0.0, bbdu = 0.0;
  for (int mu = 0; mu < 4; mu++) {
    double a = 0.0;      /* spatial-derivative and connection part of a_mu */
    for (int i = 1; i < 4; i++) a += ucon[i] * ducov[i][mu];
    double gam = 0.0;
    for (int nu = 0; nu < 4; nu++)
      for (int l = 0; l < 4; l++) gam += conn[l][nu][mu] * ucon[nu] * ucov[l];
    ba += bh[mu] * (a - gam);
  }
  for (int i = 1; i < 4; i++) {
    double s = 0.0;
    for (int nu = 0; nu < 4; nu++) s += bh[nu] * ducov[i][nu];
    bbdu += bh[i] * s;
  }
  double gbb = 0.0;
  for (int mu = 0; mu < 4; mu++)
    for (int nu = 0; nu < 4; nu++)
      for (int l = 0; l < 4; l++) gbb += conn[l][mu][nu] * bh[mu] * bh[nu] * ucov[l];
  *Xq = bgradTh + ThE * ba;
  *Xd = bbdu - gbb;
}

typedef struct {
  double bh[4];       /* bhat^mu(P_E) */
  double ThE, utE;    /* Theta(P_E), u^t(P_E) */
  double rhochi, rhonu3; /* rho chi, 3 rho nu at P_E */
  double fqE, fdE;    /* rescale factors at P_E */
  double qtE, dtE;    /* q~(P_E), dP~(P_E) */
} emhd_coef;

static void emhd_coefficients(const og_model *m, const og_geom *g, double tau, const double *PE, emhd_coef *c,
                              og_state *sE) {
  get_state(PE, g, sE);
  double ibn = 1.0 / sqrt(sE->bsq);
  for (int i = 0; i < 4; i++) c->bh[i] = sE->bcon[i] * ibn;
  c->ThE = temperature(m, PE);
  c->utE = sE->ucon[0];
  double cs2 = sound_speed2(m, PE);
  double chi, nu;
  closure(m, tau, cs2, &chi, &nu);
  c->rhochi = PE[OG_RHO] * chi;
  c->rhonu3 = 3.0 * PE[OG_RHO] * nu;
  og_rescale_factors(m, tau, PE, &c->fqE, &c->fdE);
  c->qtE = PE[OG_Q] * c->fqE;
  c->dtE = PE[OG_DP] * c->fdE;
}

/* q0 = -rho chi (Tq + Xq) (eq 37) ; dP0 = 3 rho nu ((Td + Xd) - divu/3) (eq 38 with G-5) */
static void emhd_combine(const emhd_coef *c, double Tq, double Td, double Xq, double Xd, double divu,
                         double *q0, double *dP0) {
  *q0 = -c->rhochi * (Tq + Xq);
  *dP0 = c->rhonu3 * ((Td + Xd) - (1.0 / 3.0) * divu);
}

/* full-gradient entry point used by the linear-theory pin (P-1): dTheta[mu] = d_mu Theta,
 * ducov[mu][nu] = d_mu u_nu, divu = nabla_mu u^mu */
void og_emhd_targets(const og_model *m, const og_geom *g, const double conn[4][4][4], double tau,
                     const double *PE, const double dTheta[4], const double ducov[4][4], double divu,
                     double *q0, double *dP0) {
  emhd_coef c; og_state sE;
  emhd_coefficients(m, g, tau, PE, &c, &sE);
  double Tq, Td, Xq, Xd;
  emhd_time_part(c.bh, c.ThE, c.utE, dTheta[0], ducov[0], &Tq, &Td);
  emhd_space_part(c.bh, c.ThE, sE.ucon, sE.ucov, conn, dTheta, ducov, &Xq, &Xd);
  emhd_combine(&c, Tq, Td, Xq, Xd, divu, q0, dP0);
}

/* ===================================================================================
 * Grid (L400-408; G-9): SoA P[v][k][j][i], X1 fastest, ghosts on both sides of active dimensions
 * =================================================================================== */

struct og_grid {
  og_grid_desc d;
  og_model m;
  og_solver s;
  int n[3], ngd[3], sz[3];
  int64_t zg;           /* padded zones */
  int64_t n2d;          /* sz[1]*sz[0] */
  double dx[3], idx[3];
  int metric;
  og_geom *geomC;       /* [n2d] centre */
  og_geom *geomF[3];    /* [n2d] lower face in direction d */
  double (*conn)[4][4][4];
  double *tauC, *tauF[3];
};

static inline int64_t zidx(const og_grid *g, int i, int j, int k) {
  return ((int64_t)k * g->sz[1] + j) * g->sz[0] + i;
}

og_grid *og_grid_create(const og_grid_desc *d) {
  og_grid *g = (og_grid *)calloc(1, sizeof(og_grid));
  g->d = *d;
  g->m.nvar = d->nvar; g->m.gam = d->gam; g->m.phi = d->phi; g->m.psi = d->psi; g->m.closure = d->closure;
  g->s.fd_eps = d->fd_eps; g->s.eps_bt = d->eps_bt; g->s.atol = d->atol; g->s.rtol = d->rtol;
  g->s.kmax = d->kmax; g->s.lsmax = d->lsmax;
  g->n[0] = d->n1; g->n[1] = d->n2; g->n[2] = d->n3;
  for (int a = 0; a < 3; a++) {
    g->ngd[a] = (a < d->dim) ? d->ng : 0;
    g->sz[a] = g->n[a] + 2 * g->ngd[a];
    g->dx[a] = (d->xend[a] - d->xstart[a]) / g->n[a];     /* L70 */
    g->idx[a] = 1.0 / g->dx[a];
  }
  g->zg = (int64_t)g->sz[0] * g->sz[1] * g->sz[2];
  g->n2d = (int64_t)g->sz[0] * g->sz[1];
  g->metric = -1;
  return g;
}

void og_grid_free(og_grid *g) {
  if (!g) return;
  free(g->geomC); free(g->conn); free(g->tauC);
  for (int a = 0; a < 3; a++) { free(g->geomF[a]); free(g->tauF[a]); }
  free(g);
}

int64_t og_grid_zones_padded(const og_grid *g) { return g->zg; }

static double tau_at(const og_grid *g, double X1) {
  if (g->d.tau_mode == OG_TAU_R32) { double r = exp(X1); return r * sqrt(r); }   /* C-11: tau_R = r^{3/2} */
  return g->d.tau;
}

/* params: Kerr {a, h} */
int og_grid_set_metric(og_grid *g, int kind, const double *params, int nparams) {
  if (kind == OG_KERR_MKS && nparams < 2) return -1;
  g->metric = kind;
  g->geomC = (og_geom *)malloc(sizeof(og_geom) * (size_t)g->n2d);
  g->conn = malloc(sizeof(double[4][4][4]) * (size_t)g->n2d);
  g->tauC = (double *)malloc(sizeof(double) * (size_t)g->n2d);
  for (int a = 0; a < 3; a++) {
    g->geomF[a] = (og_geom *)malloc(sizeof(og_geom) * (size_t)g->n2d);
    g->tauF[a] = (double *)malloc(sizeof(double) * (size_t)g->n2d);
  }
  for (int j = 0; j < g->sz[1]; j++)
    for (int i = 0; i < g->sz[0]; i++) {
      int64_t id = (int64_t)j * g->sz[0] + i;
      double X1 = g->d.xstart[0] + (i - g->ngd[0] + 0.5) * g->dx[0];
      double X2 = g->d.xstart[1] + (j - g->ngd[1] + 0.5) * g->dx[1];
      double X1f = g->d.xstart[0] + (i - g->ngd[0]) * g->dx[0];
      double X2f = g->d.xstart[1] + (j - g->ngd[1]) * g->dx[1];
      if (kind == OG_MINKOWSKI) {
        og_geom_minkowski(&g->geomC[id]);
        for (int a = 0; a < 3; a++) og_geom_minkowski(&g->geomF[a][id]);
        memset(g->conn[id], 0, sizeof(double[4][4][4]));
        g->tauC[id] = g->d.tau;
        for (int a = 0; a < 3; a++) g->tauF[a][id] = g->d.tau;
      } else {
        double a_ = params[0], h_ = params[1];
        og_geom_kerr_mks(a_, h_, X1, X2, &g->geomC[id]);
        og_geom_kerr_mks(a_, h_, X1f, X2, &g->geomF[0][id]);
        og_geom_kerr_mks(a_, h_, X1, X2f, &g->geomF[1][id]);
        g->geomF[2][id] = g->geomC[id];                 /* metric independent of X3 */
        og_conn_kerr_mks(a_, h_, X1, X2, g->conn[id]);
        g->tauC[id] = tau_at(g, X1);
        g->tauF[0][id] = tau_at(g, X1f);
        g->tauF[1][id] = tau_at(g, X1);
        g->tauF[2][id] = tau_at(g, X1);
      }
    }
  return 0;
}

void og_grid_get_geom(const og_grid *g, int loc, int64_t idx2d, og_geom *out) {
  *out = (loc == 0) ? g->geomC[idx2d] : g->geomF[loc - 1][idx2d];
}
void og_grid_get_conn(const og_grid *g, int64_t idx2d, double conn[4][4][4]) {
  memcpy(conn, g->conn[idx2d], sizeof(double[4][4][4]));
}
double og_grid_get_tau(const og_grid *g, int loc, int64_t idx2d) {
  return (loc == 0) ? g->tauC[idx2d] : g->tauF[loc - 1][idx2d];
}

/* Ghost fill (C-11): periodic / outflow (copy) / polar reflection (sign flip of the X2 components) / none.
 * Direction 1 first, then 2 (covering direction-1 ghosts), then 3. */
void og_fill_ghosts(const og_grid *g, double *P) {
  for (int a = 0; a < 3; a++) {
    int ng = g->ngd[a];
    if (ng == 0) continue;
    int n = g->n[a];
    for (int side = 0; side < 2; side++) {
      int bc = g->d.bc[a][side];
      if (bc == OG_BC_NONE) continue;
      for (int v = 0; v < g->m.nvar; v++) {
        double *Pv = P + (int64_t)v * g->zg;
        double sign = 1.0;
        if (bc == OG_BC_REFLECT_POLAR && (v == OG_U1 + a || v == OG_B1 + a)) sign = -1.0;
        /* loop over the two other directions fully (padded extents already filled for lower directions) */
        int lo[3] = {0, 0, 0}, hi[3] = {g->sz[0], g->sz[1], g->sz[2]};
        for (int gz = 0; gz < ng; gz++) {
          int dst = side == 0 ? (ng - 1 - gz) : (ng + n + gz);
          int src;
          if (bc == OG_BC_PERIODIC) src = side == 0 ? (ng + n - 1 - gz) : (ng + gz);
          else if (bc == OG_BC_OUTFLOW) src = side == 0 ? ng : (ng + n - 1);
          else src = side == 0 ? (ng + gz) : (ng + n - 1 - gz);
          lo[a] = dst; hi[a] = dst + 1;
          for (int k = lo[2]; k < hi[2]; k++)
            for (int j = lo[1]; j < hi[1]; j++)
              for (int i = lo[0]; i < hi[0]; i++) {
                int c[3] = {i, j, k};
                c[a] = src;
                Pv[zidx(g, i, j, k)] = sign * Pv[zidx(g, c[0], c[1], c[2])];
              }
        }
      }
    }
  }
}

static void load_prims(const og_grid *g, const double *P, int64_t z, double *out) {
  for (int v = 0; v < OG_NMAX; v++) out[v] = (v < g->m.nvar) ? P[(int64_t)v * g->zg + z] : 0.0;
}

/* ===================================================================================
 * O-5..O-7  Face fluxes and flux divergence (eq 10; C-8 face-centre geometry)
 * =================================================================================== */

/* LLF flux through the lower face, in direction dir (0..2), of zone (i,j,k); also the face speed c */
static void face_flux(const og_grid *g, const double *PE, int dir, int i, int j, int k, double *F, double *cface) {
  int nv = g->m.nvar;
  int st[3] = {0, 0, 0};
  st[dir] = 1;
  double Pm[OG_NMAX] = {0}, Pp[OG_NMAX] = {0};    /* P^- (from zone i-1), P^+ (from zone i) at the face */
  for (int v = 0; v < nv; v++) {
    const double *Pv = PE + (int64_t)v * g->zg;
    double sten[5], lu, rl;
    /* zone i-1: its stencil i-3..i+1; P^- = its left_of_upper */
    for (int s = 0; s < 5; s++) {
      int o = s - 3;
      int ok = (g->d.recon == OG_MP5) || (s >= 1 && s <= 3);
      sten[s] = ok ? Pv[zidx(g, i + o * st[0], j + o * st[1], k + o * st[2])] : 0.0;
    }
    og_reconstruct(g->d.recon, g->d.limiter_theta, sten, &lu, &rl);
    Pm[v] = lu;
    /* zone i: its stencil i-2..i+2; P^+ = its right_of_lower */
    for (int s = 0; s < 5; s++) {
      int o = s - 2;
      int ok = (g->d.recon == OG_MP5) || (s >= 1 && s <= 3);
      sten[s] = ok ? Pv[zidx(g, i + o * st[0], j + o * st[1], k + o * st[2])] : 0.0;
    }
    og_reconstruct(g->d.recon, g->d.limiter_theta, sten, &lu, &rl);
    Pp[v] = rl;
  }
  int64_t id = (int64_t)j * g->sz[0] + i;
  const og_geom *gf = &g->geomF[dir][id];
  double tau = g->tauF[dir][id];
  og_state sm, sp;
  get_state(Pm, gf, &sm);
  get_state(Pp, gf, &sp);
  double Um[OG_NMAX], Up[OG_NMAX], Fm[OG_NMAX], Fp[OG_NMAX];
  flux_vector(&g->m, gf, tau, 0, Pm, &sm, Um);
  flux_vector(&g->m, gf, tau, 0, Pp, &sp, Up);
  flux_vector(&g->m, gf, tau, dir + 1, Pm, &sm, Fm);
  flux_vector(&g->m, gf, tau, dir + 1, Pp, &sp, Fp);
  double vp, vm, vp2, vm2;
  wave_speeds_state(&g->m, gf, tau, dir + 1, Pm, &sm, &vp, &vm);
  double cm = fmax(fabs(vp), fabs(vm));
  wave_speeds_state(&g->m, gf, tau, dir + 1, Pp, &sp, &vp2, &vm2);
  double cp = fmax(fabs(vp2), fabs(vm2));
  double c = fmax(cm, cp);                     /* L164: c_max >= max |c^+-| over both states */
  if (g->d.riemann == OG_HLLE) {               /* L168: bounds on the right- and left-going speeds of both states */
    double cR = fmax(0.0, fmax(fmax(vp, vm), fmax(vp2, vm2)));
    double cL = fmax(0.0, fmax(fmax(-vp, -vm), fmax(-vp2, -vm2)));
    og_hlle(nv, Fm, Fp, Um, Up, cR, cL, F);
  } else {
    og_llf(nv, Fm, Fp, Um, Up, c, F);
  }
  *cface = c;
}

/* ===================================================================================
 * NEXT-1  Flux-CT (section 4.2).  The paper names the scheme (Toth 2000, "also being used in
 * the harm code", simple averaging without upwinding) and does not print it; this is that scheme:
 *   edge (i-1/2, j-1/2, k):  E3 = [F1(B2)(i,j) + F1(B2)(i,j-1) - F2(B1)(i,j) - F2(B1)(i-1,j)] / 4
 *   edge (i, j-1/2, k-1/2):  E1 = [F2(B3)(j,k) + F2(B3)(j,k-1) - F3(B2)(j,k) - F3(B2)(j-1,k)] / 4
 *   edge (i-1/2, j, k-1/2):  E2 = [F3(B1)(k,i) + F3(B1)(k,i-1) - F1(B3)(k,i) - F1(B3)(k-1,i)] / 4
 *   F1(B1) = 0, F1(B2)(i,j,k) =  [E3(i,j,k) + E3(i,j+1,k)]/2, F1(B3)(i,j,k) = -[E2(i,j,k) + E2(i,j,k+1)]/2
 *   F2(B2) = 0, F2(B3)(i,j,k) =  [E1(i,j,k) + E1(i,j,k+1)]/2, F2(B1)(i,j,k) = -[E3(i,j,k) + E3(i+1,j,k)]/2
 *   F3(B3) = 0, F3(B1)(i,j,k) =  [E2(i,j,k) + E2(i+1,j,k)]/2, F3(B2)(i,j,k) = -[E1(i,j,k) + E1(i,j+1,k)]/2
 * with F^j(B^i) = sqrt(-g)(b^i u^j - b^j u^i) (eq 32, G-3), so that F1(B2) = -F2(B1) etc. are the same edge field
 * seen from two faces.  A pair whose second direction is inactive (2-D: E1, E2) is left out and the fluxes it
 * would replace stay as the Riemann solver gave them.
 * =================================================================================== */
void og_flux_ct(const og_grid *g, double *const Fface[3]) {
  const int64_t zg = g->zg;
  const int act[3] = {g->ngd[0] > 0, g->ngd[1] > 0, g->ngd[2] > 0};
  int lo[3], hi[3];                      /* edges: every active index in [ng, ng+n] */
  for (int a = 0; a < 3; a++) { lo[a] = g->ngd[a]; hi[a] = g->ngd[a] + g->n[a] + (act[a] ? 1 : 0); }
  const int64_t st[3] = {1, g->sz[0], (int64_t)g->sz[0] * g->sz[1]};
  double *E[3] = {NULL, NULL, NULL};
  /* E[c]: edge field along direction c, from the fluxes of the two directions a, b = c+1, c+2 (cyclic) */
  for (int c = 0; c < 3; c++) {
    int a = (c + 1) % 3, b = (c + 2) % 3;
    if (!act[a] || !act[b]) continue;
    E[c] = (double *)calloc((size_t)zg, sizeof(double));
    const double *Fa_Bb = Fface[a] + (int64_t)(OG_B1 + b) * zg;   /* F^a(B^b) */
    const double *Fb_Ba = Fface[b] + (int64_t)(OG_B1 + a) * zg;   /* F^b(B^a) = -F^a(B^b) at the same point */
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = lo[2]; k < hi[2]; k++)
      for (int j = lo[1]; j < hi[1]; j++)
        for (int i = lo[0]; i < hi[0]; i++) {
          int64_t z = zidx(g, i, j, k);
          E[c][z] = 0.25 * (Fa_Bb[z] + Fa_Bb[z - st[b]] - Fb_Ba[z] - Fb_Ba[z - st[a]]);
        }
  }
  /* back to the faces of the interior zones */
  for (int a = 0; a < 3; a++) {
    if (!act[a]) continue;
    int b = (a + 1) % 3, c = (a + 2) % 3;   /* F^a(B^b) = +avg_b E[c];  F^a(B^c) = -avg_c E[b] */
    double *Fa_Ba = Fface[a] + (int64_t)(OG_B1 + a) * zg;
    double *Fa_Bb = Fface[a] + (int64_t)(OG_B1 + b) * zg;
    double *Fa_Bc = Fface[a] + (int64_t)(OG_B1 + c) * zg;
    int fh[3] = {g->ngd[0] + g->n[0], g->ngd[1] + g->n[1], g->ngd[2] + g->n[2]};
    fh[a] += 1;
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = g->ngd[2]; k < fh[2]; k++)
      for (int j = g->ngd[1]; j < fh[1]; j++)
        for (int i = g->ngd[0]; i < fh[0]; i++) {
          int64_t z = zidx(g, i, j, k);
          Fa_Ba[z] = 0.0;
          if (E[c]) Fa_Bb[z] = 0.5 * (E[c][z] + E[c][z + st[b]]);
          if (E[b]) Fa_Bc[z] = -(0.5 * (E[b][z] + E[b][z + st[c]]));
        }
  }
  for (int c = 0; c < 3; c++) free(E[c]);
}

/* Geometric source of the energy-momentum equations (eq 31): S_nu = sqrt(-g) T^kappa_lambda Gamma^lambda_{nu kappa},
 * nu = 0..3, conn[l][m][n] = Gamma^l_{mn}.  (For the Levi-Civita connection this equals
 * (1/2) sqrt(-g) T^{kappa lambda} d_nu g_{kappa lambda}, which is what tests/test_oracle_curved.py pins it with.) */
static void geometric_source(const og_model *m, const og_geom *gc, const double conn[4][4][4], const double *P,
                             const og_state *s, double S[4]) {
  double T[4][4];
  for (int mu = 0; mu < 4; mu++) stress_row(m, P, s, mu, T[mu]);
  for (int nu = 0; nu < 4; nu++) {
    double acc = 0.0;
    for (int kk = 0; kk < 4; kk++)
      for (int l = 0; l < 4; l++) acc += T[kk][l] * conn[l][nu][kk];
    S[nu] = gc->sqrtmg * acc;
  }
}

/* the same at a point: P padded to OG_NMAX entries is not required (nvar of the model are read) */
void og_geometric_source(const og_model *m, const og_geom *g, const double conn[4][4][4], const double *P,
                         double S[4]) {
  double Pf[OG_NMAX];
  pad_prims(m, P, Pf);
  og_state s;
  get_state(Pf, g, &s);
  geometric_source(m, g, conn, Pf, &s, S);
}

/* T^mu_nu of state P (eq 27 lowered; eqs 33-34), row-major T[mu][nu] */
void og_stress_tensor(const og_model *m, const og_geom *g, const double *P, double T[4][4]) {
  double Pf[OG_NMAX];
  pad_prims(m, P, Pf);
  og_state s;
  get_state(Pf, g, &s);
  for (int mu = 0; mu < 4; mu++) stress_row(m, Pf, &s, mu, T[mu]);
}

/* ===================================================================================
 * O-8  Stage precompute: C = -U(P_n)/dt' + divF(P_E) - S^E(P_E) and the spatial-gradient terms of
 * the EMHD sources (L438, eq 19, eq 13; C-5)
 * =================================================================================== */
void og_stage_prepare(const og_grid *g, const double *Pn, const double *PE, double dt_stage, double *C,
                      double *G, double speeds[4]) {
  int nv = g->m.nvar;
  int64_t zg = g->zg;
  double idt = 1.0 / dt_stage;
  double *Fface[3] = {NULL, NULL, NULL};
  double *cface[3] = {NULL, NULL, NULL};
  for (int a = 0; a < 3; a++) {
    if (g->ngd[a] == 0) continue;
    Fface[a] = (double *)calloc((size_t)(nv * zg), sizeof(double));
    cface[a] = (double *)calloc((size_t)zg, sizeof(double));
    int lo[3] = {g->ngd[0], g->ngd[1], g->ngd[2]};
    int hi[3] = {g->ngd[0] + g->n[0], g->ngd[1] + g->n[1], g->ngd[2] + g->n[2]};
    hi[a] += 1;
    if (g->d.flux_ct)                     /* the edge averages reach one face into the transverse ghost zones */
      for (int b = 0; b < 3; b++)
        if (b != a && g->ngd[b] > 0) { lo[b] -= 1; hi[b] += 1; }
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = lo[2]; k < hi[2]; k++)
      for (int j = lo[1]; j < hi[1]; j++)
        for (int i = lo[0]; i < hi[0]; i++) {
          double F[OG_NMAX], c;
          face_flux(g, PE, a, i, j, k, F, &c);
          int64_t z = zidx(g, i, j, k);
          for (int v = 0; v < nv; v++) Fface[a][(int64_t)v * zg + z] = F[v];
          cface[a][z] = c;
        }
  }
  if (g->d.flux_ct) og_flux_ct(g, Fface);
  double smax[4] = {0, 0, 0, 0};
#pragma omp parallel
  {
    double lmax[4] = {0, 0, 0, 0};
#pragma omp for collapse(2) schedule(static)
    for (int k = g->ngd[2]; k < g->ngd[2] + g->n[2]; k++)
      for (int j = g->ngd[1]; j < g->ngd[1] + g->n[1]; j++)
        for (int i = g->ngd[0]; i < g->ngd[0] + g->n[0]; i++) {
          int64_t z = zidx(g, i, j, k);
          int64_t id = (int64_t)j * g->sz[0] + i;
          const og_geom *gc = &g->geomC[id];
          double tau = g->tauC[id];
          double Pn_z[OG_NMAX], PE_z[OG_NMAX], Un[OG_NMAX];
          load_prims(g, Pn, z, Pn_z);
          load_prims(g, PE, z, PE_z);
          og_state sn, sE;
          get_state(Pn_z, gc, &sn);
          get_state(PE_z, gc, &sE);
          flux_vector(&g->m, gc, tau, 0, Pn_z, &sn, Un);
          /* flux divergence (eq 10) */
          double divF[OG_NMAX] = {0};
          double ssum = 0.0;
          for (int a = 0; a < 3; a++) {
            if (g->ngd[a] == 0) continue;
            int c3[3] = {i, j, k};
            c3[a] += 1;
            int64_t zu = zidx(g, c3[0], c3[1], c3[2]);
            for (int v = 0; v < nv; v++)
              divF[v] += (Fface[a][(int64_t)v * zg + zu] - Fface[a][(int64_t)v * zg + z]) * g->idx[a];
            double cz = fmax(cface[a][z], cface[a][zu]) * g->idx[a];
            if (cz > lmax[a]) lmax[a] = cz;
            ssum += cz;
          }
          if (ssum > lmax[3]) lmax[3] = ssum;
          /* explicit geometric source sqrt(-g) T^k_l Gamma^l_{nu k} at P_E (eq 31; C-5) */
          double SE[OG_NMAX] = {0};
          if (g->metric != OG_MINKOWSKI) geometric_source(&g->m, gc, g->conn[id], PE_z, &sE, SE + 1);
          for (int v = 0; v < nv; v++) C[(int64_t)v * zg + z] = -Un[v] * idt + divF[v] - SE[v];
          /* spatial-gradient parts of the EMHD sources: limited 3-point slopes of derived quantities (L115) */
          if (nv == 10) {
            double dTheta[4] = {0}, ducov[4][4] = {{0}};
            double divx = 0.0;
            for (int a = 0; a < 3; a++) {
              if (g->ngd[a] == 0) continue;
              int cm[3] = {i, j, k}, cp[3] = {i, j, k};
              cm[a] -= 1; cp[a] += 1;
              int64_t zm = zidx(g, cm[0], cm[1], cm[2]), zp = zidx(g, cp[0], cp[1], cp[2]);
              int64_t idm = (int64_t)cm[1] * g->sz[0] + cm[0], idp = (int64_t)cp[1] * g->sz[0] + cp[0];
              double Pm_[OG_NMAX], Pp_[OG_NMAX];
              load_prims(g, PE, zm, Pm_);
              load_prims(g, PE, zp, Pp_);
              og_state sm_, sp_;
              get_state(Pm_, &g->geomC[idm], &sm_);
              get_state(Pp_, &g->geomC[idp], &sp_);
              double th = g->d.limiter_theta;
              dTheta[a + 1] = og_slope(th, temperature(&g->m, Pm_), temperature(&g->m, PE_z),
                                       temperature(&g->m, Pp_)) * g->idx[a];
              for (int nu = 0; nu < 4; nu++)
                ducov[a + 1][nu] = og_slope(th, sm_.ucov[nu], sE.ucov[nu], sp_.ucov[nu]) * g->idx[a];
              divx += og_slope(th, g->geomC[idm].sqrtmg * sm_.ucon[a + 1], gc->sqrtmg * sE.ucon[a + 1],
                               g->geomC[idp].sqrtmg * sp_.ucon[a + 1]) * g->idx[a];
            }
            divx = divx / gc->sqrtmg;
            emhd_coef c; og_state sE2;
            emhd_coefficients(&g->m, gc, tau, PE_z, &c, &sE2);
            double Xq, Xd;
            emhd_space_part(c.bh, c.ThE, sE.ucon, sE.ucov, g->conn[id], dTheta, ducov, &Xq, &Xd);
            G[0 * zg + z] = Xq;
            G[1 * zg + z] = Xd;
            G[2 * zg + z] = divx;
          }
        }
#pragma omp critical
    for (int a = 0; a < 4; a++) if (lmax[a] > smax[a]) smax[a] = lmax[a];
  }
  if (speeds) for (int a = 0; a < 4; a++) speeds[a] = smax[a];
  for (int a = 0; a < 3; a++) { free(Fface[a]); free(cface[a]); }
}

/* ===================================================================================
 * O-8  Residual of one zone (eq 19 half step / eq 13 full step; eqs 15-16; eqs 39-40; C-3)
 * =================================================================================== */

typedef struct {
  const og_model *m;
  const og_geom *gc;
  double tau, idt;
  double C[OG_NMAX];
  int emhd;
  /* P_n-derived */
  double Thn, ucovn[4], utn, qtn, dtn;
  /* P_E-derived + gradient terms */
  emhd_coef c;
  double Xq, Xd, divx;
  double scale;       /* ||U(P_n)||_2 / dt' (C-2) */
} zone_ctx;

static void zone_setup(const og_grid *g, int64_t z, int64_t id2d, const double *Pn, const double *PE,
                       const double *C, const double *G, double dt_stage, zone_ctx *zc) {
  int nv = g->m.nvar;
  zc->m = &g->m;
  zc->gc = &g->geomC[id2d];
  zc->tau = g->tauC[id2d];
  zc->idt = 1.0 / dt_stage;
  zc->emhd = (nv == 10);
  for (int v = 0; v < nv; v++) zc->C[v] = C[(int64_t)v * g->zg + z];
  double Pn_z[OG_NMAX], Un[OG_NMAX];
  load_prims(g, Pn, z, Pn_z);
  og_state sn;
  get_state(Pn_z, zc->gc, &sn);
  flux_vector(&g->m, zc->gc, zc->tau, 0, Pn_z, &sn, Un);
  double s2 = 0.0;
  for (int v = 0; v < nv; v++) s2 += Un[v] * Un[v];
  zc->scale = sqrt(s2) * zc->idt;
  if (zc->emhd) {
    double PE_z[OG_NMAX];
    load_prims(g, PE, z, PE_z);
    zc->Thn = temperature(&g->m, Pn_z);
    for (int i = 0; i < 4; i++) zc->ucovn[i] = sn.ucov[i];
    zc->utn = sn.ucon[0];
    double fq, fd;
    og_rescale_factors(&g->m, zc->tau, Pn_z, &fq, &fd);
    zc->qtn = Pn_z[OG_Q] * fq;
    zc->dtn = Pn_z[OG_DP] * fd;
    og_state sE;
    emhd_coefficients(&g->m, zc->gc, zc->tau, PE_z, &zc->c, &sE);
    zc->Xq = G[0 * g->zg + z];
    zc->Xd = G[1 * g->zg + z];
    zc->divx = G[2 * g->zg + z];
  }
}

static void zone_residual(const zone_ctx *zc, const double *P, double *R) {
  const og_model *m = zc->m;
  int nv = m->nvar;
  og_state s;
  get_state(P, zc->gc, &s);
  double U[OG_NMAX];
  flux_vector(m, zc->gc, zc->tau, 0, P, &s, U);
  for (int v = 0; v < nv; v++) R[v] = U[v] * zc->idt + zc->C[v];
  if (zc->emhd) {
    /* time derivatives of derived quantities between the unknown state and P_n (C-3) */
    double dtTheta = (temperature(m, P) - zc->Thn) * zc->idt;
    double dtucov[4];
    for (int i = 0; i < 4; i++) dtucov[i] = (s.ucov[i] - zc->ucovn[i]) * zc->idt;
    double dtut = (s.ucon[0] - zc->utn) * zc->idt;
    double Tq, Td, q0, dP0;
    emhd_time_part(zc->c.bh, zc->c.ThE, zc->c.utE, dtTheta, dtucov, &Tq, &Td);
    double divu = dtut + zc->divx;                 /* nabla_mu u^mu, static metric */
    emhd_combine(&zc->c, Tq, Td, zc->Xq, zc->Xd, divu, &q0, &dP0);
    double fq, fd;
    og_rescale_factors(m, zc->tau, P, &fq, &fd);
    double qt = P[OG_Q] * fq, dt_ = P[OG_DP] * fd;
    double itau = 1.0 / zc->tau;
    /* sqrt(-g)[ -(q~ - q~0)/tau_R + q~/2 div u ] with the implicit q~ averaged between P and P_n (eqs 15-16),
     * q~0 = f_q(P_E) q0, the coefficient q~ of div u at P_E */
    double Sq = -(0.5 * (qt + zc->qtn) - zc->c.fqE * q0) * itau + 0.5 * zc->c.qtE * divu;
    double Sd = -(0.5 * (dt_ + zc->dtn) - zc->c.fdE * dP0) * itau + 0.5 * zc->c.dtE * divu;
    R[OG_Q] = R[OG_Q] - zc->gc->sqrtmg * Sq;
    R[OG_DP] = R[OG_DP] - zc->gc->sqrtmg * Sd;
  }
}

void og_zone_residual(const og_grid *g, int64_t z, const double *Pn, const double *PE, const double *C,
                      const double *G, double dt_stage, const double *P, double *R) {
  int64_t id2d = z % g->n2d;
  zone_ctx zc;
  zone_setup(g, z, id2d, Pn, PE, C, G, dt_stage, &zc);
  double Pf[OG_NMAX];
  pad_prims(&g->m, P, Pf);
  zone_residual(&zc, Pf, R);
}

/* ===================================================================================
 * O-9  Newton iteration of one zone on an abstract residual (eqs 20-25)
 * =================================================================================== */

typedef void (*resid_fn)(const void *ctx, const double *P, double *R);

static double norm2sq(int n, const double *R) {
  double s = 0.0;
  for (int v = 0; v < n; v++) s += R[v] * R[v];
  return s;
}

/* Runs at most max_iters further iterations (<=0: until done).  P, *iters, *status carry the zone's state
 * between calls.  Returns ||R(P)||_2 of the final state. */
static double newton_zone(int n, const og_solver *sv, resid_fn fn, const void *ctx, double tol, double *P,
                          int32_t *iters, int32_t *status, int max_iters, int64_t *backtracks) {
  double R0[OG_NMAX], Rt[OG_NMAX], Pt[OG_NMAX], Pe[OG_NMAX], dP[OG_NMAX], J[OG_NMAX * OG_NMAX];
  for (int v = n; v < OG_NMAX; v++) { Pt[v] = 0.0; Pe[v] = 0.0; }
  int k = *iters, st = *status, done = 0;
  fn(ctx, P, R0);
  double f0 = norm2sq(n, R0);
  if (!isfinite(f0)) { *status = st | OG_ST_NONFINITE; return sqrt(f0); }
  while (!(sqrt(f0) < tol) && k < sv->kmax && (max_iters <= 0 || done < max_iters)) {
    /* finite-difference Jacobian, one perturbed evaluation per column (eqs 22-23; G-4, C-16, C-17) */
    int singular = 0;
    for (int j = 0; j < n; j++) {
      for (int v = 0; v < n; v++) Pe[v] = P[v];
      Pe[j] = (fabs(P[j]) < 5.0 * sv->fd_eps) ? sv->fd_eps : (1.0 + sv->fd_eps) * P[j];
      double h = Pe[j] - P[j];
      if (h == 0.0) singular = 1;
      double ih = 1.0 / h;
      fn(ctx, Pe, Rt);
      for (int i = 0; i < n; i++) J[i * n + j] = (Rt[i] - R0[i]) * ih;
    }
    for (int v = 0; v < n; v++) dP[v] = -R0[v];
    if (singular || og_lu_solve(n, J, dP, NULL) != 0) { st |= OG_ST_SINGULAR; break; }   /* eq 21; C-19 */
    /* quadratic backtracking line search (L220-233; G-2, C-14) */
    double lam = 1.0, ft = f0;
    int accepted = 0;
    for (int ls = 0; ls <= sv->lsmax; ls++) {
      for (int v = 0; v < n; v++) Pt[v] = P[v] + lam * dP[v];
      fn(ctx, Pt, Rt);
      ft = norm2sq(n, Rt);
      if (sqrt(ft) < sqrt(f0) * (1.0 - sv->eps_bt * lam)) { accepted = 1; break; }
      if (ls == sv->lsmax) break;
      if (backtracks) (*backtracks)++;
      lam = isfinite(ft) ? og_linesearch_lambda(f0, ft, lam) : 0.5 * lam;
    }
    if (!accepted) st |= OG_ST_LS_EXHAUSTED;
    for (int v = 0; v < n; v++) { P[v] = Pt[v]; R0[v] = Rt[v]; }
    f0 = ft;
    k++; done++;
    if (!isfinite(f0)) { st |= OG_ST_NONFINITE; break; }
  }
  if (!(st & (OG_ST_SINGULAR | OG_ST_NONFINITE))) {
    if (sqrt(f0) < tol) st |= OG_ST_CONVERGED;
    else if (k >= sv->kmax) st |= OG_ST_KMAX;
  }
  *iters = k; *status = st;
  return sqrt(f0);
}

static void resid_stage(const void *ctx, const double *P, double *R) { zone_residual((const zone_ctx *)ctx, P, R); }

/* NEXT-2  Reduced solve (L148, L643): the induction equation has no implicit source, so
 *   sqrt(-g) B^i_new = sqrt(-g) B^i_n - dt' [div F(P_E)]_{B^i}   <=>   B^i_new = -(C_{B^i} dt') / sqrt(-g)
 * is explicit (C = -U(P_n)/dt' + div F), and Newton runs on the M = nvar - 3 unknowns rho, u, u~^i (, q, dP) with the
 * rows of the same equations; unknown s is primitive s for s < 5, s + 3 beyond. */
typedef struct {
  const zone_ctx *zc;
  int nv;
  double B[3];
} reduced_ctx;
static int reduced_prim(int s) { return s < 5 ? s : s + 3; }
static void resid_reduced(const void *ctx, const double *X, double *R) {
  const reduced_ctx *rc = (const reduced_ctx *)ctx;
  double P[OG_NMAX] = {0}, Rf[OG_NMAX];
  int M = rc->nv - 3;
  for (int s = 0; s < M; s++) P[reduced_prim(s)] = X[s];
  for (int d = 0; d < 3; d++) P[OG_B1 + d] = rc->B[d];
  zone_residual(rc->zc, P, Rf);
  for (int s = 0; s < M; s++) R[s] = Rf[reduced_prim(s)];
}

int64_t og_newton(const og_grid *g, const double *Pn, const double *PE, const double *C, const double *G,
                  double dt_stage, double *P_iter, int max_iters_this_call, double *resnorm, int32_t *status,
                  int32_t *iters, int64_t *backtracks) {
  int nv = g->m.nvar;
  int64_t nactive = 0, nbt = 0;
#pragma omp parallel for collapse(2) schedule(dynamic, 4) reduction(+ : nactive, nbt)
  for (int k = g->ngd[2]; k < g->ngd[2] + g->n[2]; k++)
    for (int j = g->ngd[1]; j < g->ngd[1] + g->n[1]; j++)
      for (int i = g->ngd[0]; i < g->ngd[0] + g->n[0]; i++) {
        int64_t z = zidx(g, i, j, k);
        if (status[z] & OG_ST_TERMINAL) continue;
        zone_ctx zc;
        zone_setup(g, z, (int64_t)j * g->sz[0] + i, Pn, PE, C, G, dt_stage, &zc);
        double P[OG_NMAX];
        load_prims(g, P_iter, z, P);
        double tol = g->s.atol + g->s.rtol * zc.scale;
        int64_t bt = 0;
        double rn;
        if (g->d.reduced) {
          reduced_ctx rc;
          rc.zc = &zc;
          rc.nv = nv;
          double sg = g->geomC[(int64_t)j * g->sz[0] + i].sqrtmg;
          for (int d = 0; d < 3; d++) {
            rc.B[d] = -(C[(int64_t)(OG_B1 + d) * g->zg + z] * dt_stage) / sg;
            P[OG_B1 + d] = rc.B[d];
          }
          double X[OG_NMAX];
          for (int s = 0; s < nv - 3; s++) X[s] = P[reduced_prim(s)];
          rn = newton_zone(nv - 3, &g->s, resid_reduced, &rc, tol, X, &iters[z], &status[z], max_iters_this_call,
                           &bt);
          for (int s = 0; s < nv - 3; s++) P[reduced_prim(s)] = X[s];
        } else {
          rn = newton_zone(nv, &g->s, resid_stage, &zc, tol, P, &iters[z], &status[z], max_iters_this_call, &bt);
        }
        for (int v = 0; v < nv; v++) P_iter[(int64_t)v * g->zg + z] = P[v];
        resnorm[z] = rn;
        nbt += bt;
        if (!(status[z] & OG_ST_TERMINAL)) nactive++;
      }
  if (backtracks) *backtracks += nbt;
  return nactive;
}

/* ===================================================================================
 * O-11  Time step: two stages (L117-130; C-7 guesses; C-15 dt)
 * =================================================================================== */

double og_choose_dt(const og_grid *g, const double *P) {
  int64_t n = (int64_t)g->m.nvar * g->zg;
  double *Pc = (double *)malloc(sizeof(double) * (size_t)n);
  double *C = (double *)malloc(sizeof(double) * (size_t)n);
  double *G = (double *)calloc((size_t)(3 * g->zg), sizeof(double));
  memcpy(Pc, P, sizeof(double) * (size_t)n);
  og_fill_ghosts(g, Pc);
  double sp[4];
  og_stage_prepare(g, Pc, Pc, 1.0, C, G, sp);
  free(Pc); free(C); free(G);
  return g->d.cfl / sp[3];
}

static void collect_stats(const og_grid *g, int stage, const double *Pn, const double *resnorm,
                          const int32_t *status, const int32_t *iters, double dt_stage, og_step_stats *st) {
  for (int k = g->ngd[2]; k < g->ngd[2] + g->n[2]; k++)
    for (int j = g->ngd[1]; j < g->ngd[1] + g->n[1]; j++)
      for (int i = g->ngd[0]; i < g->ngd[0] + g->n[0]; i++) {
        int64_t z = zidx(g, i, j, k);
        int it = iters[z] > 15 ? 15 : iters[z];
        st->iters_hist[stage][it]++;
        if (!(status[z] & OG_ST_CONVERGED)) st->unconverged[stage]++;
        int64_t id = (int64_t)j * g->sz[0] + i;
        double Pz[OG_NMAX], Un[OG_NMAX];
        load_prims(g, Pn, z, Pz);
        og_state s; get_state(Pz, &g->geomC[id], &s);
        flux_vector(&g->m, &g->geomC[id], g->tauC[id], 0, Pz, &s, Un);
        double sc = sqrt(norm2sq(g->m.nvar, Un)) / dt_stage;
        double rel = resnorm[z] / sc;
        if (rel > st->max_resnorm[stage]) st->max_resnorm[stage] = rel;
      }
}

void og_timestep(const og_grid *g, double *P, double dt, og_step_stats *stats) {
  int nv = g->m.nvar;
  int64_t n = (int64_t)nv * g->zg;
  double *Ph = (double *)malloc(sizeof(double) * (size_t)n);
  double *Pnew = (double *)malloc(sizeof(double) * (size_t)n);
  double *C = (double *)calloc((size_t)n, sizeof(double));
  double *G = (double *)calloc((size_t)(3 * g->zg), sizeof(double));
  double *rn = (double *)calloc((size_t)g->zg, sizeof(double));
  int32_t *st = (int32_t *)calloc((size_t)g->zg, sizeof(int32_t));
  int32_t *it = (int32_t *)calloc((size_t)g->zg, sizeof(int32_t));
  if (stats) { memset(stats, 0, sizeof(*stats)); stats->zones = (int64_t)g->n[0] * g->n[1] * g->n[2]; }
  int64_t bt = 0;
  /* stage 1: P_E = P_n, dt' = dt/2, guess P_n */
  og_fill_ghosts(g, P);
  og_stage_prepare(g, P, P, 0.5 * dt, C, G, NULL);
  memcpy(Ph, P, sizeof(double) * (size_t)n);
  og_newton(g, P, P, C, G, 0.5 * dt, Ph, 0, rn, st, it, &bt);
  if (stats) { collect_stats(g, 0, P, rn, st, it, 0.5 * dt, stats); stats->backtracks[0] = bt; }
  /* stage 2: P_E = P_{n+1/2}, dt' = dt, guess P_{n+1/2} */
  og_fill_ghosts(g, Ph);
  og_stage_prepare(g, P, Ph, dt, C, G, NULL);
  memcpy(Pnew, Ph, sizeof(double) * (size_t)n);
  memset(st, 0, sizeof(int32_t) * (size_t)g->zg);
  memset(it, 0, sizeof(int32_t) * (size_t)g->zg);
  bt = 0;
  og_newton(g, P, Ph, C, G, dt, Pnew, 0, rn, st, it, &bt);
  if (stats) { collect_stats(g, 1, P, rn, st, it, dt, stats); stats->backtracks[1] = bt; }
  memcpy(P, Pnew, sizeof(double) * (size_t)n);
  free(Ph); free(Pnew); free(C); free(G); free(rn); free(st); free(it);
}

/* ===================================================================================
 * O-10  Standalone inversion: R(P) = (U(P) - U*) / ||U*||_2, tol = rtol
 * =================================================================================== */

typedef struct {
  const og_model *m;
  const og_geom *g;
  double tau;
  double Ustar[OG_NMAX];
  double iscale;
} inv_ctx;

static void resid_invert(const void *ctx, const double *P, double *R) {
  const inv_ctx *c = (const inv_ctx *)ctx;
  og_state s;
  get_state(P, c->g, &s);
  double U[OG_NMAX];
  flux_vector(c->m, c->g, c->tau, 0, P, &s, U);
  for (int v = 0; v < c->m->nvar; v++) R[v] = (U[v] - c->Ustar[v]) * c->iscale;
}

void og_invert(const og_model *m, const og_solver *s, double tau, int64_t nz, const double *Ustar,
               const og_geom *geom_or_null, double *P, int32_t *iters, int32_t *status, double *resnorm,
               int64_t *backtracks) {
  og_geom mink;
  og_geom_minkowski(&mink);
  int nv = m->nvar;
  int64_t nbt = 0;
#pragma omp parallel for schedule(dynamic, 256) reduction(+ : nbt)
  for (int64_t z = 0; z < nz; z++) {
    inv_ctx c;
    c.m = m; c.g = geom_or_null ? &geom_or_null[z] : &mink; c.tau = tau;
    double s2 = 0.0;
    for (int v = 0; v < nv; v++) { c.Ustar[v] = Ustar[(int64_t)v * nz + z]; s2 += c.Ustar[v] * c.Ustar[v]; }
    c.iscale = 1.0 / sqrt(s2);
    double Pz[OG_NMAX] = {0};
    for (int v = 0; v < nv; v++) Pz[v] = P[(int64_t)v * nz + z];
    int64_t bt = 0;
    iters[z] = 0; status[z] = 0;
    double rn = newton_zone(nv, s, resid_invert, &c, s->rtol, Pz, &iters[z], &status[z], 0, &bt);
    for (int v = 0; v < nv; v++) P[(int64_t)v * nz + z] = Pz[v];
    resnorm[z] = rn;
    nbt += bt;
  }
  if (backtracks) *backtracks = nbt;
}
