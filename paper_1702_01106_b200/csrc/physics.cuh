// physics.cuh -- zone-local GRMHD / EMHD algebra of grim (arXiv 1702.01106) as device functions.
//
// State from primitives (L41, L248, L297; reading C-9), stress tensor (eq 27, eqs 33-34),
// conserved variables and fluxes (eqs 30-32 L256-262 with G-3's sign, eqs 39-42), wave-speed bound
// (eqs 43-48).  The state is split into the pieces that depend on different primitives
// (velocity / magnetic field / thermodynamics) so that the finite-difference Jacobian (eqs 22-23) can reuse
// the pieces a perturbed column leaves unchanged -- recomputing them would reproduce the same bits.
//
// Arithmetic contract: compiled with -fmad=false; each expression below is written
// in its evaluation order, left to right, and that order is part of the library's definition.  The flat-space
// specialisation drops only operations that are exact no-ops (x*1, x+0, 0*x+y).
#pragma once

#include <cuda_runtime.h>
#include <math.h>

#include "fp64ops.cuh"

namespace grim {

enum { RHO = 0, UU = 1, U1 = 2, U2 = 3, U3 = 4, B1 = 5, B2 = 6, B3 = 7, QQ = 8, DPP = 9 };

struct ModelParams {
  double gam, gm1;   // adiabatic index, gam - 1 (L248)
  double phi, psi;   // closure coefficients (L299)
  int closure;       // 0: chi = phi cs^2 tau, nu = psi cs^2 tau (L299); 1: chi = phi, nu = psi constants (L566)
};

// thermal diffusivity and kinematic viscosity of a state with sound speed cs2 (L299; constant variant L566)
__device__ __forceinline__ void closure_coeffs(const ModelParams &m, double cs2, double tau, double &chi, double &nu) {
  const double c = m.phi * cs2 * tau, n = m.psi * cs2 * tau;
  chi = m.closure ? m.phi : c;
  nu = m.closure ? m.psi : n;
}

// ---------------------------------------------------------------------------------------------------------
// Geometry of one evaluation point.  Minkowski is a compile-time constant; a general stationary metric is a
// small record loaded from the context's 2-D tables (grim_set_metric).
// ---------------------------------------------------------------------------------------------------------
__host__ __device__ constexpr int sym4(int m, int n) {
  // index into the 10 stored components 00 01 02 03 11 12 13 22 23 33
  return (m <= n) ? (m * 4 - (m * (m - 1)) / 2 + (n - m)) : (n * 4 - (n * (n - 1)) / 2 + (m - n));
}

struct GeomFlat {
  static constexpr bool flat = true;
  __device__ __forceinline__ double sqrtmg() const { return 1.0; }
};

struct GeomGen {
  static constexpr bool flat = false;
  double g[10];      // g_mu_nu
  double bfac[3];    // alpha * g^{t i}  (= beta^i/alpha), i = 1..3
  double alpha;      // lapse
  double sg;         // sqrt(-g)
  double gcon00, gcon0d, gcondd;  // g^tt, g^td, g^dd of the face direction d (wave speeds; faces only)
  __device__ __forceinline__ double sqrtmg() const { return sg; }
  __device__ __forceinline__ double cov(int m, int n) const { return g[sym4(m, n)]; }
};

// u^mu, u_mu
struct Vel {
  double ucon[4], ucov[4];
};
// b^mu, b_mu, b^2
struct Mag {
  double bcon[4], bcov[4], bsq;
};
// bhat^mu, bhat_mu (eqs 33-34)
struct BHat {
  double con[4], cov[4];
};
// P_g, Theta and the rescaling factors of eqs 41-42
struct Thermo {
  double Pg, Th, fq, fdp;
};

template <class G>
__device__ __forceinline__ void lower(const G &g, const double (&vcon)[4], double (&vcov)[4]) {
  if constexpr (G::flat) {
    vcov[0] = -vcon[0];
    vcov[1] = vcon[1];
    vcov[2] = vcon[2];
    vcov[3] = vcon[3];
  } else {
#pragma unroll
    for (int m = 0; m < 4; m++) {
      double v = g.cov(m, 0) * vcon[0];
      v = v + g.cov(m, 1) * vcon[1];
      v = v + g.cov(m, 2) * vcon[2];
      v = v + g.cov(m, 3) * vcon[3];
      vcov[m] = v;
    }
  }
}

// W = sqrt(1 + g_ij u~^i u~^j); u^t = W/alpha; u^i = u~^i - W beta^i/alpha (C-9)
template <class A, class G>
__device__ __forceinline__ void vel_state(A &ar, const G &g, double ut1, double ut2, double ut3, Vel &v) {
  if constexpr (G::flat) {
    double usq = ut1 * ut1;
    usq = usq + ut2 * ut2;
    usq = usq + ut3 * ut3;
    double W = ar.sqrt(1.0 + usq);
    v.ucon[0] = W;
    v.ucon[1] = ut1;
    v.ucon[2] = ut2;
    v.ucon[3] = ut3;
  } else {
    const double ut[3] = {ut1, ut2, ut3};
    double usq = 0.0;
#pragma unroll
    for (int i = 1; i < 4; i++)
#pragma unroll
      for (int j = 1; j < 4; j++) usq = usq + g.cov(i, j) * ut[i - 1] * ut[j - 1];
    double W = ar.sqrt(1.0 + usq);
    v.ucon[0] = ar.div(W, g.alpha);
#pragma unroll
    for (int i = 1; i < 4; i++) v.ucon[i] = ut[i - 1] - W * g.bfac[i - 1];
  }
  lower(g, v.ucon, v.ucov);
}

// b^t = B^i u_i ; b^i = (B^i + b^t u^i)/u^t (L248)
template <class A, class G>
__device__ __forceinline__ void mag_state(A &ar, const G &g, const Vel &v, double Bx, double By, double Bz, Mag &b) {
  double bt = Bx * v.ucov[1];
  bt = bt + By * v.ucov[2];
  bt = bt + Bz * v.ucov[3];
  b.bcon[0] = bt;
  double iut = ar.rcp(v.ucon[0]);
  b.bcon[1] = (Bx + bt * v.ucon[1]) * iut;
  b.bcon[2] = (By + bt * v.ucon[2]) * iut;
  b.bcon[3] = (Bz + bt * v.ucon[3]) * iut;
  lower(g, b.bcon, b.bcov);
  double bsq = b.bcon[0] * b.bcov[0];
  bsq = bsq + b.bcon[1] * b.bcov[1];
  bsq = bsq + b.bcon[2] * b.bcov[2];
  bsq = bsq + b.bcon[3] * b.bcov[3];
  b.bsq = bsq;
}

template <class A>
__device__ __forceinline__ void bhat_state(A &ar, const Mag &b, BHat &h) {
  double ibn = ar.rcp(ar.sqrt(b.bsq));
#pragma unroll
  for (int i = 0; i < 4; i++) {
    h.con[i] = b.bcon[i] * ibn;
    h.cov[i] = b.bcov[i] * ibn;
  }
}

// c_s^2 = gam P_g/(rho + gam u) (eq 45; L501)
template <class A>
__device__ __forceinline__ double sound_speed2(A &ar, const ModelParams &m, double rho, double u) {
  double Pg = m.gm1 * u;
  return ar.div(m.gam * Pg, rho + m.gam * u);
}

// eqs 41-42 (L291-293): q~ = q sqrt(tau/(chi rho Theta^2)), dP~ = dP sqrt(tau/(nu rho Theta)), closure of the
// same state (C-4): chi = phi cs^2 tau, nu = psi cs^2 tau (L299)
template <int N, class A>
__device__ __forceinline__ void thermo_state(A &ar, const ModelParams &m, double tau, double rho, double u, Thermo &t) {
  t.Pg = m.gm1 * u;
  if constexpr (N == 10) {
    t.Th = ar.div(t.Pg, rho);
    double cs2 = ar.div(m.gam * t.Pg, rho + m.gam * u);
    double chi, nu;
    closure_coeffs(m, cs2, tau, chi, nu);
    t.fq = ar.sqrt(ar.div(tau, chi * rho * t.Th * t.Th));
    t.fdp = ar.sqrt(ar.div(tau, nu * rho * t.Th));
  } else {
    t.Th = 0.0;
    t.fq = 0.0;
    t.fdp = 0.0;
  }
}

// Row mu of T^mu_nu (eq 27 lowered; eqs 33-34; G-7)
template <int N>
__device__ __forceinline__ void stress_row(int mu, double rho, double u, double q, double dP, const Thermo &th,
                                           const Vel &v, const Mag &b, const BHat &h, double (&T)[4]) {
  double w = rho + u + th.Pg + b.bsq;
  double ptot = th.Pg + 0.5 * b.bsq;
  double wu = w * v.ucon[mu];
#pragma unroll
  for (int nu = 0; nu < 4; nu++) {
    double t = wu * v.ucov[nu];
    if (mu == nu) t = t + ptot;
    t = t - b.bcon[mu] * b.bcov[nu];
    if constexpr (N == 10) {
      t = t + q * (h.con[mu] * v.ucov[nu] + v.ucon[mu] * h.cov[nu]);
      double uu = v.ucon[mu] * v.ucov[nu];
      if (mu == nu) uu = 1.0 + uu;
      t = t - dP * (h.con[mu] * h.cov[nu] - (1.0 / 3.0) * uu);
    }
    T[nu] = t;
  }
}

// mu = 0: U(P); mu = 1..3: F^mu(P), all times sqrt(-g) (eqs 30-32, 39-40)
template <int N, class G>
__device__ __forceinline__ void flux_vector(const G &g, int mu, const double (&P)[N], const Thermo &th,
                                            const Vel &v, const Mag &b, const BHat &h, double (&out)[N]) {
  double T[4];
  double q = 0.0, dP = 0.0;
  if constexpr (N == 10) {
    q = P[QQ];
    dP = P[DPP];
  }
  stress_row<N>(mu, P[RHO], P[UU], q, dP, th, v, b, h, T);
  if constexpr (G::flat) {
    out[0] = P[RHO] * v.ucon[mu];
#pragma unroll
    for (int nu = 0; nu < 4; nu++) out[1 + nu] = T[nu];
#pragma unroll
    for (int i = 1; i < 4; i++)
      out[4 + i] = (mu == 0) ? P[B1 + i - 1] : (b.bcon[i] * v.ucon[mu] - b.bcon[mu] * v.ucon[i]);
    if constexpr (N == 10) {
      out[8] = (P[QQ] * th.fq) * v.ucon[mu];
      out[9] = (P[DPP] * th.fdp) * v.ucon[mu];
    }
  } else {
    const double sg = g.sqrtmg();
    out[0] = sg * (P[RHO] * v.ucon[mu]);
#pragma unroll
    for (int nu = 0; nu < 4; nu++) out[1 + nu] = sg * T[nu];
#pragma unroll
    for (int i = 1; i < 4; i++)
      out[4 + i] = (mu == 0) ? sg * P[B1 + i - 1] : sg * (b.bcon[i] * v.ucon[mu] - b.bcon[mu] * v.ucon[i]);
    if constexpr (N == 10) {
      out[8] = sg * ((P[QQ] * th.fq) * v.ucon[mu]);
      out[9] = sg * ((P[DPP] * th.fdp) * v.ucon[mu]);
    }
  }
}

// Full state of P in one call
template <int N, class A, class G>
__device__ __forceinline__ void full_state(A &ar, const ModelParams &m, const G &g, double tau, const double (&P)[N],
                                           Thermo &th, Vel &v, Mag &b, BHat &h) {
  vel_state(ar, g, P[U1], P[U2], P[U3], v);
  mag_state(ar, g, v, P[B1], P[B2], P[B3], b);
  if constexpr (N == 10) bhat_state(ar, b, h);
  thermo_state<N>(ar, m, tau, P[RHO], P[UU], th);
}

// v_max^2 (eqs 43-48; eq 46 rather than the simplified eq 49)
template <int N, class A>
__device__ __forceinline__ double vmax2(A &ar, const ModelParams &m, double tau, double rho, double u, double bsq) {
  double cs2 = sound_speed2(ar, m, rho, u);
  double va2 = ar.div_z(bsq, rho + m.gam * u + bsq);
  double cst2 = cs2;
  if constexpr (N == 10) {
    double chi, nu;
    closure_coeffs(m, cs2, tau, chi, nu);
    double vq2 = ar.div(m.gm1 * chi, tau);
    double vdp2 = ar.div(4.0 * nu, 3.0 * tau);
    cst2 = 0.5 * (cs2 + vq2 + ar.sqrt(cs2 * cs2 + vq2 * vq2)) + vdp2;
  }
  return cst2 + va2 - cst2 * va2;
}

// Grid-frame bound along direction d (1..3) of waves moving at +-v_max in the fluid frame (L303; O-4):
// (k.u)^2 = vmax^2 (g^{mn} + u^m u^n) k_m k_n, k = (-v, delta^d)
template <class A, class G>
__device__ __forceinline__ void wave_speeds_dir(A &ar, const G &g, double vm2, double ut, double ud, double &vp,
                                                double &vn) {
  double g00, g0d, gdd;
  if constexpr (G::flat) {
    g00 = -1.0;
    g0d = 0.0;
    gdd = 1.0;
  } else {
    g00 = g.gcon00;
    g0d = g.gcon0d;
    gdd = g.gcondd;
  }
  double qa = ut * ut - (g00 + ut * ut) * vm2;
  double qb = 2.0 * (ud * ut - (g0d + ud * ut) * vm2);
  double qc = ud * ud - (gdd + ud * ud) * vm2;
  double disc = ar.sqrt_z(fmax(qb * qb - 4.0 * qa * qc, 0.0));
  double i2A = ar.rcp(2.0 * qa);
  vp = (qb + disc) * i2A;
  vn = (qb - disc) * i2A;
}
template <class A, class G>
__device__ __forceinline__ double cmax_dir(A &ar, const G &g, double vm2, double ut, double ud) {
  double vp, vn;
  wave_speeds_dir(ar, g, vm2, ut, ud, vp, vn);
  return fmax(fabs(vp), fabs(vn));
}

}  // namespace grim
