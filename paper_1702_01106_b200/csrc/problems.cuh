// problems.cuh -- the two residual functions the Newton iteration is applied to.
//   StageProblem : residual of one stage of the semi-implicit time step (eq 19 L185-188 half step, eq 13
//                  L127-130 full step; eqs 15-16; EMHD rows eqs 39-40; readings C-3, C-4)
//   InvertProblem: standalone primitive recovery R(P) = (U(P) - U*)/||U*||_2 (O-10; BASELINE config 2)
#pragma once

#include "newton.cuh"

namespace grim {

// CS: stride (in doubles) of the per-thread shared-memory vector that holds the stage constant C
template <int N, class G, int CS>
struct StageProblem {
  ModelParams m;
  G g;
  double tau_, idt, itau;
  const double *Cs;  // C[v] at Cs[v * CS] (shared memory: read once per residual evaluation, 2N registers saved)
  double scale;      // ||U(P_n)||_2 / dt' (C-2)
  // EMHD only.  P_n-derived:
  double Thn, ucovn[4], utn, qtn, dtn;
  // P_E-derived coefficients, frozen during the iteration (O-8), and the spatial-gradient terms of the stage:
  double bh[4], ThE, utE, nrhochi, rhonu3, fqE, fdE, hqtE, hdtE;
  double Xq, Xd, divx;

  __device__ __forceinline__ const ModelParams &model() const { return m; }
  __device__ __forceinline__ const G &geom() const { return g; }
  __device__ __forceinline__ double tau() const { return tau_; }

  // Everything that depends only on P_n and P_E (L438)
  template <class A>
  // pc0: the state pieces of the initial iterate, already computed by the caller.  In grim_timestep the guess is
  // P_E, and in its first stage P_n is P_E too: the states of P_E / P_n are then pc0 itself (same inputs, same code,
  // same bits) and are not computed again.
  __device__ __forceinline__ void setup(A &ar, const double (&Pn)[N], const double (&PE)[N], double dt_stage,
                                        const Pieces &pc0, bool pe_is_guess, bool pn_is_guess) {
    idt = ar.rcp(dt_stage);
    itau = ar.rcp(tau_);
    Pieces pn;
    if (pn_is_guess) pn = pc0;
    else full_state<N>(ar, m, g, tau_, Pn, pn.th, pn.v, pn.b, pn.h);
    double Un[N];
    flux_vector<N>(g, 0, Pn, pn.th, pn.v, pn.b, pn.h, Un);
    scale = ar.sqrt_z(norm2sq<N>(Un)) * idt;
    if constexpr (N == 10) {
      Thn = pn.th.Th;
#pragma unroll
      for (int i = 0; i < 4; i++) ucovn[i] = pn.v.ucov[i];
      utn = pn.v.ucon[0];
      qtn = Pn[QQ] * pn.th.fq;
      dtn = Pn[DPP] * pn.th.fdp;
      Pieces pe;
      if (pe_is_guess) pe = pc0;
      else full_state<N>(ar, m, g, tau_, PE, pe.th, pe.v, pe.b, pe.h);
#pragma unroll
      for (int i = 0; i < 4; i++) bh[i] = pe.h.con[i];
      ThE = pe.th.Th;
      utE = pe.v.ucon[0];
      double cs2 = sound_speed2(ar, m, PE[RHO], PE[UU]);
      double chi, nu;
      closure_coeffs(m, cs2, tau_, chi, nu);
      nrhochi = -(PE[RHO] * chi);
      rhonu3 = 3.0 * PE[RHO] * nu;
      fqE = pe.th.fq;
      fdE = pe.th.fdp;
      hqtE = 0.5 * (PE[QQ] * fqE);
      hdtE = 0.5 * (PE[DPP] * fdE);
    }
  }

  __device__ __forceinline__ void assemble(const double (&P)[N], const Pieces &pc, double (&R)[N]) const {
    double U[N];
    flux_vector<N>(g, 0, P, pc.th, pc.v, pc.b, pc.h, U);
#pragma unroll
    for (int v = 0; v < N; v++) R[v] = U[v] * idt + Cs[v * CS];
    if constexpr (N == 10) {
      // time derivatives of derived quantities between the unknown state and P_n (C-3)
      double dtTheta = (pc.th.Th - Thn) * idt;
      double dtucov[4];
#pragma unroll
      for (int i = 0; i < 4; i++) dtucov[i] = (pc.v.ucov[i] - ucovn[i]) * idt;
      double dtut = (pc.v.ucon[0] - utn) * idt;
      double bdu = bh[0] * dtucov[0];
      bdu = bdu + bh[1] * dtucov[1];
      bdu = bdu + bh[2] * dtucov[2];
      bdu = bdu + bh[3] * dtucov[3];
      double Tq = bh[0] * dtTheta + ThE * (utE * bdu);
      double Td = bh[0] * bdu;
      double divu = dtut + divx;
      double q0 = nrhochi * (Tq + Xq);                              // eq 37
      double dP0 = rhonu3 * ((Td + Xd) - (1.0 / 3.0) * divu);        // eq 38 (G-5)
      double qt = P[QQ] * pc.th.fq, dpt = P[DPP] * pc.th.fdp;
      double Sq = -(0.5 * (qt + qtn) - fqE * q0) * itau + hqtE * divu;    // eq 39, eqs 15-16
      double Sd = -(0.5 * (dpt + dtn) - fdE * dP0) * itau + hdtE * divu;  // eq 40
      if constexpr (G::flat) {
        R[QQ] = R[QQ] - Sq;
        R[DPP] = R[DPP] - Sd;
      } else {
        R[QQ] = R[QQ] - g.sqrtmg() * Sq;
        R[DPP] = R[DPP] - g.sqrtmg() * Sd;
      }
    }
  }
};

template <int N, class G, int CS>
struct InvertProblem {
  ModelParams m;
  G g;
  double tau_;
  const double *Us;  // U*[v] at Us[v * CS] (shared memory)
  double iscale;

  __device__ __forceinline__ const ModelParams &model() const { return m; }
  __device__ __forceinline__ const G &geom() const { return g; }
  __device__ __forceinline__ double tau() const { return tau_; }

  template <class A>
  __device__ __forceinline__ void setup(A &ar) {
    double Ustar[N];
#pragma unroll
    for (int v = 0; v < N; v++) Ustar[v] = Us[v * CS];
    double s2 = norm2sq<N>(Ustar);
    iscale = ar.rcp(ar.sqrt(s2));
  }
  __device__ __forceinline__ void assemble(const double (&P)[N], const Pieces &pc, double (&R)[N]) const {
    double U[N];
    flux_vector<N>(g, 0, P, pc.th, pc.v, pc.b, pc.h, U);
#pragma unroll
    for (int v = 0; v < N; v++) R[v] = (U[v] - Us[v * CS]) * iscale;
  }
};

}  // namespace grim
