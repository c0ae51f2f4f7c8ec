// problems.cuh -- the two residual functions the Newton iteration is applied to.
//   StageProblem : residual of one stage of the semi-implicit time step (eq 19 L185-188 half step, eq 13
//                  L127-130 full step; eqs 15-16; EMHD rows eqs 39-40; readings C-3, C-4)
//   InvertProblem: standalone primitive recovery R(P) = (U(P) - U*)/||U*||_2 (O-10; BASELINE config 2)
#pragma once

#include "newton.cuh"

namespace grim {

// The P_n- / P_E-derived constants of the EMHD rows (O-8), frozen during the iteration.
enum {
  K_THN, K_UCOVN0, K_UCOVN1, K_UCOVN2, K_UCOVN3, K_UTN, K_QTN, K_DTN,           // P_n
  K_BH0, K_BH1, K_BH2, K_BH3, K_THE, K_UTE, K_NRHOCHI, K_RHONU3, K_FQE, K_FDE,  // P_E
  K_HQTE, K_HDTE, K_XQ, K_XD, K_DIVX, K_ITAU,
  K_COUNT
};

// Where the constants live.  KSM = false: in registers.  KSM = true: in the thread's shared-memory words that the
// structured solve leaves unused -- the off-diagonal entries of the Jacobian's B rows (newton.cuh: 27 words, never
// written or read) -- which frees 2 K_COUNT registers for the finite-difference columns; constant i sits at
// Ks[kslot(i) * CS].
template <int N>
__host__ __device__ constexpr int kslot(int i) {
  const int r = B1 + i / (N - 1), c = i % (N - 1);
  return r * N + (c < r ? c : c + 1);
}

// CS: stride (in doubles) of the per-thread shared-memory vector that holds the stage constant C
template <int N, class G, int CS, bool KSM = false>
struct StageProblem {
  ModelParams m;
  G g;
  double tau_, idt;
  const double *Cs;  // C[v] at Cs[v * CS] (shared memory: read once per residual evaluation, 2N registers saved)
  double *Ks;        // KSM: the thread's Jacobian base (shared memory)
  double scale;      // ||U(P_n)||_2 / dt' (C-2)
  double kreg[KSM ? 1 : K_COUNT];

  __device__ __forceinline__ const ModelParams &model() const { return m; }
  __device__ __forceinline__ const G &geom() const { return g; }
  __device__ __forceinline__ double tau() const { return tau_; }
  __device__ __forceinline__ double K(int i) const {
    if constexpr (KSM) return Ks[kslot<N>(i) * CS];
    else return kreg[i];
  }
  __device__ __forceinline__ void setK(int i, double v) {
    if constexpr (KSM) Ks[kslot<N>(i) * CS] = v;
    else kreg[i] = v;
  }

  // Everything that depends only on P_n and P_E (L438)
  template <class A>
  // pc0: the state pieces of the initial iterate, already computed by the caller.  In grim_timestep the guess is
  // P_E, and in its first stage P_n is P_E too: the states of P_E / P_n are then pc0 itself (same inputs, same code,
  // same bits) and are not computed again.
  __device__ __forceinline__ void setup(A &ar, const double (&Pn)[N], const double (&PE)[N], double dt_stage,
                                        const Pieces &pc0, bool pe_is_guess, bool pn_is_guess, double Xq, double Xd,
                                        double divx) {
    idt = ar.rcp(dt_stage);
    Pieces pn;
    if (pn_is_guess) pn = pc0;
    else full_state<N>(ar, m, g, tau_, Pn, pn.th, pn.v, pn.b, pn.h);
    double Un[N];
    flux_vector<N>(g, 0, Pn, pn.th, pn.v, pn.b, pn.h, Un);
    scale = ar.sqrt_z(norm2sq<N>(Un)) * idt;
    if constexpr (N == 10) {
      setK(K_ITAU, ar.rcp(tau_));
      setK(K_XQ, Xq);
      setK(K_XD, Xd);
      setK(K_DIVX, divx);
      setK(K_THN, pn.th.Th);
#pragma unroll
      for (int i = 0; i < 4; i++) setK(K_UCOVN0 + i, pn.v.ucov[i]);
      setK(K_UTN, pn.v.ucon[0]);
      setK(K_QTN, Pn[QQ] * pn.th.fq);
      setK(K_DTN, Pn[DPP] * pn.th.fdp);
      Pieces pe;
      if (pe_is_guess) pe = pc0;
      else full_state<N>(ar, m, g, tau_, PE, pe.th, pe.v, pe.b, pe.h);
#pragma unroll
      for (int i = 0; i < 4; i++) setK(K_BH0 + i, pe.h.con[i]);
      setK(K_THE, pe.th.Th);
      setK(K_UTE, pe.v.ucon[0]);
      double cs2 = sound_speed2(ar, m, PE[RHO], PE[UU]);
      double chi, nu;
      closure_coeffs(m, cs2, tau_, chi, nu);
      setK(K_NRHOCHI, -(PE[RHO] * chi));
      setK(K_RHONU3, 3.0 * PE[RHO] * nu);
      const double fqE = pe.th.fq, fdE = pe.th.fdp;
      setK(K_FQE, fqE);
      setK(K_FDE, fdE);
      setK(K_HQTE, 0.5 * (PE[QQ] * fqE));
      setK(K_HDTE, 0.5 * (PE[DPP] * fdE));
    }
  }

  __device__ __forceinline__ void assemble(const double (&P)[N], const Pieces &pc, double (&R)[N]) const {
    double U[N];
    flux_vector<N>(g, 0, P, pc.th, pc.v, pc.b, pc.h, U);
#pragma unroll
    for (int v = 0; v < N; v++) R[v] = U[v] * idt + Cs[v * CS];
    if constexpr (N == 10) {
      // time derivatives of derived quantities between the unknown state and P_n (C-3)
      double dtTheta = (pc.th.Th - K(K_THN)) * idt;
      double dtucov[4];
#pragma unroll
      for (int i = 0; i < 4; i++) dtucov[i] = (pc.v.ucov[i] - K(K_UCOVN0 + i)) * idt;
      double dtut = (pc.v.ucon[0] - K(K_UTN)) * idt;
      double bdu = K(K_BH0) * dtucov[0];
      bdu = bdu + K(K_BH1) * dtucov[1];
      bdu = bdu + K(K_BH2) * dtucov[2];
      bdu = bdu + K(K_BH3) * dtucov[3];
      double Tq = K(K_BH0) * dtTheta + K(K_THE) * (K(K_UTE) * bdu);
      double Td = K(K_BH0) * bdu;
      double divu = dtut + K(K_DIVX);
      double q0 = K(K_NRHOCHI) * (Tq + K(K_XQ));                              // eq 37
      double dP0 = K(K_RHONU3) * ((Td + K(K_XD)) - (1.0 / 3.0) * divu);        // eq 38 (G-5)
      double qt = P[QQ] * pc.th.fq, dpt = P[DPP] * pc.th.fdp;
      double Sq = -(0.5 * (qt + K(K_QTN)) - K(K_FQE) * q0) * K(K_ITAU) + K(K_HQTE) * divu;    // eq 39, eqs 15-16
      double Sd = -(0.5 * (dpt + K(K_DTN)) - K(K_FDE) * dP0) * K(K_ITAU) + K(K_HDTE) * divu;  // eq 40
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
