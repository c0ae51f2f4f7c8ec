// newton.cuh -- the per-zone Newton-Raphson iteration of grim (eqs 20-25), one thread per
// zone, the whole iteration on chip:
//   * residual pieces cached in registers and reused by the finite-difference columns they do not depend on
//     (eqs 22-23; G-4, C-16, C-17),
//   * the N x N Jacobian in shared memory, one column of 8-byte words per thread (bank-conflict free for any
//     run-time row index), factorised by a left-looking LU with partial pivoting whose row exchanges are
//     exchanges of row *pointers* held in registers (eq 21; L434 "LAPACK" -> dgetf2/dgesv semantics: pivot =
//     first row of maximal |a_ik|, multipliers formed with the reciprocal of the pivot; C-19),
//   * quadratic backtracking line search (L218-235, eqs 24-25; G-2, C-14),
//   * over all N primitives (BASELINE) or, reduced solve, over the N - 3 that have implicit terms (L148, L643).
// The left-looking order applies to every matrix element the same updates in the same order (k ascending) as
// the textbook right-looking elimination, so the factors are identical; it reads each multiplier column from
// shared memory once per later column and writes each element once.
#pragma once

#include "physics.cuh"

namespace grim {

struct SolverParams {
  double fd_eps, eps_bt, atol, rtol;
  int kmax, lsmax;
};

enum {
  ST_CONVERGED = 1, ST_KMAX = 2, ST_LS_EXHAUSTED = 4, ST_SINGULAR = 8, ST_NONFINITE = 16,
  ST_TERMINAL = ST_CONVERGED | ST_KMAX | ST_SINGULAR | ST_NONFINITE
};

struct Pieces {
  Thermo th;
  Vel v;
  Mag b;
  BHat h;
};

template <int N>
__device__ __forceinline__ double norm2sq(const double (&R)[N]) {
  double s = R[0] * R[0];
#pragma unroll
  for (int v = 1; v < N; v++) s = s + R[v] * R[v];
  return s;
}

// The unknowns of the Newton iteration.  Full solve: all N primitives (BASELINE; C-1).  Reduced solve (RED; the
// paper's own split, L148 / L643): B^i is advanced explicitly by the caller and stays fixed, the M = N - 3 unknowns
// are rho, u, u~^i (, q, dP) and the residual rows are those of the same equations; unknown s is primitive prim(s).
template <int N, bool RED>
struct Unknowns {
  static constexpr int M = RED ? N - 3 : N;
  static __host__ __device__ constexpr int prim(int s) { return (!RED || s < B1) ? s : s + 3; }
};

template <int N, bool RED>
__device__ __forceinline__ double norm2sq_rows(const double (&R)[N]) {
  using U = Unknowns<N, RED>;
  double s = R[U::prim(0)] * R[U::prim(0)];
#pragma unroll
  for (int v = 1; v < U::M; v++) s = s + R[U::prim(v)] * R[U::prim(v)];
  return s;
}

// Residual at P with every piece recomputed; the pieces are returned for reuse.
template <int N, class A, class Prob>
__device__ __forceinline__ void eval_full(A &ar, const Prob &prob, const double (&P)[N], Pieces &pc, double (&R)[N]) {
  full_state<N>(ar, prob.model(), prob.geom(), prob.tau(), P, pc.th, pc.v, pc.b, pc.h);
  prob.assemble(P, pc, R);
}

// Residual at P with component J replaced by pj (eq 23): only the pieces that depend on component J are
// recomputed; the others are those of the unperturbed state.
template <int J, int N, class A, class Prob>
__device__ __forceinline__ void eval_column(A &ar, const Prob &prob, const double (&P)[N], double pj, const Pieces &base,
                                            double (&R)[N]) {
  double Pe[N];
#pragma unroll
  for (int v = 0; v < N; v++) Pe[v] = P[v];
  Pe[J] = pj;
  Pieces pc = base;
  if constexpr (J == RHO || J == UU) {
    thermo_state<N>(ar, prob.model(), prob.tau(), Pe[RHO], Pe[UU], pc.th);
  } else if constexpr (J >= U1 && J <= U3) {
    vel_state(ar, prob.geom(), Pe[U1], Pe[U2], Pe[U3], pc.v);
    mag_state(ar, prob.geom(), pc.v, Pe[B1], Pe[B2], Pe[B3], pc.b);
    if constexpr (N == 10) bhat_state(ar, pc.b, pc.h);
  } else if constexpr (J >= B1 && J <= B3) {
    mag_state(ar, prob.geom(), pc.v, Pe[B1], Pe[B2], Pe[B3], pc.b);
    if constexpr (N == 10) bhat_state(ar, pc.b, pc.h);
  }
  prob.assemble(Pe, pc, R);
}

// Shared-memory Jacobian of one thread: element (row r, column c) at sJ[(r*N + c)*BLOCK], sJ already offset by
// the thread index.
template <int N, int BLOCK>
struct JacView {
  double *base;
  __device__ __forceinline__ double &at(int rowoff, int c) const { return base[rowoff + c * BLOCK]; }
  static __device__ __forceinline__ constexpr int row(int r) { return r * N * BLOCK; }
};

// Structure of the Jacobian that holds for both residuals (problems.cuh) whatever the state: entry (row, col) is
// (R_row(P_eps,col) - R_row(P)) * ih with R_row(P_eps,col) the SAME bits as R_row(P) -- exactly +0 * ih -- when
// R_row does not read primitive col:
//   * row B^i reads B^i only (U_{B^i} = sqrt(-g) B^i, no source; eq 30, O-3),
//   * row rho reads rho and u~^i only (U_rho = sqrt(-g) rho u^t),
//   * rows q, dP read rho, u (rescale factors, Theta), u~^i and their own primitive; not B^i (the bhat of the source
//     terms is P_E's, O-8), not each other.
// Those 41 of the 100 entries are stored as that signed zero without evaluating the row (the perturbed evaluation
// then skips the row altogether), and the B rows, which the structured solve below never reads, are not stored.
template <int N>
__host__ __device__ constexpr bool jac_zero(int row, int col) {
  if (row >= B1 && row <= B3) return col != row;
  if (row == RHO) return col == UU || (col >= B1 && col <= B3) || col >= QQ;
  if (row >= QQ) return (col >= B1 && col <= B3) || (col >= QQ && col != row);
  return false;
}
// full solves of both problems use the structure; the reduced solve has no B rows and keeps the general path
template <int N, bool RED>
__host__ __device__ constexpr bool use_structure() { return !RED; }

__device__ __forceinline__ double zero_times(double ih) {  // (+0) * ih for finite ih
  return __hiloint2double(__double2hiint(ih) & 0x80000000, 0);
}

// One finite-difference column (eqs 22-23): J[:,j] = (R(P_eps,j) - R0) / (P_eps,j - P_j)
// (column S of the M x M Jacobian: unknown S = primitive prim(S))
template <int S, int N, bool RED, int BLOCK, class A, class Prob>
__device__ __forceinline__ void fd_column(A &ar, const Prob &prob, const SolverParams &sp, const double (&P)[N],
                                          const Pieces &base, const double (&R0)[N],
                                          const JacView<Unknowns<N, RED>::M, BLOCK> &jac, bool &singular) {
  using U = Unknowns<N, RED>;
  constexpr int J = U::prim(S);
  constexpr bool STRUCT = use_structure<N, RED>();
  double pj = (fabs(P[J]) < 5.0 * sp.fd_eps) ? sp.fd_eps : (1.0 + sp.fd_eps) * P[J];
  double h = pj - P[J];
  if (h == 0.0) singular = true;
  double ih = ar.rcp(h);
  double Rt[N];
  eval_column<J, N>(ar, prob, P, pj, base, Rt);
#pragma unroll
  for (int i = 0; i < U::M; i++) {
    const int row = U::prim(i);
    if (jac_zero<N>(row, J)) {
      if (!(STRUCT && row >= B1 && row <= B3)) jac.at(JacView<U::M, BLOCK>::row(i), S) = zero_times(ih);
    } else {
      jac.at(JacView<U::M, BLOCK>::row(i), S) = (Rt[row] - R0[row]) * ih;
    }
  }
}

// Order in which the (independent) columns are evaluated: first those that reuse every piece of the unperturbed
// state (q, dP), then the thermodynamic ones (reuse velocity, field, bhat), the field ones (velocity, thermo), last
// the velocity ones (thermo only) -- so the cached pieces die as early as possible and the later, more expensive
// columns have the registers.  The Jacobian does not depend on the order.
template <int N, bool RED>
__host__ __device__ constexpr int fd_order(int s) {
  if (RED) {  // unknown indices: rho u u~1 u~2 u~3 (q dP)
    constexpr int red10[7] = {5, 6, 0, 1, 2, 3, 4};
    return N == 10 ? red10[s] : s;
  }
  constexpr int ord10[10] = {QQ, DPP, RHO, UU, B1, B2, B3, U1, U2, U3};
  constexpr int ord8[8] = {RHO, UU, B1, B2, B3, U1, U2, U3};
  return N == 10 ? ord10[s] : ord8[s];
}

template <int S, int N, bool RED, int BLOCK, class A, class Prob, bool DONE = (S == Unknowns<N, RED>::M)>
struct FdColumns {
  static __device__ __forceinline__ void run(A &ar, const Prob &prob, const SolverParams &sp, const double (&P)[N],
                                             const Pieces &base, const double (&R0)[N],
                                             const JacView<Unknowns<N, RED>::M, BLOCK> &jac, bool &singular) {
    fd_column<fd_order<N, RED>(S), N, RED, BLOCK>(ar, prob, sp, P, base, R0, jac, singular);
    FdColumns<S + 1, N, RED, BLOCK, A, Prob>::run(ar, prob, sp, P, base, R0, jac, singular);
  }
};
template <int S, int N, bool RED, int BLOCK, class A, class Prob>
struct FdColumns<S, N, RED, BLOCK, A, Prob, true> {
  static __device__ __forceinline__ void run(A &, const Prob &, const SolverParams &, const double (&)[N], const Pieces &,
                                             const double (&)[N], const JacView<Unknowns<N, RED>::M, BLOCK> &,
                                             bool &) {}
};

// Solves J x = b (b in, x out) for the Jacobian held in shared memory.  Returns false if a pivot is zero or
// non-finite (C-19).  Registers hold one column at a time, in pivoted order: position i of the order is the
// matrix row at shared-memory offset rowoff[i].  A row exchange exchanges two entries of rowoff and nothing
// else -- the column in registers dies when it is stored, the right-hand side is permuted once, through the
// storage of the last column, when the order is final -- and the diagonal slot receives the reciprocal of the
// pivot, which is all the back substitution needs of it.
template <int N, int BLOCK, class A>
__device__ __forceinline__ bool lu_solve(A &ar, const JacView<N, BLOCK> &jac, double (&b)[N]) {
  int rowoff[N];
#pragma unroll
  for (int i = 0; i < N; i++) rowoff[i] = JacView<N, BLOCK>::row(i);
  bool ok = true;
#pragma unroll
  for (int j = 0; j < N; j++) {
    double x[N];
#pragma unroll
    for (int i = 0; i < N; i++) x[i] = jac.at(rowoff[i], j);
    if (j == N - 1) {
      // positions 0..N-2 are final and position N-1 is the row that is left: permute b through this column's
      // storage, which the loads above have just emptied
#pragma unroll
      for (int i = 0; i < N; i++) jac.at(JacView<N, BLOCK>::row(i), j) = b[i];
#pragma unroll
      for (int i = 0; i < N; i++) b[i] = jac.at(rowoff[i], j);
    }
    // updates of the earlier pivots, k ascending; the last column carries the right-hand side along
#pragma unroll
    for (int k = 0; k < j; k++) {
#pragma unroll
      for (int i = k + 1; i < N; i++) {
        double l = jac.at(rowoff[i], k);
        x[i] = x[i] - l * x[k];
        if (j == N - 1) b[i] = b[i] - l * b[k];
      }
    }
    // pivot: first position of maximal |x_i|, i >= j
    int p = j, rop = rowoff[j];
    double xp = x[j], amax = fabs(x[j]);
#pragma unroll
    for (int i = j + 1; i < N; i++) {
      double v = fabs(x[i]);
      if (v > amax) {
        amax = v;
        xp = x[i];
        p = i;
        rop = rowoff[i];
      }
    }
    if (!(amax > 0.0) || !isfinite(amax)) ok = false;
    double r = ar.rcp(xp);
    // U above the diagonal; multipliers x_i / pivot for every candidate row (the pivot row's own slot is then
    // overwritten by 1/pivot)
#pragma unroll
    for (int i = 0; i < j; i++) jac.at(rowoff[i], j) = x[i];
#pragma unroll
    for (int i = j; i < N; i++) jac.at(rowoff[i], j) = x[i] * r;
    jac.at(rop, j) = r;
    // exchange positions j and p
#pragma unroll
    for (int i = j + 1; i < N; i++)
      if (p == i) rowoff[i] = rowoff[j];
    rowoff[j] = rop;
  }
  // back substitution with U
#pragma unroll
  for (int i = N - 1; i >= 0; i--) {
    double s = b[i];
#pragma unroll
    for (int j = i + 1; j < N; j++) s = s - jac.at(rowoff[i], j) * b[j];
    b[i] = s * jac.at(rowoff[i], i);
  }
  return ok;
}

// ---------------------------------------------------------------------------------------------------------
// The same factorisation by register panels.  Shared memory moves 128 B per cycle and SM -- a warp's 8-byte
// load costs as much as four of its fp64 instructions -- and the column-at-a-time LU above loads every
// multiplier once per later column (285 loads for N = 10): the solve was bound by the shared-memory pipe
// (DESIGN.md 15.2).  Here a panel of columns is held in registers at a time: the multipliers
// of the earlier pivots are loaded once per panel, those of the panel's own pivots are never loaded, and the
// last panel carries the right-hand side along and is never stored -- the back substitution reads its U from
// the registers.  N = 10 with panels of 5 + 5 columns loads 35 multipliers; N <= 8 is one panel (no stores).
//
// Every matrix element still receives the updates of the pivots k = 0, 1, ... in ascending order, each as
// x - l * x_k with the multiplier l = x * (1/pivot): the same rounded operations as og_lu_solve / dgetf2, so
// the factors, the pivot sequence (first position of maximal |x_i|) and the solution are identical.  A row
// exchange swaps two entries of rowoff (for the columns in shared memory) and positions j and p of the panel
// columns still in registers (select chains; p is a run-time index).
// ---------------------------------------------------------------------------------------------------------
template <int M>
__device__ __forceinline__ void swap_positions(double (&x)[M], int j, int p) {
  // branch-free: selects on the run-time index p (a conditional assignment would send the column to local memory)
  const double xj = x[j];
  double xp = xj;
#pragma unroll
  for (int i = j + 1; i < M; i++) xp = (p == i) ? x[i] : xp;
#pragma unroll
  for (int i = j + 1; i < M; i++) x[i] = (p == i) ? xj : x[i];
  x[j] = xp;
}

// Factorises columns C0 .. C0+CB-1 held in X (pivoted order, updates of the pivots < C0 applied).  RHS: b is
// carried along as a passenger column.  STORE: the finished columns go to shared memory (L below the
// diagonal, U above, 1/pivot on it).
template <int M, int BLOCK, int C0, int CB, bool RHS, bool STORE, class A>
__device__ __forceinline__ void lu_panel(A &ar, const JacView<M, BLOCK> &jac, int (&rowoff)[M], double (&X)[CB][M],
                                         double (&b)[M], double (&rinv)[CB], bool &ok) {
#pragma unroll
  for (int jj = 0; jj < CB; jj++) {
    const int j = C0 + jj;
    // pivot: first position of maximal |x_i|, i >= j
    int p = j;
    double xp = X[jj][j], amax = fabs(X[jj][j]);
#pragma unroll
    for (int i = j + 1; i < M; i++) {
      const double v = fabs(X[jj][i]);
      const bool gt = v > amax;
      amax = gt ? v : amax;
      xp = gt ? X[jj][i] : xp;
      p = gt ? i : p;
    }
    ok = ok && (amax > 0.0) && isfinite(amax);
    const double r = ar.rcp(xp);
    rinv[jj] = r;
    // exchange positions j and p
    const int roj = rowoff[j];
    int rop = roj;
#pragma unroll
    for (int i = j + 1; i < M; i++) rop = (p == i) ? rowoff[i] : rop;
#pragma unroll
    for (int i = j + 1; i < M; i++) rowoff[i] = (p == i) ? roj : rowoff[i];
    rowoff[j] = rop;
#pragma unroll
    for (int c = jj; c < CB; c++) swap_positions<M>(X[c], j, p);
    if (RHS) swap_positions<M>(b, j, p);
    // multipliers, then the update of the later panel columns and of the right-hand side
#pragma unroll
    for (int i = j + 1; i < M; i++) X[jj][i] = X[jj][i] * r;
#pragma unroll
    for (int c = jj + 1; c < CB; c++)
#pragma unroll
      for (int i = j + 1; i < M; i++) X[c][i] = X[c][i] - X[jj][i] * X[c][j];
    if (RHS) {
#pragma unroll
      for (int i = j + 1; i < M; i++) b[i] = b[i] - X[jj][i] * b[j];
    }
    if (STORE) {
#pragma unroll
      for (int i = 0; i < M; i++) jac.at(rowoff[i], j) = (i == j) ? r : X[jj][i];
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// The factorisation of the full N x N Jacobian with its structure (jac_zero) used.  The B rows are zero in the
// columns of rho, u, u~^i, so in the elimination steps k = 0..4 they are never the pivot (a zero is never the
// first maximal |x_i| unless every candidate is zero, which is the singular exit either way), their
// multipliers are exact zeros and their updates x - 0 * x_k are no-ops: steps 0..4 run on the N - 3 other rows
// ("active": positions 0..4 and, for EMHD, 8, 9) and leave the B rows in positions 5..7 as they were stored.
//   A  columns 0..4, left-looking, one column of the active rows in registers (as lu_solve above);
//   B  columns 5..N-1 and the right-hand side: active rows updated by the pivots 0..4 (G columns at a time share
//      one load of the multipliers); rows 0..4 of the result are final entries of U and go to shared memory;
//   C  the trailing (N-5) x (N-5) block -- B rows: diagonal only; positions 8, 9: from B -- is factorised and
//      solved in registers with full partial pivoting (lu_panel), so a B row losing the pivot to a q / dP row
//      is handled like any other exchange;
//   D  back substitution of the unknowns 4..0.
// Every element receives the same updates in the same order as in og_lu_solve / lu_solve except those skipped
// no-ops, which can change nothing but the sign of an exact zero.
// ---------------------------------------------------------------------------------------------------------
template <int N, int BLOCK, class A>
__device__ __forceinline__ bool lu_solve_structured(A &ar, const JacView<N, BLOCK> &jac, double (&b)[N]) {
  constexpr int NA = N - 3;   // active rows
  constexpr int NT = N - 5;   // trailing block
  constexpr int G = 5;   // columns of block B updated per load of the multipliers (1, 2 and 5 measured: 5)
  int ro[NA];
  double ba[NA];
#pragma unroll
  for (int a = 0; a < NA; a++) {
    const int pos = a < 5 ? a : a + 3;
    ro[a] = JacView<N, BLOCK>::row(pos);
    ba[a] = b[pos];
  }
  bool ok = true;
  // A
#pragma unroll
  for (int j = 0; j < 5; j++) {
    double x[NA];
#pragma unroll
    for (int a = 0; a < NA; a++) x[a] = jac.at(ro[a], j);
#pragma unroll
    for (int k = 0; k < j; k++) {
#pragma unroll
      for (int a = k + 1; a < NA; a++) {
        const double l = jac.at(ro[a], k);
        x[a] = x[a] - l * x[k];
      }
    }
    int p = j;
    double xp = x[j], amax = fabs(x[j]);
#pragma unroll
    for (int a = j + 1; a < NA; a++) {
      const double v = fabs(x[a]);
      const bool gt = v > amax;
      amax = gt ? v : amax;
      xp = gt ? x[a] : xp;
      p = gt ? a : p;
    }
    ok = ok && (amax > 0.0) && isfinite(amax);
    const double r = ar.rcp(xp);
    const int roj = ro[j];
    int rop = roj;
#pragma unroll
    for (int a = j + 1; a < NA; a++) rop = (p == a) ? ro[a] : rop;
#pragma unroll
    for (int a = 0; a < j; a++) jac.at(ro[a], j) = x[a];
#pragma unroll
    for (int a = j; a < NA; a++) jac.at(ro[a], j) = x[a] * r;
    jac.at(rop, j) = r;
#pragma unroll
    for (int a = j + 1; a < NA; a++) ro[a] = (p == a) ? roj : ro[a];
    ro[j] = rop;
    swap_positions<NA>(ba, j, p);
  }
  // B
  double T[NT][NT], t[NT];
#pragma unroll
  for (int c0 = 5; c0 < N; c0 += G) {
    double x[G][NA];
#pragma unroll
    for (int g = 0; g < G; g++)
#pragma unroll
      for (int a = 0; a < NA; a++)
        if (c0 + g < N) x[g][a] = jac.at(ro[a], c0 + g);
    const bool with_rhs = (c0 + G >= N);
#pragma unroll
    for (int k = 0; k < 5; k++) {
#pragma unroll
      for (int a = k + 1; a < NA; a++) {
        const double l = jac.at(ro[a], k);
#pragma unroll
        for (int g = 0; g < G; g++)
          if (c0 + g < N) x[g][a] = x[g][a] - l * x[g][k];
        if (with_rhs) ba[a] = ba[a] - l * ba[k];
      }
    }
#pragma unroll
    for (int g = 0; g < G; g++) {
      if (c0 + g < N) {
#pragma unroll
        for (int a = 0; a < 5; a++) jac.at(ro[a], c0 + g) = x[g][a];
#pragma unroll
        for (int a = 5; a < NA; a++) T[c0 + g - 5][a - 2] = x[g][a];
      }
    }
  }
  // C
#pragma unroll
  for (int c = 0; c < NT; c++)
#pragma unroll
    for (int i = 0; i < 3; i++) T[c][i] = (c == i) ? jac.at(JacView<N, BLOCK>::row(5 + i), 5 + i) : 0.0;
#pragma unroll
  for (int i = 0; i < 3; i++) t[i] = b[5 + i];
#pragma unroll
  for (int a = 5; a < NA; a++) t[a - 2] = ba[a];
  {
    int rdummy[NT];
#pragma unroll
    for (int i = 0; i < NT; i++) rdummy[i] = 0;
    double tinv[NT];
    const JacView<NT, BLOCK> nojac{jac.base};
    lu_panel<NT, BLOCK, 0, NT, true, false>(ar, nojac, rdummy, T, t, tinv, ok);
#pragma unroll
    for (int i = NT - 1; i >= 0; i--) {
      double sacc = t[i];
#pragma unroll
      for (int j = i + 1; j < NT; j++) sacc = sacc - T[j][i] * t[j];
      t[i] = sacc * tinv[i];
    }
  }
  // D
#pragma unroll
  for (int a = 4; a >= 0; a--) {
    double sacc = ba[a];
#pragma unroll
    for (int j = a + 1; j < N; j++) sacc = sacc - jac.at(ro[a], j) * (j < 5 ? ba[j] : t[j - 5]);
    ba[a] = sacc * jac.at(ro[a], a);
  }
#pragma unroll
  for (int i = 0; i < 5; i++) b[i] = ba[i];
#pragma unroll
  for (int i = 5; i < N; i++) b[i] = t[i - 5];
  return ok;
}

// eq 25 (L230): minimiser of the quadratic through f(0), f'(0) = -2 f(0), f(lam)
template <class A>
__device__ __forceinline__ double linesearch_lambda(A &ar, double f0, double flam, double lam) {
  return ar.div(f0, flam + (2.0 * lam - 1.0) * f0) * lam * lam;
}

// Runs at most max_iters further Newton iterations (<= 0: until terminal) of one zone.  P, iters, status carry
// the zone's state between calls.  Returns ||R(P)||_2 of the final state.
template <int N, bool RED, int BLOCK, class A, class Prob>
__device__ __forceinline__ double newton_zone(A &ar, const Prob &prob, const SolverParams &sp, double tol, double (&P)[N],
                                              int &iters, int &status, int max_iters,
                                              const JacView<Unknowns<N, RED>::M, BLOCK> &jac, int &backtracks,
                                              const Pieces *pc0 = nullptr) {
  using U = Unknowns<N, RED>;
  constexpr int M = U::M;
  double R0[N];
  Pieces pc;
  int k = iters, st = status, done = 0;
  if (pc0) {  // the caller has the state pieces of P already
    pc = *pc0;
    prob.assemble(P, pc, R0);
  } else {
    eval_full<N>(ar, prob, P, pc, R0);
  }
  double f0 = norm2sq_rows<N, RED>(R0);
  if (!isfinite(f0)) {
    status = st | ST_NONFINITE;
    return ExactArith().sqrt(f0);
  }
  while (!(ar.sqrt_z(f0) < tol) && k < sp.kmax && (max_iters <= 0 || done < max_iters)) {
    bool singular = false;
    FdColumns<0, N, RED, BLOCK, A, Prob>::run(ar, prob, sp, P, pc, R0, jac, singular);
    double dP[M];
#pragma unroll
    for (int v = 0; v < M; v++) dP[v] = -R0[U::prim(v)];
    bool ok;
    if constexpr (use_structure<N, RED>()) {
      ok = lu_solve_structured<M, BLOCK>(ar, jac, dP);
    } else {
      ok = lu_solve<M, BLOCK>(ar, jac, dP);
    }
    if (singular || !ok) {
      st |= ST_SINGULAR;
      break;
    }
    double lam = 1.0, ft = f0;
    bool accepted = false;
    double Pt[N], Rt[N];
    for (int ls = 0; ls <= sp.lsmax; ls++) {
#pragma unroll
      for (int v = 0; v < N; v++) Pt[v] = P[v];  // the fixed B^i of the reduced solve
#pragma unroll
      for (int v = 0; v < M; v++) Pt[U::prim(v)] = P[U::prim(v)] + lam * dP[v];
      eval_full<N>(ar, prob, Pt, pc, Rt);
      ft = norm2sq_rows<N, RED>(Rt);
      if (isfinite(ft) && ar.sqrt_z(ft) < ar.sqrt_z(f0) * (1.0 - sp.eps_bt * lam)) {
        accepted = true;
        break;
      }
      if (ls == sp.lsmax) break;
      backtracks++;
      lam = isfinite(ft) ? linesearch_lambda(ar, f0, ft, lam) : 0.5 * lam;
    }
    if (!accepted) st |= ST_LS_EXHAUSTED;
#pragma unroll
    for (int v = 0; v < N; v++) {
      P[v] = Pt[v];
      R0[v] = Rt[v];
    }
    f0 = ft;
    k++;
    done++;
    if (!isfinite(f0)) {
      st |= ST_NONFINITE;
      break;
    }
  }
  if (!(st & (ST_SINGULAR | ST_NONFINITE))) {
    if (ar.sqrt_z(f0) < tol) st |= ST_CONVERGED;
    else if (k >= sp.kmax) st |= ST_KMAX;
  }
  iters = k;
  status = st;
  return ar.sqrt_z(f0);
}

}  // namespace grim
