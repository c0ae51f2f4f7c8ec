// kernels_newton.cu -- the fused per-zone Newton kernels (steps a4-a7 of the hot path).
//   newton_stage_kernel : one stage of the time step, one thread per interior zone.  Reads P^k, P_n, P_E, C, G
//                         once, iterates on chip, writes P^{k'}, ||R||, status, iterations once.
//   invert_kernel       : standalone primitive recovery on flat arrays, over a compacted list of active zones.
#include "grim_internal.h"
#include "problems.cuh"

namespace grim {

static constexpr int NB = 128;  // threads per block; 2 blocks/SM: 2 x 128 x (N*N*8 B) of Jacobian + 255 registers

struct StageArgs {
  const double *Pn, *PE, *C, *Gx;
  const double *Pguess;  // P^k is read from here and P^k' written to Piter (the two may be the same array)
  double dt_stage;
  int max_iters;
  int fresh;             // != 0: a new solve; status and iters start at zero without being read
  double *Piter, *resnorm;
  int32_t *status, *iters;
  // Active-set sweeps (SURVEY 7.2 "Divergence"): with next_list set (and kmax lowered to the sweep length by the
  // caller), a zone that stops at kmax stores NOTHING and its interior index is appended to next_list
  // (cnt->list_count); a later launch over that list (list != null) solves it afresh with the real kmax.
  const long long *list;
  long long nlist;
  long long *next_list;
};

// One zone of one stage under arithmetic policy A: loads, set-up, Newton iteration, stores.  Returns false
// WITHOUT storing when a speculative operation saw an operand outside its safe range (fp64ops.cuh); the caller
// then replays the zone with ExactArith.  Otherwise packs (rejected line-search trials << 1) | still-active.
template <int N, class G, bool RED, bool APPEND, class A>
__device__ __forceinline__ int stage_zone(A &ar, const GridView &gv, const StageArgs &a, long long z, int i, int j,
                                          int st, double *sj) {
  constexpr int M = Unknowns<N, RED>::M;
  // EMHD full solve: the constants of the q / dP rows go to the unused words of the Jacobian's B rows
  constexpr bool KSM = N == 10 && use_structure<N, RED>();
  static_assert(!KSM || K_COUNT <= 3 * (N - 1), "constants do not fit the free Jacobian words");
  StageProblem<N, G, NB, KSM> prob;
  prob.m = gv.m;
  prob.Cs = sj + M * M * NB;
  prob.Ks = sj;
  if constexpr (G::flat) {
    prob.tau_ = gv.tau_const;
  } else {
    load_geom<0>(gv.geomC, gv.n2d, (long long)j * gv.sz[0] + i, prob.g, prob.tau_);
  }
  double P[N];
  Pieces pc0;
  {
    double Pn_z[N], PE_z[N];
#pragma unroll
    for (int v = 0; v < N; v++) {
      Pn_z[v] = a.Pn[v * gv.zg + z];
      PE_z[v] = a.PE[v * gv.zg + z];
      P[v] = a.Pguess[v * gv.zg + z];
      sj[(M * M + v) * NB] = a.C[v * gv.zg + z];
    }
    if constexpr (RED) {
      // reduced solve (L148): the induction equation has no implicit source, so B^i_new = -(C_B dt') / sqrt(-g)
      // is explicit; it stays fixed during the iteration
#pragma unroll
      for (int d = 0; d < 3; d++) {
        const double b = -(prob.Cs[(B1 + d) * NB] * a.dt_stage);
        if constexpr (G::flat) P[B1 + d] = b;
        else P[B1 + d] = ar.div_z(b, prob.g.sqrtmg());
      }
    }
    double Xq = 0.0, Xd = 0.0, divx = 0.0;
    if constexpr (N == 10) {
      Xq = a.Gx[0 * gv.zg + z];
      Xd = a.Gx[1 * gv.zg + z];
      divx = a.Gx[2 * gv.zg + z];
    }
    full_state<N>(ar, prob.m, prob.g, prob.tau_, P, pc0.th, pc0.v, pc0.b, pc0.h);
    prob.setup(ar, Pn_z, PE_z, a.dt_stage, pc0, !RED && a.PE == a.Pguess, !RED && a.Pn == a.Pguess, Xq, Xd, divx);
  }
  const double tol = gv.sp.atol + gv.sp.rtol * prob.scale;
  int it = a.fresh ? 0 : a.iters[z];
  int nbt = 0;
  JacView<M, NB> jac{sj};
  double rn = newton_zone<N, RED, NB>(ar, prob, gv.sp, tol, P, it, st, a.max_iters, jac, nbt, &pc0);
  if (!ar.good()) return -1;
  // first sweep (launched with kmax = the sweep length): a zone that ran out of iterations is deferred to the next
  // sweep -- nothing stored, nothing counted
  if (APPEND && (st & ST_KMAX)) return 1;
#pragma unroll
  for (int v = 0; v < N; v++) a.Piter[v * gv.zg + z] = P[v];
  a.resnorm[z] = rn;
  a.status[z] = st;
  a.iters[z] = it;
  return (nbt << 1) | ((st & ST_TERMINAL) ? 0 : 1);
}

template <int N, class G, bool RED, bool APPEND>
__device__ __noinline__ int stage_zone_replay(const GridView &gv, const StageArgs &a, long long z, int i, int j,
                                              int st, double *sj) {
  ExactArith ar;
  return stage_zone<N, G, RED, APPEND>(ar, gv, a, z, i, j, st, sj);
}

// Resident blocks per SM.  Ideal MHD (64 + 8 doubles of shared memory per zone) and the reduced solve ((N-3)^2 + N) would
// have room for 3 blocks at 170 registers; 2 at 255 registers measured faster.
static constexpr int N8_MINB = 2, RED_MINB = 2;
// One thread's zone of a launch: interior zone zt (have = false: the thread has none).  Returns the packed result of
// stage_zone with the deferred zones appended to a.next_list and removed from the count.
template <int N, class G, bool RED, bool APPEND>
__device__ __forceinline__ int stage_thread(const GridView &gv, const StageArgs &a, Counters *cnt, long long zt, bool have,
                                            double *sj) {
  int res = 0;
  if (have) {
    int i, j, k;
    zone_coords(gv, zt, i, j, k);
    const long long z = zone_index(gv, i, j, k);
    const int st = a.fresh ? 0 : a.status[z];
    if (!(st & ST_TERMINAL)) {
      SpecArith ar;
      res = stage_zone<N, G, RED, APPEND>(ar, gv, a, z, i, j, st, sj);
      if (res < 0) res = stage_zone_replay<N, G, RED, APPEND>(gv, a, z, i, j, st, sj);
    }
  }
  if constexpr (APPEND) {
    // warp-aggregated append of the deferred zones (order not deterministic; the per-zone results are)
    const unsigned ballot = __ballot_sync(0xffffffffu, res & 1);
    const int lane = threadIdx.x & 31;
    unsigned long long base = 0;
    if (lane == 0 && ballot) base = atomicAdd(&cnt->list_count, (unsigned long long)__popc(ballot));
    base = __shfl_sync(0xffffffffu, base, 0);
    if (res & 1) a.next_list[base + __popc(ballot & ((1u << lane) - 1u))] = zt;
    res &= ~1;
  }
  return res;
}

// APPEND: first sweep (zones that stop at the lowered kmax are deferred to a.next_list)
template <int N, class G, bool RED, bool APPEND>
__global__ void __launch_bounds__(NB, RED ? RED_MINB : (N == 8 ? N8_MINB : 256 / NB))
newton_stage_kernel(const __grid_constant__ GridView gv, const __grid_constant__ StageArgs a, Counters *cnt) {
  extern __shared__ double smem[];
  const long long t = (long long)blockIdx.x * NB + threadIdx.x;
  const int res = stage_thread<N, G, RED, APPEND>(gv, a, cnt, t, t < gv.nint, smem + threadIdx.x);
  // warp-aggregated counters
  unsigned long long na = __reduce_add_sync(0xffffffffu, (unsigned)(res & 1));
  unsigned long long nb = __reduce_add_sync(0xffffffffu, (unsigned)(res >> 1));
  if ((threadIdx.x & 31) == 0) {
    if (na) atomicAdd(&cnt->n_active, na);
    if (nb) atomicAdd(&cnt->backtracks, nb);
  }
}

// The launch over a list of deferred zones whose length is on the device (cnt->list_count, written by the launch
// before): a resident grid of blocks strides over the list, so that the host need not know the length.
template <int N, class G, bool RED>
__global__ void __launch_bounds__(NB, RED ? RED_MINB : (N == 8 ? N8_MINB : 256 / NB))
newton_stage_list_kernel(const __grid_constant__ GridView gv, const __grid_constant__ StageArgs a, Counters *cnt) {
  extern __shared__ double smem[];
  const long long nlist = (long long)cnt->list_count;
  unsigned n_act = 0, n_bt = 0;
  for (long long t0 = (long long)blockIdx.x * NB; t0 < nlist; t0 += (long long)gridDim.x * NB) {
    const long long t = t0 + threadIdx.x;
    const bool have = t < nlist;
    const int res = stage_thread<N, G, RED, false>(gv, a, cnt, have ? a.list[t] : 0, have, smem + threadIdx.x);
    n_act += (unsigned)(res & 1);
    n_bt += (unsigned)(res >> 1);
  }
  unsigned long long na = __reduce_add_sync(0xffffffffu, n_act);
  unsigned long long nb = __reduce_add_sync(0xffffffffu, n_bt);
  if ((threadIdx.x & 31) == 0) {
    if (na) atomicAdd(&cnt->n_active, na);
    if (nb) atomicAdd(&cnt->backtracks, nb);
  }
}

template <int N, class G, bool RED>
static int launch_stage_t(const GridView &gv, const double *Pn, const double *PE, const double *C, const double *Gx,
                          const double *Pguess, int fresh, double dt_stage, int max_iters, double *Piter, double *resnorm, int32_t *status,
                          int32_t *iters, Counters *cnt, cudaStream_t s, const long long *list, long long nlist,
                          long long *next_list) {
  constexpr int M = Unknowns<N, RED>::M;
  const size_t smem = (size_t)(M * M + N) * NB * sizeof(double);  // Jacobian + C per thread
  // per device and context, so set before every launch (cheap); a failure surfaces as the launch error
  const StageArgs a{Pn, PE, C, Gx, Pguess, dt_stage, max_iters, fresh, Piter, resnorm, status, iters, list, nlist, next_list};
  if (list) {
    // the list's length is cnt->list_count on the device: a resident grid strides over it (nothing to do: ~5 us)
    cudaFuncSetAttribute(newton_stage_list_kernel<N, G, RED>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const int per_sm = RED ? RED_MINB : (N == 8 ? N8_MINB : 256 / NB);
    newton_stage_list_kernel<N, G, RED><<<(unsigned)(per_sm * (gv.nsm > 0 ? gv.nsm : 148)), NB, smem, s>>>(gv, a, cnt);
    return 1;
  }
  const long long blocks = (gv.nint + NB - 1) / NB;
  if (blocks == 0) return 0;
  if (next_list) {
    cudaFuncSetAttribute(newton_stage_kernel<N, G, RED, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    newton_stage_kernel<N, G, RED, true><<<(unsigned)blocks, NB, smem, s>>>(gv, a, cnt);
  } else {
    cudaFuncSetAttribute(newton_stage_kernel<N, G, RED, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    newton_stage_kernel<N, G, RED, false><<<(unsigned)blocks, NB, smem, s>>>(gv, a, cnt);
  }
  return 1;
}

int launch_newton_stage(const GridView &gv, const double *Pn, const double *PE, const double *C, const double *G,
                        const double *Pguess, int fresh, double dt_stage, int max_iters, double *Piter, double *resnorm, int32_t *status,
                        int32_t *iters, Counters *cnt, cudaStream_t s, const long long *list, long long nlist,
                        long long *next_list) {
  const bool flat = (gv.metric == 0);
#define GRIM_STAGE(NV, GG, RR)                                                                                      \
  launch_stage_t<NV, GG, RR>(gv, Pn, PE, C, G, Pguess, fresh, dt_stage, max_iters, Piter, resnorm, status, iters, cnt, s, \
                             list, nlist, next_list)
  if (gv.reduced) {
    if (gv.nvar == 10) return flat ? GRIM_STAGE(10, GeomFlat, true) : GRIM_STAGE(10, GeomGen, true);
    return flat ? GRIM_STAGE(8, GeomFlat, true) : GRIM_STAGE(8, GeomGen, true);
  }
  if (gv.nvar == 10) return flat ? GRIM_STAGE(10, GeomFlat, false) : GRIM_STAGE(10, GeomGen, false);
  return flat ? GRIM_STAGE(8, GeomFlat, false) : GRIM_STAGE(8, GeomGen, false);
#undef GRIM_STAGE
}

// ---------------------------------------------------------------------------------------------------------
// Standalone inversion.  `first` != 0: thread t handles zone t of all nz zones, iters/status start at zero.
// Otherwise thread t handles zone list[t], t < nlist.  Zones left without a terminal status are appended to
// next_list (order is not deterministic; the per-zone results are).
// ---------------------------------------------------------------------------------------------------------
struct InvertArgs {
  long long nz, nlist;
  const long long *list;
  const double *Ustar;
  double *Pio;
  int32_t *iters, *status;
  double *resnorm;
  int max_iters, first;
  long long *next_list;
  const double *geom;  // per-zone geometry, INV_GEOM_NCOMP x nz (include/grim.h), or null: Minkowski
};

// One zone of the standalone inversion under arithmetic policy A; same protocol as stage_zone.
template <int N, class G, class A>
__device__ __forceinline__ int invert_zone(A &ar, const GridView &gv, const InvertArgs &a, long long z, double *sj) {
  InvertProblem<N, G, NB> prob;
  prob.m = gv.m;
  prob.Us = sj + N * N * NB;
  prob.tau_ = gv.tau_const;
  if constexpr (!G::flat) {
    // g_mu_nu (sym4 order), g^{t i}, sqrt(-g), alpha of this zone; beta^i/alpha = alpha g^{t i} (C-9)
#pragma unroll
    for (int c = 0; c < 10; c++) prob.g.g[c] = a.geom[c * a.nz + z];
    prob.g.sg = a.geom[13 * a.nz + z];
    prob.g.alpha = a.geom[14 * a.nz + z];
#pragma unroll
    for (int i = 0; i < 3; i++) prob.g.bfac[i] = prob.g.alpha * a.geom[(10 + i) * a.nz + z];
    prob.g.gcon00 = prob.g.gcon0d = prob.g.gcondd = 0.0;
  }
  double P[N];
#pragma unroll
  for (int v = 0; v < N; v++) {
    sj[(N * N + v) * NB] = a.Ustar[v * a.nz + z];
    P[v] = a.Pio[v * a.nz + z];
  }
  prob.setup(ar);
  int it = a.first ? 0 : a.iters[z];
  int st = a.first ? 0 : a.status[z];
  int nbt = 0;
  JacView<N, NB> jac{sj};
  double rn = newton_zone<N, false, NB>(ar, prob, gv.sp, gv.sp.rtol, P, it, st, a.max_iters, jac, nbt);
  if (!ar.good()) return -1;
#pragma unroll
  for (int v = 0; v < N; v++) a.Pio[v * a.nz + z] = P[v];
  a.resnorm[z] = rn;
  a.status[z] = st;
  a.iters[z] = it;
  return (nbt << 1) | ((st & ST_TERMINAL) ? 0 : 1);
}

template <int N, class G>
__device__ __noinline__ int invert_zone_replay(const GridView &gv, const InvertArgs &a, long long z, double *sj) {
  ExactArith ar;
  return invert_zone<N, G>(ar, gv, a, z, sj);
}

template <int N, class G>
__global__ void __launch_bounds__(NB, N == 8 ? N8_MINB : 256 / NB)
invert_kernel(const __grid_constant__ GridView gv, const __grid_constant__ InvertArgs a, Counters *cnt) {
  extern __shared__ double smem[];
  const long long t = (long long)blockIdx.x * NB + threadIdx.x;
  int res = 0;
  long long z = -1;
  if (t < a.nlist) {
    z = a.first ? t : a.list[t];
    SpecArith ar;
    res = invert_zone<N, G>(ar, gv, a, z, smem + threadIdx.x);
    if (res < 0) res = invert_zone_replay<N, G>(gv, a, z, smem + threadIdx.x);
  }
  const int active_after = res & 1;
  // warp-aggregated append to the next active list
  const unsigned ballot = __ballot_sync(0xffffffffu, active_after);
  const int lane = threadIdx.x & 31;
  unsigned long long base = 0;
  if (lane == 0 && ballot) base = atomicAdd(&cnt->list_count, (unsigned long long)__popc(ballot));
  base = __shfl_sync(0xffffffffu, base, 0);
  if (active_after) a.next_list[base + __popc(ballot & ((1u << lane) - 1u))] = z;
  unsigned long long b = __reduce_add_sync(0xffffffffu, (unsigned)(res >> 1));
  if (lane == 0 && b) atomicAdd(&cnt->backtracks, b);
}

template <int N, class G>
static int launch_invert_t(const GridView &gv, long long nz, long long nlist, const long long *list,
                           const double *Ustar, const double *geom, double *P, int32_t *iters, int32_t *status,
                           double *resnorm, int max_iters, int first, long long *next_list, Counters *cnt,
                           cudaStream_t s) {
  const size_t smem = (size_t)(N * N + N) * NB * sizeof(double);  // Jacobian + C (or U*) per thread
  cudaFuncSetAttribute(invert_kernel<N, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  const long long blocks = (nlist + NB - 1) / NB;
  if (blocks == 0) return 0;
  const InvertArgs a{nz, nlist, list, Ustar, P, iters, status, resnorm, max_iters, first, next_list, geom};
  invert_kernel<N, G><<<(unsigned)blocks, NB, smem, s>>>(gv, a, cnt);
  return 1;
}

int launch_invert(const GridView &gv, long long nz, long long nlist, const long long *list, const double *Ustar,
                  const double *geom, double *P, int32_t *iters, int32_t *status, double *resnorm, int max_iters,
                  int first, long long *next_list, Counters *cnt, cudaStream_t s) {
#define GRIM_INV(NV, GG) \
  launch_invert_t<NV, GG>(gv, nz, nlist, list, Ustar, geom, P, iters, status, resnorm, max_iters, first, next_list, cnt, s)
  if (gv.nvar == 10) return geom ? GRIM_INV(10, GeomGen) : GRIM_INV(10, GeomFlat);
  return geom ? GRIM_INV(8, GeomGen) : GRIM_INV(8, GeomFlat);
#undef GRIM_INV
}

// U(P) on flat arrays, Minkowski (workload construction on the device)
template <int N>
__global__ void prim_to_conserved_kernel(GridView gv, long long nz, const double *__restrict__ Pin,
                                         double *__restrict__ Uout) {
  const long long z = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (z >= nz) return;
  double P[N], U[N];
#pragma unroll
  for (int v = 0; v < N; v++) P[v] = Pin[v * nz + z];
  Pieces pc;
  GeomFlat g;
  ExactArith ar;
  full_state<N>(ar, gv.m, g, gv.tau_const, P, pc.th, pc.v, pc.b, pc.h);
  flux_vector<N>(g, 0, P, pc.th, pc.v, pc.b, pc.h, U);
#pragma unroll
  for (int v = 0; v < N; v++) Uout[v * nz + z] = U[v];
}

int launch_prim_to_conserved(const GridView &gv, long long nz, const double *P, double *U, cudaStream_t s) {
  const int tb = 256;
  const long long blocks = (nz + tb - 1) / tb;
  if (blocks == 0) return 0;
  if (gv.nvar == 10) prim_to_conserved_kernel<10><<<(unsigned)blocks, tb, 0, s>>>(gv, nz, P, U);
  else prim_to_conserved_kernel<8><<<(unsigned)blocks, tb, 0, s>>>(gv, nz, P, U);
  return 1;
}

}  // namespace grim

// ---------------------------------------------------------------------------------------------------------
// grim_invert_primitives_static (include/grim.h): the standalone inversion for callers that cannot allocate
// device memory -- plug-ins of an application whose memory pool already owns the device, and time-critical
// loops that cannot afford the device-wide wait of cudaMalloc / cudaFree.  It needs no grim_ctx (whose
// creation allocates) and allocates nothing itself.  The scratch of the sweeps -- the counters and the two
// lists of zones that are still iterating -- is the array below: part of the library's device image, so
// every GPU that loads the library carries its 8 MiB + 256 B until the process ends.
//
// Everything that touches the array is in this file.  Device code may name `static_scratch` directly.  HOST
// code may not: on the host the name is only a handle for the runtime (a kernel handed `static_scratch` from
// host code would fault, or on a system where the GPU can read host memory, quietly use the wrong bytes).
// The host gets the real device address once per device from cudaGetSymbolAddress, with that device current,
// and passes it to the kernels and to cudaMemsetAsync.
//
// Layout: [0, 56)  Counters      [256, 256 + 4 MAXZ)  list 0      [256 + 4 MAXZ, 256 + 8 MAXZ)  list 1
// (zone numbers fit 32 bits because nz <= GRIM_STATIC_MAX_ZONES).  The array is shared by every call on the
// device and keeps the previous call's contents; see the header for what that means for the caller.
// ---------------------------------------------------------------------------------------------------------
#include <string.h>

#include <mutex>
#include <string>

#include "../../include/grim.h"

namespace grim {

static constexpr long long STATIC_MAXZ = GRIM_STATIC_MAX_ZONES;
static constexpr size_t STATIC_LIST_OFFSET = 256;
static constexpr size_t STATIC_SCRATCH_BYTES = STATIC_LIST_OFFSET + 2 * sizeof(uint32_t) * (size_t)STATIC_MAXZ;
static_assert(sizeof(Counters) <= STATIC_LIST_OFFSET, "counters must fit in front of the lists");

static __device__ __align__(256) unsigned char static_scratch[STATIC_SCRATCH_BYTES];

// invert_kernel with 32-bit lists at caller-supplied addresses (the host passes addresses inside static_scratch).
// Zones are solved by the same invert_zone as the allocating path, so a zone's result is the same bits.
template <int N, class G>
__global__ void __launch_bounds__(NB, N == 8 ? N8_MINB : 256 / NB)
invert_static_kernel(const __grid_constant__ GridView gv, const __grid_constant__ InvertArgs a, Counters *cnt,
                     const uint32_t *__restrict__ list, uint32_t *__restrict__ next_list) {
  extern __shared__ double smem[];
  const long long t = (long long)blockIdx.x * NB + threadIdx.x;
  int res = 0;
  long long z = -1;
  if (t < a.nlist) {
    z = a.first ? t : (long long)list[t];
    SpecArith ar;
    res = invert_zone<N, G>(ar, gv, a, z, smem + threadIdx.x);
    if (res < 0) res = invert_zone_replay<N, G>(gv, a, z, smem + threadIdx.x);
  }
  const int active_after = res & 1;
  const unsigned ballot = __ballot_sync(0xffffffffu, active_after);
  const int lane = threadIdx.x & 31;
  unsigned long long base = 0;
  if (lane == 0 && ballot) base = atomicAdd(&cnt->list_count, (unsigned long long)__popc(ballot));
  base = __shfl_sync(0xffffffffu, base, 0);
  if (active_after) next_list[base + __popc(ballot & ((1u << lane) - 1u))] = (uint32_t)z;
  unsigned long long b = __reduce_add_sync(0xffffffffu, (unsigned)(res >> 1));
  if (lane == 0 && b) atomicAdd(&cnt->backtracks, b);
}

template <int N, class G>
static cudaError_t static_kernel_setup() {
  return cudaFuncSetAttribute(invert_static_kernel<N, G>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)((size_t)(N * N + N) * NB * sizeof(double)));
}

template <int N, class G>
static void static_kernel_launch(const GridView &gv, const InvertArgs &a, Counters *cnt, const uint32_t *list,
                                 uint32_t *next_list, cudaStream_t s) {
  const size_t smem = (size_t)(N * N + N) * NB * sizeof(double);
  const long long blocks = (a.nlist + NB - 1) / NB;
  invert_static_kernel<N, G><<<(unsigned)blocks, NB, smem, s>>>(gv, a, cnt, list, next_list);
}

// Device address of static_scratch on `device` (which must be current); the first call per device asks the runtime
// and configures the four kernel variants.  Returns cudaSuccess or the failing call's code.
static constexpr int STATIC_MAX_DEVICES = 64;
static std::mutex static_mu;
static unsigned char *static_addr[STATIC_MAX_DEVICES];

static cudaError_t static_scratch_address(int device, unsigned char **out) {
  std::lock_guard<std::mutex> lock(static_mu);
  if (!static_addr[device]) {
    int major = 0;
    cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device);
    if (e != cudaSuccess) return e;
    if (major != 10) return cudaErrorNoKernelImageForDevice;  // sm_100a only, as grim_init_grid
    unsigned char *p = nullptr;
    e = cudaGetSymbolAddress((void **)&p, static_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    if ((e = static_kernel_setup<8, GeomFlat>()) != cudaSuccess) return e;
    if ((e = static_kernel_setup<8, GeomGen>()) != cudaSuccess) return e;
    if ((e = static_kernel_setup<10, GeomFlat>()) != cudaSuccess) return e;
    if ((e = static_kernel_setup<10, GeomGen>()) != cudaSuccess) return e;
    static_addr[device] = p;
  }
  *out = static_addr[device];
  return cudaSuccess;
}

void set_global_error(const char *msg);  // api.cu: the text grim_last_error(NULL) returns

static int static_fail(int code, const std::string &msg) {
  set_global_error(msg.c_str());
  return code;
}

}  // namespace grim

extern "C" int grim_invert_primitives_static(const grim_grid_desc *d, int64_t nz, const double *U_target,
                                             const double *geom, double *P_inout, int32_t *iters, int32_t *status,
                                             double *resnorm) {
  using namespace grim;
  const char *me = "grim_invert_primitives_static: ";
  if (!d) return static_fail(GRIM_EINVAL, std::string(me) + "null descriptor");
  if (nz < 0 || (nz > 0 && (!U_target || !P_inout || !iters || !status || !resnorm)))
    return static_fail(GRIM_EINVAL, std::string(me) + "bad argument");
  if (nz > STATIC_MAXZ)
    return static_fail(GRIM_EINVAL, std::string(me) + "nz = " + std::to_string((long long)nz) +
                                        " exceeds GRIM_STATIC_MAX_ZONES = " + std::to_string(STATIC_MAXZ) +
                                        " (the fixed scratch array holds no more): split the batch or use "
                                        "grim_invert_primitives");
  if (d->model != GRIM_IDEAL && d->model != GRIM_EMHD) return static_fail(GRIM_EINVAL, std::string(me) + "model must be 8 or 10");
  if (!(d->gamma > 1.0)) return static_fail(GRIM_EINVAL, std::string(me) + "adiabatic index must exceed 1");
  if (!(d->fd_eps > 0.0) || d->kmax < 0 || d->lsmax < 0) return static_fail(GRIM_EINVAL, std::string(me) + "bad solver parameters");
  if (d->closure != GRIM_CLOSURE_CS2TAU && d->closure != GRIM_CLOSURE_CONST)
    return static_fail(GRIM_EINVAL, std::string(me) + "unknown closure");
  if (d->model == GRIM_EMHD && !(d->tau_mode == GRIM_TAU_R32 || d->tau > 0.0))
    return static_fail(GRIM_EINVAL, std::string(me) + "tau_R must be positive");
  if (nz == 0) return GRIM_OK;

#define SCU(call)                                                                                       \
  do {                                                                                                  \
    cudaError_t e_ = (call);                                                                            \
    if (e_ != cudaSuccess) return static_fail(GRIM_ECUDA, std::string(me) + #call + ": " + cudaGetErrorString(e_)); \
  } while (0)

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
    return static_fail(GRIM_ECUDA, std::string(me) + "no CUDA device: this library has no CPU fallback");
  if (d->device < 0 || d->device >= ndev || d->device >= STATIC_MAX_DEVICES)
    return static_fail(GRIM_EINVAL, std::string(me) + "device ordinal out of range");
  SCU(cudaSetDevice(d->device));
  unsigned char *base = nullptr;
  SCU(static_scratch_address(d->device, &base));
  Counters *cnt = (Counters *)base;
  uint32_t *lists[2] = {(uint32_t *)(base + STATIC_LIST_OFFSET),
                        (uint32_t *)(base + STATIC_LIST_OFFSET + sizeof(uint32_t) * (size_t)STATIC_MAXZ)};
  cudaStream_t s = (cudaStream_t)d->stream;

  // the part of the grid view the inversion reads: model, solver parameters, constant tau_R
  GridView gv;
  memset(&gv, 0, sizeof(gv));
  gv.nvar = d->model;
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

  // Sweeps of 4 iterations over the zones that are still iterating, as grim_invert_primitives runs them (where a
  // zone's iteration pauses does not change its result).  The counters start every sweep at zero; the list a sweep
  // reads was written in full by the sweep before it, so stale entries of earlier calls are never read.
  const int sweep = 4;
  long long nlist = nz;
  int first = 1, cur = 0, done_iters = 0;
  while (nlist > 0) {
    SCU(cudaMemsetAsync(cnt, 0, sizeof(Counters), s));
    const InvertArgs a{nz, nlist, nullptr, U_target, P_inout, iters, status, resnorm, sweep, first, nullptr, geom};
    if (gv.nvar == 10) {
      if (geom) static_kernel_launch<10, GeomGen>(gv, a, cnt, lists[cur], lists[cur ^ 1], s);
      else static_kernel_launch<10, GeomFlat>(gv, a, cnt, lists[cur], lists[cur ^ 1], s);
    } else {
      if (geom) static_kernel_launch<8, GeomGen>(gv, a, cnt, lists[cur], lists[cur ^ 1], s);
      else static_kernel_launch<8, GeomFlat>(gv, a, cnt, lists[cur], lists[cur ^ 1], s);
    }
    SCU(cudaGetLastError());
    unsigned long long left = 0;
    SCU(cudaMemcpyAsync(&left, &cnt->list_count, sizeof(left), cudaMemcpyDeviceToHost, s));
    SCU(cudaStreamSynchronize(s));
    nlist = (long long)left;
    cur ^= 1;
    first = 0;
    done_iters += sweep;
    if (done_iters > d->kmax + 8) break;  // cannot happen: every zone reaches kmax
  }
#undef SCU
  return GRIM_OK;
}
