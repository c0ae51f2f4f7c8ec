// kernels_flux.cu -- steps a1-a3 of the hot path: reconstruction (L154-160), LLF fluxes (eq 17) with the
// wave-speed bound of eqs 43-48, flux divergence (eq 10) and the stage constant
//     C = -U(P_n)/dt' + div F(P_E) - S^E(P_E)                                       (L438; eq 19 / eq 13; C-5)
// plus, for EMHD, the spatial-gradient terms (Xq, Xd, divx) of the relaxation targets (eqs 37-38; O-8).
//
//   face_flux_kernel<DIR> : one thread per lower face of direction DIR, on block tiles whose stencil zones are
//                           staged in shared memory; reconstructs the two face states from the 4- (minmod) or
//                           6-point (MP5) stencil, evaluates U, F^DIR, c at both with the face-centre geometry
//                           (C-8) and stores the LLF (eq 17) or HLLE (eq 18) flux and the face speed.
//   face_box_kernel<DIR>  : the same for the faces the tiles leave out (upper boundary plane; with flux-CT the
//                           transverse ghost fringe), stencil read directly.
//   emf_kernel            : flux-CT, face -> edge averages (L327-335).
//   stage_const_kernel    : one thread per interior zone; differences the face fluxes, adds -U(P_n)/dt' and the
//                           explicit sources, limited slopes of the derived quantities, max wave-speed figures.
#include <type_traits>

#include "grim_internal.h"
#include "problems.cuh"
#include "recon.cuh"
#include "tma.cuh"

namespace grim {

static constexpr int FB = 128;

// Stencil sources of a face: m = 0 .. H-1 counts the zones of the stencil upwards along DIR, H = 6 (MP5:
// zones i-3 .. i+2 of lower face i) or 4 (minmod: i-2 .. i+1).
struct GlobalStencil {  // straight from the grid array (replay path)
  const double *p;      // variable 0 at the lowest zone of the stencil
  long long stride, zg;
  __device__ __forceinline__ double operator()(int v, int m) const { return p[v * zg + m * stride]; }
};
template <int VS, int MS>
struct TileStencil {    // from the block's shared-memory tile: variable stride VS, stencil stride MS (doubles)
  const double *p;
  __device__ __forceinline__ double operator()(int v, int m) const { return p[v * VS + m * MS]; }
};

// LLF flux and face speed of one lower DIR-face under arithmetic policy A
template <int N, int RECON, class G, int DIR, class A, class S>
__device__ __forceinline__ void face_compute(A &ar, const GridView &gv, const S &st, int i, int j, double (&F)[N],
                                             double &c) {
  double Pm[N], Pp[N];  // P^- (from zone i-1) and P^+ (from zone i) at the face (L158-160)
#pragma unroll
  for (int v = 0; v < N; v++) {
    double hi, lo, unused;
    if constexpr (RECON == 1) {
      const double s0 = st(v, 0), s1 = st(v, 1), s2 = st(v, 2), s3 = st(v, 3), s4 = st(v, 4), s5 = st(v, 5);
      hi = mp5_face(ar, s0, s1, s2, s3, s4);
      lo = mp5_face(ar, s5, s4, s3, s2, s1);
    } else {
      const double s1 = st(v, 0), s2 = st(v, 1), s3 = st(v, 2), s4 = st(v, 3);
      reconstruct<0>(ar, gv.theta, 0.0, s1, s2, s3, 0.0, hi, unused);
      reconstruct<0>(ar, gv.theta, 0.0, s2, s3, s4, 0.0, unused, lo);
    }
    Pm[v] = hi;
    Pp[v] = lo;
  }

  G g;
  double tau = gv.tau_const;
  if constexpr (!G::flat) load_geom<DIR + 1>(gv.geomF[DIR], gv.n2d, (long long)j * gv.sz[0] + i, g, tau);

  Pieces sm, sp;
  full_state<N>(ar, gv.m, g, tau, Pm, sm.th, sm.v, sm.b, sm.h);
  full_state<N>(ar, gv.m, g, tau, Pp, sp.th, sp.v, sp.b, sp.h);
  double Um[N], Up[N], Fm[N], Fp[N];
  flux_vector<N>(g, 0, Pm, sm.th, sm.v, sm.b, sm.h, Um);
  flux_vector<N>(g, 0, Pp, sp.th, sp.v, sp.b, sp.h, Up);
  flux_vector<N>(g, DIR + 1, Pm, sm.th, sm.v, sm.b, sm.h, Fm);
  flux_vector<N>(g, DIR + 1, Pp, sp.th, sp.v, sp.b, sp.h, Fp);
  double vpm, vnm, vpp, vnp;  // upper / lower speed bound of the minus state, of the plus state
  wave_speeds_dir(ar, g, vmax2<N>(ar, gv.m, tau, Pm[RHO], Pm[UU], sm.b.bsq), sm.v.ucon[0], sm.v.ucon[DIR + 1], vpm,
                  vnm);
  wave_speeds_dir(ar, g, vmax2<N>(ar, gv.m, tau, Pp[RHO], Pp[UU], sp.b.bsq), sp.v.ucon[0], sp.v.ucon[DIR + 1], vpp,
                  vnp);
  const double cm = fmax(fabs(vpm), fabs(vnm));
  const double cp = fmax(fabs(vpp), fabs(vnp));
  c = fmax(cm, cp);  // L164: c_max >= max |c^+-| over both states
  if (gv.riemann == 1) {  // HLLE, eq 18 (L168-170): bounds on the right- and left-going speeds of both states
    const double cR = fmax(0.0, fmax(fmax(vpm, vnm), fmax(vpp, vnp)));
    const double cL = fmax(0.0, fmax(fmax(-vpm, -vnm), fmax(-vpp, -vnp)));
    const double den = cL + cR;
#pragma unroll
    for (int v = 0; v < N; v++) F[v] = ar.div_z(cR * Fm[v] + cL * Fp[v] - cR * cL * (Up[v] - Um[v]), den);
  } else {
#pragma unroll
    for (int v = 0; v < N; v++) F[v] = 0.5 * (Fp[v] + Fm[v]) - 0.5 * c * (Up[v] - Um[v]);  // eq 17
  }
}

template <int N, int RECON, class G, int DIR>
__device__ __noinline__ void face_replay(const GridView &gv, const double *__restrict__ PE, long long z, int i, int j,
                                         double *__restrict__ Fface, double *__restrict__ cface) {
  ExactArith ar;
  double F[N], c;
  const long long stride = (DIR == 0) ? 1 : (DIR == 1) ? (long long)gv.sz[0] : (long long)gv.sz[0] * gv.sz[1];
  const GlobalStencil st{PE + z - (RECON == 1 ? 3 : 2) * stride, stride, gv.zg};
  face_compute<N, RECON, G, DIR>(ar, gv, st, i, j, F, c);
#pragma unroll
  for (int v = 0; v < N; v++) Fface[v * gv.zg + z] = F[v];
  cface[z] = c;
}

// Block tile of faces: 128 x 1 x 1 for DIR 0, 32 x 4 x 1 for DIR 1, 32 x 1 x 4 for DIR 2 -- X^1 stays the fast
// index of every load and store, and the tile is 4 faces deep along DIR so that its stencil zones
// (tile + H-1 along DIR) are staged once in shared memory and read 6H/(4+H-1) times: one batch of independent
// coalesced loads per block instead of H dependent-latency loads per variable and thread.
template <int DIR>
struct FaceTile {
  static constexpr int T0 = (DIR == 0) ? 128 : 32, T1 = (DIR == 1) ? 4 : 1, T2 = (DIR == 2) ? 4 : 1;
};

// resident blocks per SM the face kernels are compiled for (flat and general metric: 4 x 128 threads, 128 registers)
static constexpr int FLUX_MINB = 4, FLUX_MINB_GEN = 4;
template <int N, int RECON, class G, int DIR>  // DIR = 0..2
__global__ void __launch_bounds__(FB, G::flat ? FLUX_MINB : FLUX_MINB_GEN)
face_flux_kernel(const __grid_constant__ GridView gv, const double *__restrict__ PE, double *__restrict__ Fface,
                 double *__restrict__ cface) {
  using T = FaceTile<DIR>;
  constexpr int H = (RECON == 1) ? 6 : 4, LO = H / 2;
  constexpr int E0 = T::T0 + (DIR == 0 ? H - 1 : 0), E1 = T::T1 + (DIR == 1 ? H - 1 : 0),
                E2 = T::T2 + (DIR == 2 ? H - 1 : 0), EZ = E0 * E1 * E2;
  constexpr int MS = (DIR == 0) ? 1 : (DIR == 1) ? E0 : E0 * E1;
  __shared__ double tile[N * EZ];

  // padded coordinates of the tile's first face, and of the first staged zone (LO zones below it along DIR)
  const int fi = gv.ngd[0] + (int)blockIdx.x * T::T0, fj = gv.ngd[1] + (int)blockIdx.y * T::T1,
            fk = gv.ngd[2] + gv.koff + (int)blockIdx.z * T::T2;
  const int zi = fi - (DIR == 0 ? LO : 0), zj = fj - (DIR == 1 ? LO : 0), zk = fk - (DIR == 2 ? LO : 0);
  constexpr int ITER = (EZ + FB - 1) / FB;
#pragma unroll
  for (int it = 0; it < ITER; it++) {
    const int e = it * FB + (int)threadIdx.x;
    const int e0 = e % E0, e1 = (e / E0) % E1, e2 = e / (E0 * E1);
    const int ci = zi + e0, cj = zj + e1, ck = zk + e2;
    if (e < EZ && ci < gv.sz[0] && cj < gv.sz[1] && ck < gv.sz[2]) {
      const long long zz = zone_index(gv, ci, cj, ck);
      double tmp[N];
#pragma unroll
      for (int v = 0; v < N; v++) tmp[v] = PE[v * gv.zg + zz];
#pragma unroll
      for (int v = 0; v < N; v++) tile[v * EZ + e] = tmp[v];
    }
  }
  __syncthreads();

  const int t0 = (int)threadIdx.x % T::T0, t1 = ((int)threadIdx.x / T::T0) % T::T1,
            t2 = (int)threadIdx.x / (T::T0 * T::T1);
  const int i = fi + t0, j = fj + t1, k = fk + t2;
  // the tiles cover the n lower faces of the interior zones; the one upper boundary face per line goes to
  // face_edge_kernel, so that the tile grid divides the interior evenly
  if (i >= gv.ngd[0] + gv.n[0] || j >= gv.ngd[1] + gv.n[1] || k >= gv.ngd[2] + gv.koff + gv.n[2]) return;
  const long long z = zone_index(gv, i, j, k);
  SpecArith ar;
  double F[N], c;
  const TileStencil<EZ, MS> st{tile + (t2 * E1 + t1) * E0 + t0};
  face_compute<N, RECON, G, DIR>(ar, gv, st, i, j, F, c);
  if (ar.good()) {
#pragma unroll
    for (int v = 0; v < N; v++) Fface[v * gv.zg + z] = F[v];
    cface[z] = c;
  } else {
    face_replay<N, RECON, G, DIR>(gv, PE, z, i, j, Fface, cface);
  }
}

// The same tiles with the stencil zones brought in by TMA: one bulk tensor copy per block brings the tile's box -- all N
// variables, (T0 + halo) x (T1 + halo) x (T2 + halo) zones, out-of-range zones read as zero -- into shared memory and
// signals the block's mbarrier.  One thread issues the copy; nobody computes addresses or holds staging registers.  (A TMA
// box row starts on a 16-byte boundary and is a multiple of 16 bytes long: the box starts at the even X^1 index at or
// below the first stencil zone and has an even X^1 extent.)  One tile per block: with 4 resident blocks per SM the copies
// of some blocks overlap the arithmetic of others; a persistent, double-buffered form measured slower.
template <int RECON, int DIR>
struct TmaTile {
  using T = FaceTile<DIR>;
  static constexpr int H = (RECON == 1) ? 6 : 4, LO = H / 2;
  // one more zone than the stencil needs, rounded up to even: the box starts at an even X^1 index (see below)
  static constexpr int E0 = (T::T0 + (DIR == 0 ? H - 1 : 0) + 2) / 2 * 2, E1 = T::T1 + (DIR == 1 ? H - 1 : 0),
                       E2 = T::T2 + (DIR == 2 ? H - 1 : 0), EZ = E0 * E1 * E2;
  static constexpr int MS = (DIR == 0) ? 1 : (DIR == 1) ? E0 : E0 * E1;
};
template <int N, int RECON, int DIR>
__host__ __device__ constexpr size_t tma_tile_bytes() {
  return ((size_t)N * TmaTile<RECON, DIR>::EZ * sizeof(double) + 127) / 128 * 128;
}

template <int N, int RECON, class G, int DIR>
__global__ void __launch_bounds__(FB, G::flat ? FLUX_MINB : FLUX_MINB_GEN)
face_flux_tma_kernel(const __grid_constant__ GridView gv, const __grid_constant__ CUtensorMap tmap,
                     const double *__restrict__ PE, double *__restrict__ Fface, double *__restrict__ cface, int ntx,
                     int nty) {
  using T = FaceTile<DIR>;
  using X = TmaTile<RECON, DIR>;
  constexpr uint32_t BYTES = (uint32_t)(N * X::EZ * sizeof(double));
  extern __shared__ __align__(128) unsigned char tma_smem[];
  __shared__ uint64_t bar;
  double *buf = (double *)tma_smem;
  const unsigned tl = blockIdx.x, nx = (unsigned)ntx, ny = (unsigned)nty;  // (the tile count fits 32 bits)
  const int tx = (int)(tl % nx), ty = (int)((tl / nx) % ny), tz = (int)(tl / (nx * ny));
  const int fi = gv.ngd[0] + tx * T::T0, fj = gv.ngd[1] + ty * T::T1, fk = gv.ngd[2] + gv.koff + tz * T::T2;
  if (threadIdx.x == 0) {
    mbar_init(&bar, 1);
    mbar_init_fence();
    mbar_expect_tx(&bar, BYTES);
    tma_load_4d(buf, &tmap, &bar, (fi - (DIR == 0 ? X::LO : 0)) & ~1, fj - (DIR == 1 ? X::LO : 0),
                fk - (DIR == 2 ? X::LO : 0), 0);
  }
  __syncthreads();
  const int xshift = (gv.ngd[0] - (DIR == 0 ? X::LO : 0)) & 1;  // tile origins advance by an even T0
  const int t0 = (int)threadIdx.x % T::T0, t1 = ((int)threadIdx.x / T::T0) % T::T1,
            t2 = (int)threadIdx.x / (T::T0 * T::T1);
  mbar_wait(&bar, 0);
  const int i = fi + t0, j = fj + t1, k = fk + t2;
  if (i < gv.ngd[0] + gv.n[0] && j < gv.ngd[1] + gv.n[1] && k < gv.ngd[2] + gv.koff + gv.n[2]) {
    const long long z = zone_index(gv, i, j, k);
    SpecArith ar;
    double F[N], c;
    const TileStencil<X::EZ, X::MS> st{buf + (t2 * X::E1 + t1) * X::E0 + t0 + xshift};
    face_compute<N, RECON, G, DIR>(ar, gv, st, i, j, F, c);
    if (ar.good()) {
#pragma unroll
      for (int v = 0; v < N; v++) Fface[v * gv.zg + z] = F[v];
      cface[z] = c;
    } else {
      face_replay<N, RECON, G, DIR>(gv, PE, z, i, j, Fface, cface);
    }
  }
}

// Faces of direction DIR in a box of padded coordinates [lo, lo + cnt): one thread per face, stencil read directly
// from the grid array.  Used for what the tiles do not cover: the upper boundary faces (face index n along DIR),
// and with flux-CT the faces one zone into the transverse ghost layers.
struct FaceBox {
  int lo[3], cnt[3];
};
template <int N, int RECON, class G, int DIR>
__global__ void __launch_bounds__(FB, G::flat ? FLUX_MINB : FLUX_MINB_GEN)
face_box_kernel(const __grid_constant__ GridView gv, const __grid_constant__ FaceBox bx,
                const double *__restrict__ PE, double *__restrict__ Fface, double *__restrict__ cface) {
  const long long t = (long long)blockIdx.x * FB + threadIdx.x;
  if (t >= (long long)bx.cnt[0] * bx.cnt[1] * bx.cnt[2]) return;
  const int i = bx.lo[0] + (int)(t % bx.cnt[0]);
  const long long r = t / bx.cnt[0];
  const int j = bx.lo[1] + (int)(r % bx.cnt[1]);
  const int k = bx.lo[2] + (int)(r / bx.cnt[1]);
  const long long z = zone_index(gv, i, j, k);
  const long long stride = (DIR == 0) ? 1 : (DIR == 1) ? (long long)gv.sz[0] : (long long)gv.sz[0] * gv.sz[1];
  SpecArith ar;
  double F[N], c;
  const GlobalStencil st{PE + z - (RECON == 1 ? 3 : 2) * stride, stride, gv.zg};
  face_compute<N, RECON, G, DIR>(ar, gv, st, i, j, F, c);
  if (ar.good()) {
#pragma unroll
    for (int v = 0; v < N; v++) Fface[v * gv.zg + z] = F[v];
    cface[z] = c;
  } else {
    face_replay<N, RECON, G, DIR>(gv, PE, z, i, j, Fface, cface);
  }
}

// Flux-CT, face -> edge (PAPER.md 4.2 L327-335; Toth 2000 as in harm): the edge field along direction c is the
// simple average of the four face fluxes that represent it, E_c = [F^a(B^b)(z) + F^a(B^b)(z - e_b) - F^b(B^a)(z)
// - F^b(B^a)(z - e_a)] / 4 with (a, b, c) cyclic; one thread per edge index in [ng, ng + n] of every active
// direction.  Pairs with an inactive direction are left out.
template <int N>
__global__ void __launch_bounds__(256)
emf_kernel(const __grid_constant__ GridView gv, const double *__restrict__ Fface, double *__restrict__ emf) {
  const int c0 = gv.n[0] + (gv.ngd[0] > 0), c1 = gv.n[1] + (gv.ngd[1] > 0), c2 = gv.n[2] + (gv.ngd[2] > 0);
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long long)c0 * c1 * c2) return;
  const int i = gv.ngd[0] + (int)(t % c0);
  const long long r = t / c0;
  const int j = gv.ngd[1] + (int)(r % c1), k = gv.ngd[2] + (int)(r / c1);
  const long long z = zone_index(gv, i, j, k);
  const long long st[3] = {1, (long long)gv.sz[0], (long long)gv.sz[0] * gv.sz[1]};
#pragma unroll
  for (int c = 0; c < 3; c++) {
    const int a = (c + 1) % 3, b = (c + 2) % 3;
    if (gv.ngd[a] == 0 || gv.ngd[b] == 0) continue;
    const double *Fa_Bb = Fface + ((long long)a * N + B1 + b) * gv.zg;
    const double *Fb_Ba = Fface + ((long long)b * N + B1 + a) * gv.zg;
    emf[c * gv.zg + z] = 0.25 * (Fa_Bb[z] + Fa_Bb[z - st[b]] - Fb_Ba[z] - Fb_Ba[z - st[a]]);
  }
}

// Flux-CT, edge -> face: the flux of B^comp (comp = 0..2) through the lower a-face of zone z.  F^a(B^a) = 0,
// F^a(B^b) = [E_c(z) + E_c(z + e_b)] / 2, F^a(B^c) = -[E_b(z) + E_b(z + e_c)] / 2, (a, b, c) cyclic; where the
// edge field does not exist (inactive direction) the Riemann solver's flux stays.
template <int N>
__device__ __forceinline__ double ct_face_flux(const GridView &gv, const double *__restrict__ Fface, int a, int comp,
                                               long long z, const long long (&st)[3]) {
  const int b = (a + 1) % 3, c = (a + 2) % 3;
  if (comp == a) return 0.0;
  if (comp == b) {
    if (gv.ngd[b] == 0) return Fface[((long long)a * N + B1 + comp) * gv.zg + z];
    const double *E = gv.emf + c * gv.zg;
    return 0.5 * (E[z] + E[z + st[b]]);
  }
  if (gv.ngd[c] == 0) return Fface[((long long)a * N + B1 + comp) * gv.zg + z];
  const double *E = gv.emf + b * gv.zg;
  return -(0.5 * (E[z] + E[z + st[c]]));
}

__device__ __forceinline__ void atomic_max_nonneg(unsigned long long *addr, double v) {
  atomicMax(addr, (unsigned long long)__double_as_longlong(v));
}

// Where the face fluxes of a zone come from: fs(a, v, up) = flux of variable v through the lower (up = 0) or upper
// (up = 1) a-face of the zone.
template <int N>
struct GlobalFlux {  // straight from the face-flux arrays
  const double *F;
  long long zg, z, st[3];
  __device__ __forceinline__ double operator()(int a, int v, int up) const {
    return F[((long long)a * N + v) * zg + z + (up ? st[a] : 0)];
  }
};
// from the block's shared-memory tile of T0 x T1 zones (X^1 x X^2): per direction the faces the tile's zones
// touch, (T0+1) x T1, T0 x (T1+1), T0 x T1 x 2
template <int N, int T0, int T1>
struct TileFlux {
  static constexpr int S0 = (T0 + 1) * T1, S1 = T0 * (T1 + 1), S2 = 2 * T0 * T1;
  static constexpr int SIZE = N * (S0 + S1 + S2);
  const double *s;
  int t0, t1;
  __device__ __forceinline__ double operator()(int a, int v, int up) const {
    if (a == 0) return s[v * S0 + t1 * (T0 + 1) + t0 + up];
    if (a == 1) return s[N * S0 + v * S1 + (t1 + up) * T0 + t0];
    return s[N * (S0 + S1) + v * S2 + up * T0 * T1 + t1 * T0 + t0];
  }
};

// Stage constant, EMHD gradient terms and wave-speed figures of padded zone z under arithmetic policy A
template <int N, class G, bool CT, class A, class FS>
__device__ __forceinline__ void stage_const_compute(A &ar, const GridView &gv, const FS &fs,
                                                    const double (&Pn_z)[N], const double (&PE_z)[N],
                                                    const double *__restrict__ PE,
                                                    const double *__restrict__ Pn, double dt_stage,
                                                    const double *__restrict__ Fface,
                                                    const double *__restrict__ cface, bool want_speeds, long long z,
                                                    long long id, double (&Cout)[N], double (&Gout)[3],
                                                    double (&sp_loc)[4]) {
  const double idt = ar.rcp(dt_stage);
  G gc;
  double tau = gv.tau_const;
  if constexpr (!G::flat) load_geom<0>(gv.geomC, gv.n2d, id, gc, tau);

  Pieces sn, sE;
  full_state<N>(ar, gv.m, gc, tau, PE_z, sE.th, sE.v, sE.b, sE.h);
  if (G::flat && Pn == PE) sn = sE;  // first stage: P_n is P_E, same state, same bits (general metric: slower)
  else full_state<N>(ar, gv.m, gc, tau, Pn_z, sn.th, sn.v, sn.b, sn.h);
  double Un[N];
  flux_vector<N>(gc, 0, Pn_z, sn.th, sn.v, sn.b, sn.h, Un);

  // flux divergence (eq 10) and wave-speed figures (C-15)
  double divF[N];
#pragma unroll
  for (int v = 0; v < N; v++) divF[v] = 0.0;
  double ssum = 0.0;
  const long long strides[3] = {1, (long long)gv.sz[0], (long long)gv.sz[0] * gv.sz[1]};
#pragma unroll
  for (int a = 0; a < 3; a++) {
    if (gv.ngd[a] == 0) continue;
    const double *ca = cface + (long long)a * gv.zg;
    const long long zu = z + strides[a];
#pragma unroll
    for (int v = 0; v < N; v++) {
      if (CT && v >= B1 && v <= B3) {  // flux-CT: the B-field fluxes are the edge averages
        const double fu = ct_face_flux<N>(gv, Fface, a, v - B1, zu, strides);
        const double fl = ct_face_flux<N>(gv, Fface, a, v - B1, z, strides);
        divF[v] = divF[v] + (fu - fl) * gv.idx[a];
      } else {
        divF[v] = divF[v] + (fs(a, v, 1) - fs(a, v, 0)) * gv.idx[a];
      }
    }
    if (want_speeds) {  // only the dt probe needs them (C-15)
      const double cz = fmax(ca[z], ca[zu]) * gv.idx[a];
      sp_loc[a] = cz;
      ssum = ssum + cz;
    }
  }
  sp_loc[3] = ssum;

  // the zone's connection coefficients, one batch of independent loads; the three contractions below read them
  // from registers (they were 3 x 64 loads feeding serial sums)
  double cn[G::flat ? 1 : CONN_NCOMP];
  if constexpr (!G::flat) {
#pragma unroll
    for (int l = 0; l < 4; l++)
#pragma unroll
      for (int m = 0; m < 4; m++)
#pragma unroll
        for (int n = m; n < 4; n++) {  // Gamma^l_{mn} = Gamma^l_{nm}: the tables hold both, 40 loads serve 64
          const double c = __ldg(gv.conn + (l * 16 + m * 4 + n) * gv.n2d + id);
          cn[l * 16 + m * 4 + n] = c;
          cn[l * 16 + n * 4 + m] = c;
        }
  }

  // explicit geometric source sqrt(-g) T^k_l Gamma^l_{nu k} at P_E (eq 31; C-5)
  double SE[4] = {0.0, 0.0, 0.0, 0.0};
  if constexpr (!G::flat) {
    double T[4][4];
    double q = 0.0, dP = 0.0;
    if constexpr (N == 10) { q = PE_z[QQ]; dP = PE_z[DPP]; }
#pragma unroll
    for (int mu = 0; mu < 4; mu++) stress_row<N>(mu, PE_z[RHO], PE_z[UU], q, dP, sE.th, sE.v, sE.b, sE.h, T[mu]);
#pragma unroll
    for (int nu = 0; nu < 4; nu++) {
      double s = 0.0;
#pragma unroll
      for (int kk = 0; kk < 4; kk++)
#pragma unroll
        for (int l = 0; l < 4; l++) s = s + T[kk][l] * cn[l * 16 + nu * 4 + kk];
      SE[nu] = gc.sqrtmg() * s;
    }
  }
#pragma unroll
  for (int v = 0; v < N; v++) {
    double c = -Un[v] * idt + divF[v];
    if constexpr (!G::flat) {
      if (v >= 1 && v <= 4) c = c - SE[v - 1];
    }
    Cout[v] = c;
  }

  // spatial-gradient parts of the EMHD sources: limited 3-point slopes of derived quantities (L115; O-8)
  if constexpr (N == 10) {
    double dTheta[4] = {0.0, 0.0, 0.0, 0.0};
    double ducov[4][4];
#pragma unroll
    for (int a = 0; a < 4; a++)
#pragma unroll
      for (int b = 0; b < 4; b++) ducov[a][b] = 0.0;
    double divx = 0.0;
    const double th = gv.theta;
#pragma unroll
    for (int a = 0; a < 3; a++) {
      if (gv.ngd[a] == 0) continue;
      const long long zm = z - strides[a], zp = z + strides[a];
      double Pm_[N], Pp_[N];
#pragma unroll
      for (int v = 0; v < N; v++) {
        Pm_[v] = PE[v * gv.zg + zm];
        Pp_[v] = PE[v * gv.zg + zp];
      }
      G gm, gp;
      double taum = tau, taup = tau;
      double sgm = 1.0, sgp = 1.0, sgc = 1.0;
      if constexpr (!G::flat) {
        const long long idm = (a == 0) ? id - 1 : (a == 1) ? id - gv.sz[0] : id;
        const long long idp = (a == 0) ? id + 1 : (a == 1) ? id + gv.sz[0] : id;
        load_geom<0>(gv.geomC, gv.n2d, idm, gm, taum);
        load_geom<0>(gv.geomC, gv.n2d, idp, gp, taup);
        sgm = gm.sg; sgp = gp.sg; sgc = gc.sg;
      }
      Vel vm_, vp_;
      vel_state(ar, gm, Pm_[U1], Pm_[U2], Pm_[U3], vm_);
      vel_state(ar, gp, Pp_[U1], Pp_[U2], Pp_[U3], vp_);
      const double Thm = ar.div(gv.m.gm1 * Pm_[UU], Pm_[RHO]);
      const double Thp = ar.div(gv.m.gm1 * Pp_[UU], Pp_[RHO]);
      dTheta[a + 1] = limited_slope(th, Thm, sE.th.Th, Thp) * gv.idx[a];
#pragma unroll
      for (int nu = 0; nu < 4; nu++)
        ducov[a + 1][nu] = limited_slope(th, vm_.ucov[nu], sE.v.ucov[nu], vp_.ucov[nu]) * gv.idx[a];
      if constexpr (G::flat) {
        divx = divx + limited_slope(th, vm_.ucon[a + 1], sE.v.ucon[a + 1], vp_.ucon[a + 1]) * gv.idx[a];
      } else {
        divx = divx + limited_slope(th, sgm * vm_.ucon[a + 1], sgc * sE.v.ucon[a + 1], sgp * vp_.ucon[a + 1]) *
                          gv.idx[a];
      }
    }
    if constexpr (!G::flat) divx = ar.div_z(divx, gc.sqrtmg());
    // Xq = bhat^i d_i Theta + Theta bhat^mu (u^i d_i u_mu - Gamma^l_{nu mu} u^nu u_l)
    // Xd = bhat^i bhat^nu d_i u_nu - Gamma^l_{mu nu} bhat^mu bhat^nu u_l
    const double *bh = sE.h.con;
    const double *ucon = sE.v.ucon, *ucov = sE.v.ucov;
    double bgradTh = bh[1] * dTheta[1];
    bgradTh = bgradTh + bh[2] * dTheta[2];
    bgradTh = bgradTh + bh[3] * dTheta[3];
    double ba = 0.0;
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
      double acc = ucon[1] * ducov[1][mu];
      acc = acc + ucon[2] * ducov[2][mu];
      acc = acc + ucon[3] * ducov[3][mu];
      if constexpr (!G::flat) {
        double gam = 0.0;
#pragma unroll
        for (int nu = 0; nu < 4; nu++)
#pragma unroll
          for (int l = 0; l < 4; l++)
            gam = gam + cn[l * 16 + nu * 4 + mu] * ucon[nu] * ucov[l];
        acc = acc - gam;
      }
      ba = ba + bh[mu] * acc;
    }
    double bbdu = 0.0;
#pragma unroll
    for (int ii = 1; ii < 4; ii++) {
      double s = bh[0] * ducov[ii][0];
      s = s + bh[1] * ducov[ii][1];
      s = s + bh[2] * ducov[ii][2];
      s = s + bh[3] * ducov[ii][3];
      bbdu = bbdu + bh[ii] * s;
    }
    double Xd = bbdu;
    if constexpr (!G::flat) {
      double gbb = 0.0;
#pragma unroll
      for (int mu = 0; mu < 4; mu++)
#pragma unroll
        for (int nu = 0; nu < 4; nu++)
#pragma unroll
          for (int l = 0; l < 4; l++)
            gbb = gbb + cn[l * 16 + mu * 4 + nu] * bh[mu] * bh[nu] * ucov[l];
      Xd = bbdu - gbb;
    }
    Gout[0] = bgradTh + sE.th.Th * ba;
    Gout[1] = Xd;
    Gout[2] = divx;
  }
}

template <int N, class G, bool CT>
__device__ __noinline__ void stage_const_replay(const GridView &gv, const double *__restrict__ PE,
                                                const double *__restrict__ Pn, double dt_stage,
                                                const double *__restrict__ Fface, const double *__restrict__ cface,
                                                bool want_speeds, long long z, long long id, double *Cout,
                                                double *Gout, double *sp_loc) {
  ExactArith ar;
  double C_[N], G_[3] = {0.0, 0.0, 0.0}, s_[4] = {0.0, 0.0, 0.0, 0.0};
  const GlobalFlux<N> fs{Fface, gv.zg, z, {1, (long long)gv.sz[0], (long long)gv.sz[0] * gv.sz[1]}};
  double Pn_z[N], PE_z[N];
  for (int v = 0; v < N; v++) {
    Pn_z[v] = Pn[v * gv.zg + z];
    PE_z[v] = PE[v * gv.zg + z];
  }
  stage_const_compute<N, G, CT>(ar, gv, fs, Pn_z, PE_z, PE, Pn, dt_stage, Fface, cface, want_speeds, z, id, C_, G_, s_);
  for (int v = 0; v < N; v++) Cout[v] = C_[v];
  for (int v = 0; v < 3; v++) Gout[v] = G_[v];
  for (int v = 0; v < 4; v++) sp_loc[v] = s_[v];
}

// resident blocks per SM of the stage-constant kernels; general metric: connection contractions and 6 neighbour
// geometries need 255 registers -> 2
static constexpr int SC_MINB = 4, SC_MINB_GEN = 2;
template <int N, class G, bool CT>
__global__ void __launch_bounds__(FB, G::flat ? SC_MINB : SC_MINB_GEN)
stage_const_kernel(const __grid_constant__ GridView gv, const double *__restrict__ PE,
                   const double *__restrict__ Pn, double dt_stage, const double *__restrict__ Fface,
                   const double *__restrict__ cface, double *__restrict__ C, double *__restrict__ Gx,
                   Counters *cnt) {
  const long long t = (long long)blockIdx.x * FB + threadIdx.x;
  double sp_loc[4] = {0.0, 0.0, 0.0, 0.0};
  if (t < gv.nint) {
    int i, j, k;
    zone_coords(gv, t, i, j, k);
    const long long z = zone_index(gv, i, j, k);
    const long long id = (long long)j * gv.sz[0] + i;
    double Cout[N], Gout[3] = {0.0, 0.0, 0.0};
    SpecArith ar;
    const GlobalFlux<N> fs{Fface, gv.zg, z, {1, (long long)gv.sz[0], (long long)gv.sz[0] * gv.sz[1]}};
    double Pn_z[N], PE_z[N];
#pragma unroll
    for (int v = 0; v < N; v++) {
      Pn_z[v] = Pn[v * gv.zg + z];
      PE_z[v] = PE[v * gv.zg + z];
    }
    stage_const_compute<N, G, CT>(ar, gv, fs, Pn_z, PE_z, PE, Pn, dt_stage, Fface, cface, cnt != nullptr, z, id, Cout,
                                  Gout, sp_loc);
    if (!ar.good())
      stage_const_replay<N, G, CT>(gv, PE, Pn, dt_stage, Fface, cface, cnt != nullptr, z, id, Cout, Gout, sp_loc);
#pragma unroll
    for (int v = 0; v < N; v++) C[v * gv.zg + z] = Cout[v];
    if constexpr (N == 10) {
#pragma unroll
      for (int v = 0; v < 3; v++) Gx[v * gv.zg + z] = Gout[v];
    }
  }
  // block max of the wave-speed figures -> global atomic max
  if (cnt) {
#pragma unroll
    for (int a = 0; a < 4; a++) {
      double v = sp_loc[a];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
      if ((threadIdx.x & 31) == 0 && v > 0.0) atomic_max_nonneg(&cnt->speeds[a], v);
    }
  }
}

// The same on block tiles of 32 x 4 zones (X^1 x X^2) at one X^3 index: the 6N face fluxes of a zone come from a
// shared-memory tile that the block fills with one batch of independent coalesced loads, instead of 6N loads per
// thread consumed by a serial sum.  Used for Minkowski grids with X^2 active (2.40 -> 2.28 ms at 256^3); the untiled
// kernel serves 1-D grids, general metrics and the dt probe (which also reduces the face speeds).
template <int N, class G, bool CT>
__global__ void __launch_bounds__(FB, G::flat ? SC_MINB : SC_MINB_GEN)
stage_const_tiled_kernel(const __grid_constant__ GridView gv, const double *__restrict__ PE,
                         const double *__restrict__ Pn, double dt_stage, const double *__restrict__ Fface,
                         const double *__restrict__ cface, double *__restrict__ C, double *__restrict__ Gx) {
  constexpr int T0 = 32, T1 = 4;
  using TF = TileFlux<N, T0, T1>;
  __shared__ double tile[TF::SIZE];
  const int i0 = gv.ngd[0] + (int)blockIdx.x * T0, j0 = gv.ngd[1] + (int)blockIdx.y * T1,
            k = gv.ngd[2] + gv.koff + (int)blockIdx.z;
  const long long zg = gv.zg;
  // the zone's own primitives are requested first, so that they arrive while the tile is being staged
  const int t0 = (int)threadIdx.x % T0, t1 = (int)threadIdx.x / T0;
  const int i = i0 + t0, j = j0 + t1;
  const bool valid = i < gv.ngd[0] + gv.n[0] && j < gv.ngd[1] + gv.n[1];
  const long long z = zone_index(gv, valid ? i : gv.ngd[0], valid ? j : gv.ngd[1], k);
  double Pn_z[N], PE_z[N];
#pragma unroll
  for (int v = 0; v < N; v++) {
    Pn_z[v] = Pn[v * zg + z];
    PE_z[v] = PE[v * zg + z];
  }
  // direction 0: faces (i0 .. i0+T0, j0 .. j0+T1-1); direction 1: (i0 .. i0+T0-1, j0 .. j0+T1);
  // direction 2: (i0 .. , j0 .. ) at k and k+1.  Coordinates beyond the padded array are skipped (their zones are not
  // computed either).
  for (int e = (int)threadIdx.x; e < TF::S0; e += FB) {
    const int ci = i0 + e % (T0 + 1), cj = j0 + e / (T0 + 1);
    if (ci < gv.sz[0] && cj < gv.sz[1]) {
      const double *src = Fface + zone_index(gv, ci, cj, k);
#pragma unroll
      for (int v = 0; v < N; v++) tile[v * TF::S0 + e] = src[v * zg];
    }
  }
  for (int e = (int)threadIdx.x; e < TF::S1; e += FB) {
    const int ci = i0 + e % T0, cj = j0 + e / T0;
    if (ci < gv.sz[0] && cj < gv.sz[1]) {
      const double *src = Fface + (long long)N * zg + zone_index(gv, ci, cj, k);
#pragma unroll
      for (int v = 0; v < N; v++) tile[N * TF::S0 + v * TF::S1 + e] = src[v * zg];
    }
  }
  if (gv.ngd[2] > 0) {
    for (int e = (int)threadIdx.x; e < TF::S2; e += FB) {
      const int up = e / (T0 * T1), r = e % (T0 * T1);
      const int ci = i0 + r % T0, cj = j0 + r / T0;
      if (ci < gv.sz[0] && cj < gv.sz[1]) {
        const double *src = Fface + 2LL * N * zg + zone_index(gv, ci, cj, k + up);
#pragma unroll
        for (int v = 0; v < N; v++) tile[N * (TF::S0 + TF::S1) + v * TF::S2 + e] = src[v * zg];
      }
    }
  }
  __syncthreads();
  if (!valid) return;
  const long long id = (long long)j * gv.sz[0] + i;
  double Cout[N], Gout[3] = {0.0, 0.0, 0.0}, sp_loc[4];
  SpecArith ar;
  const TF fs{tile, t0, t1};
  stage_const_compute<N, G, CT>(ar, gv, fs, Pn_z, PE_z, PE, Pn, dt_stage, Fface, cface, false, z, id, Cout, Gout,
                                sp_loc);
  if (!ar.good()) stage_const_replay<N, G, CT>(gv, PE, Pn, dt_stage, Fface, cface, false, z, id, Cout, Gout, sp_loc);
#pragma unroll
  for (int v = 0; v < N; v++) C[v * zg + z] = Cout[v];
  if constexpr (N == 10) {
#pragma unroll
    for (int v = 0; v < 3; v++) Gx[v * zg + z] = Gout[v];
  }
}

// The tiled stage-constant kernel with its three face-flux tiles brought in by TMA (one 4-D box per direction, all N
// variables): rows of W = T0 + 2 faces starting at the even X^1 index at or below the tile's first face.
template <int N, int T0, int T1>
struct TileFluxTma {
  static constexpr int W = T0 + 2;
  static constexpr int S0 = W * T1, S1 = W * (T1 + 1), S2 = 2 * W * T1;
  // offsets of the three boxes in doubles, each on a 128-byte boundary (TMA destination)
  static constexpr int O1 = (N * S0 + 15) / 16 * 16, O2 = (O1 + N * S1 + 15) / 16 * 16;
  static constexpr int SIZE = O2 + N * S2;
  const double *s;
  int t0, t1;  // t0 includes the shift of the box start
  __device__ __forceinline__ double operator()(int a, int v, int up) const {
    if (a == 0) return s[v * S0 + t1 * W + t0 + up];
    if (a == 1) return s[O1 + v * S1 + (t1 + up) * W + t0];
    return s[O2 + v * S2 + up * W * T1 + t1 * W + t0];
  }
};

struct FluxMaps {
  CUtensorMap m[3];
};

template <int N, class G, bool CT>
__global__ void __launch_bounds__(FB, G::flat ? SC_MINB : SC_MINB_GEN)
stage_const_tma_kernel(const __grid_constant__ GridView gv, const __grid_constant__ FluxMaps maps,
                       const double *__restrict__ PE, const double *__restrict__ Pn, double dt_stage,
                       const double *__restrict__ Fface, const double *__restrict__ cface, double *__restrict__ C,
                       double *__restrict__ Gx) {
  constexpr int T0 = 32, T1 = 4;
  using TF = TileFluxTma<N, T0, T1>;
  extern __shared__ __align__(128) unsigned char sc_smem[];
  __shared__ uint64_t bar;
  double *tile = (double *)sc_smem;
  const int i0 = gv.ngd[0] + (int)blockIdx.x * T0, j0 = gv.ngd[1] + (int)blockIdx.y * T1,
            k = gv.ngd[2] + gv.koff + (int)blockIdx.z;
  const long long zg = gv.zg;
  if (threadIdx.x == 0) {
    mbar_init(&bar, 1);
    mbar_init_fence();
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    const bool d3 = gv.ngd[2] > 0;
    mbar_expect_tx(&bar, (uint32_t)(N * (TF::S0 + TF::S1 + (d3 ? TF::S2 : 0)) * sizeof(double)));
    tma_load_4d(tile, &maps.m[0], &bar, i0 & ~1, j0, k, 0);
    tma_load_4d(tile + TF::O1, &maps.m[1], &bar, i0 & ~1, j0, k, 0);
    if (d3) tma_load_4d(tile + TF::O2, &maps.m[2], &bar, i0 & ~1, j0, k, 0);
  }
  // the zone's own primitives are requested while the tiles are in flight
  const int t0 = (int)threadIdx.x % T0, t1 = (int)threadIdx.x / T0;
  const int i = i0 + t0, j = j0 + t1;
  const bool valid = i < gv.ngd[0] + gv.n[0] && j < gv.ngd[1] + gv.n[1];
  const long long z = zone_index(gv, valid ? i : gv.ngd[0], valid ? j : gv.ngd[1], k);
  double Pn_z[N], PE_z[N];
#pragma unroll
  for (int v = 0; v < N; v++) {
    Pn_z[v] = Pn[v * zg + z];
    PE_z[v] = PE[v * zg + z];
  }
  mbar_wait(&bar, 0);
  if (!valid) return;
  const long long id = (long long)j * gv.sz[0] + i;
  double Cout[N], Gout[3] = {0.0, 0.0, 0.0}, sp_loc[4];
  SpecArith ar;
  const TF fs{tile, t0 + (i0 & 1), t1};
  stage_const_compute<N, G, CT>(ar, gv, fs, Pn_z, PE_z, PE, Pn, dt_stage, Fface, cface, false, z, id, Cout, Gout,
                                sp_loc);
  if (!ar.good()) stage_const_replay<N, G, CT>(gv, PE, Pn, dt_stage, Fface, cface, false, z, id, Cout, Gout, sp_loc);
#pragma unroll
  for (int v = 0; v < N; v++) C[v * zg + z] = Cout[v];
  if constexpr (N == 10) {
#pragma unroll
    for (int v = 0; v < 3; v++) Gx[v * zg + z] = Gout[v];
  }
}

// max over interior zones of c^d/dX^d (d = 1..3) and of their sum (C-15), from the face speeds: the same expressions,
// in the same order, as the wave-speed figures of stage_const_compute
__global__ void __launch_bounds__(256)
speeds_kernel(const __grid_constant__ GridView gv, const double *__restrict__ cface, Counters *cnt) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  double sp_loc[4] = {0.0, 0.0, 0.0, 0.0};
  if (t < gv.nint) {
    int i, j, k;
    zone_coords(gv, t, i, j, k);
    const long long z = zone_index(gv, i, j, k);
    const long long strides[3] = {1, (long long)gv.sz[0], (long long)gv.sz[0] * gv.sz[1]};
    double ssum = 0.0;
#pragma unroll
    for (int a = 0; a < 3; a++) {
      if (gv.ngd[a] == 0) continue;
      const double *ca = cface + (long long)a * gv.zg;
      const double cz = fmax(ca[z], ca[z + strides[a]]) * gv.idx[a];
      sp_loc[a] = cz;
      ssum = ssum + cz;
    }
    sp_loc[3] = ssum;
  }
  // warp maxima -> block maxima in shared memory -> one atomic per figure and block
  __shared__ double red[4][8];
#pragma unroll
  for (int a = 0; a < 4; a++) {
    double v = sp_loc[a];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if ((threadIdx.x & 31) == 0) red[a][threadIdx.x >> 5] = v;
  }
  __syncthreads();
  if (threadIdx.x < 4) {
    double v = red[threadIdx.x][0];
#pragma unroll
    for (int w = 1; w < 8; w++) v = fmax(v, red[threadIdx.x][w]);
    if (v > 0.0) atomic_max_nonneg(&cnt->speeds[threadIdx.x], v);
  }
}

int launch_speeds(const GridView &gv, const double *cface, Counters *cnt, cudaStream_t s) {
  speeds_kernel<<<(unsigned)((gv.nint + 255) / 256), 256, 0, s>>>(gv, cface, cnt);
  return 1;
}

// what: bit 0 = the face fluxes (a1, a2), bit 1 = the stage constant and gradient terms (a3)
template <int N, int RECON, class G>
static int launch_fluxes_t(const GridView &gv, const double *PE, const double *Pn, double dt_stage, double *C,
                           double *Gx, double *Fface, double *cface, Counters *cnt, cudaStream_t s, int what) {
  int launches = 0;
  for (int a = 0; a < 3; a++) {
    if (gv.ngd[a] == 0 || !(what & 1)) continue;
    const int f0 = gv.n[0], f1 = gv.n[1], f2 = gv.n[2];  // tiled faces per direction (+ one edge plane along a)
    double *Fa = Fface + (long long)a * N * gv.zg;
    double *ca = cface + (long long)a * gv.zg;
    auto tiles = [&](int t0, int t1, int t2) {
      return dim3((unsigned)((f0 + t0 - 1) / t0), (unsigned)((f1 + t1 - 1) / t1), (unsigned)((f2 + t2 - 1) / t2));
    };
    bool by_tma = false;   // false: no tensor map for this array (odd X^1 extent: rows not 16-byte aligned) -> staging kernels
    {
      auto tma = [&](auto dirc) {
        constexpr int D = decltype(dirc)::value;
        using X = TmaTile<RECON, D>;
        using T = FaceTile<D>;
        CUtensorMap map;
        if (!make_tile_map(&map, PE, gv.sz[0], gv.sz[1], gv.sz[2], N, gv.zg, X::E0, X::E1, X::E2)) return false;
        const dim3 tg = tiles(T::T0, T::T1, T::T2);
        const long long nt = (long long)tg.x * tg.y * tg.z;
        const size_t smem = tma_tile_bytes<N, RECON, D>();
        auto kern = face_flux_tma_kernel<N, RECON, G, D>;
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (nt >= (1LL << 31)) return false;
        kern<<<(unsigned)nt, FB, smem, s>>>(gv, map, PE, Fa, ca, (int)tg.x, (int)tg.y);
        return true;
      };
      if (a == 0) by_tma = tma(std::integral_constant<int, 0>());
      if (a == 1) by_tma = tma(std::integral_constant<int, 1>());
      if (a == 2) by_tma = tma(std::integral_constant<int, 2>());
    }
    if (!by_tma) {
      if (a == 0) face_flux_kernel<N, RECON, G, 0><<<tiles(128, 1, 1), FB, 0, s>>>(gv, PE, Fa, ca);
      if (a == 1) face_flux_kernel<N, RECON, G, 1><<<tiles(32, 4, 1), FB, 0, s>>>(gv, PE, Fa, ca);
      if (a == 2) face_flux_kernel<N, RECON, G, 2><<<tiles(32, 1, 4), FB, 0, s>>>(gv, PE, Fa, ca);
    }
    // what the tiles leave: the upper boundary plane along a, and with flux-CT one layer of faces in every active
    // transverse ghost direction (the edge averages reach there)
    auto box = [&](const FaceBox &bx) {
      const long long nf = (long long)bx.cnt[0] * bx.cnt[1] * bx.cnt[2];
      if (nf <= 0) return;
      const unsigned nb = (unsigned)((nf + FB - 1) / FB);
      if (a == 0) face_box_kernel<N, RECON, G, 0><<<nb, FB, 0, s>>>(gv, bx, PE, Fa, ca);
      if (a == 1) face_box_kernel<N, RECON, G, 1><<<nb, FB, 0, s>>>(gv, bx, PE, Fa, ca);
      if (a == 2) face_box_kernel<N, RECON, G, 2><<<nb, FB, 0, s>>>(gv, bx, PE, Fa, ca);
      launches++;
    };
    const int ext = gv.flux_ct ? 1 : 0;
    FaceBox edge;
    for (int d = 0; d < 3; d++) {
      const int e = (d != a && gv.ngd[d] > 0) ? ext : 0;
      edge.lo[d] = gv.ngd[d] - e;
      edge.cnt[d] = gv.n[d] + 2 * e;
    }
    edge.lo[a] = gv.ngd[a] + gv.n[a];
    edge.cnt[a] = 1;
    edge.lo[2] += gv.koff;  // launches over a range of X^3 planes (flux-CT fringes are not offered there)
    box(edge);
    if (ext) {
      bool first = true;  // the first transverse direction takes the corners shared with the second
      for (int b = 0; b < 3; b++) {
        if (b == a || gv.ngd[b] == 0) continue;
        for (int side = 0; side < 2; side++) {
          FaceBox fr;
          for (int d = 0; d < 3; d++) {
            const int e = (d != a && d != b && gv.ngd[d] > 0 && first) ? 1 : 0;
            fr.lo[d] = gv.ngd[d] - e;
            fr.cnt[d] = gv.n[d] + 2 * e;
          }
          fr.lo[b] = side ? gv.ngd[b] + gv.n[b] : gv.ngd[b] - 1;
          fr.cnt[b] = 1;
          box(fr);
        }
        first = false;
      }
    }
    launches++;
  }
  if (gv.flux_ct && (what & 1)) {
    const long long ne = (long long)(gv.n[0] + (gv.ngd[0] > 0)) * (gv.n[1] + (gv.ngd[1] > 0)) * (gv.n[2] + (gv.ngd[2] > 0));
    emf_kernel<N><<<(unsigned)((ne + 255) / 256), 256, 0, s>>>(gv, Fface, gv.emf);
    launches++;
  }
  if (!(what & 2)) return launches;
  const unsigned blocks = (unsigned)((gv.nint + FB - 1) / FB);
  if (!cnt && gv.ngd[1] > 0) {
    const dim3 tg((unsigned)((gv.n[0] + 31) / 32), (unsigned)((gv.n[1] + 3) / 4), (unsigned)gv.n[2]);
    bool by_tma = false;
    {
      using TF = TileFluxTma<N, 32, 4>;
      FluxMaps maps;
      bool ok = true;
      const int b1[3] = {4, 5, 4}, b2[3] = {1, 1, 2};
      for (int a = 0; a < 3 && ok; a++) {
        if (gv.ngd[a] == 0) {
          maps.m[a] = maps.m[0];
          continue;
        }
        ok = make_tile_map(&maps.m[a], Fface + (long long)a * N * gv.zg, gv.sz[0], gv.sz[1], gv.sz[2], N, gv.zg, TF::W,
                           b1[a], b2[a]);
      }
      if (ok) {
        const size_t smem = (size_t)TF::SIZE * sizeof(double);
        if (gv.flux_ct) {
          cudaFuncSetAttribute(stage_const_tma_kernel<N, G, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
          stage_const_tma_kernel<N, G, true><<<tg, FB, smem, s>>>(gv, maps, PE, Pn, dt_stage, Fface, cface, C, Gx);
        } else {
          cudaFuncSetAttribute(stage_const_tma_kernel<N, G, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
          stage_const_tma_kernel<N, G, false><<<tg, FB, smem, s>>>(gv, maps, PE, Pn, dt_stage, Fface, cface, C, Gx);
        }
        by_tma = true;
      }
    }
    if (by_tma) {
    } else if (gv.flux_ct) stage_const_tiled_kernel<N, G, true><<<tg, FB, 0, s>>>(gv, PE, Pn, dt_stage, Fface, cface, C, Gx);
    else stage_const_tiled_kernel<N, G, false><<<tg, FB, 0, s>>>(gv, PE, Pn, dt_stage, Fface, cface, C, Gx);
  } else if (gv.flux_ct) {
    stage_const_kernel<N, G, true><<<blocks, FB, 0, s>>>(gv, PE, Pn, dt_stage, Fface, cface, C, Gx, cnt);
  } else {
    stage_const_kernel<N, G, false><<<blocks, FB, 0, s>>>(gv, PE, Pn, dt_stage, Fface, cface, C, Gx, cnt);
  }
  return launches + 1;
}

int launch_fluxes(const GridView &gv, const double *PE, const double *Pn, double dt_stage, double *C, double *G,
                  double *Fface, double *cface, Counters *cnt, cudaStream_t s, int what) {
  const bool flat = (gv.metric == 0);
  const bool mp5 = (gv.recon == 1);
#define GRIM_DISPATCH(NV)                                                                                   \
  if (flat) {                                                                                               \
    return mp5 ? launch_fluxes_t<NV, 1, GeomFlat>(gv, PE, Pn, dt_stage, C, G, Fface, cface, cnt, s, what)   \
               : launch_fluxes_t<NV, 0, GeomFlat>(gv, PE, Pn, dt_stage, C, G, Fface, cface, cnt, s, what);  \
  } else {                                                                                                  \
    return mp5 ? launch_fluxes_t<NV, 1, GeomGen>(gv, PE, Pn, dt_stage, C, G, Fface, cface, cnt, s, what)    \
               : launch_fluxes_t<NV, 0, GeomGen>(gv, PE, Pn, dt_stage, C, G, Fface, cface, cnt, s, what);   \
  }
  if (gv.nvar == 10) { GRIM_DISPATCH(10) }
  GRIM_DISPATCH(8)
#undef GRIM_DISPATCH
}

}  // namespace grim
