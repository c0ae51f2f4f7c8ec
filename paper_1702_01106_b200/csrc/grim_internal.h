// grim_internal.h -- host/device shared declarations of the library (not part of the ABI).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "physics.cuh"
#include "newton.cuh"

namespace grim {

// geometry tables: SoA [component][idx2d], idx2d = j*s1 + i over the padded 2-D (X^1, X^2) plane
enum {
  GT_GCOV = 0,    // 10 components, sym4 order
  GT_GCON = 10,   // 10 components
  GT_SQRTMG = 20,
  GT_ALPHA = 21,
  GT_TAU = 22,
  GT_BFAC = 23,   // 3 components: alpha * g^{t i}
  GT_NCOMP = 26
};
enum { CONN_NCOMP = 64 };  // Gamma^l_{mn} at [l*16 + m*4 + n]

struct GridView {
  int n[3], ngd[3], sz[3];
  int dim, nvar, recon, metric, riemann;
  long long zg, n2d, nint;   // padded zones, padded 2-D zones, interior zones
  double dx[3], idx[3];
  double xstart[3];
  double theta;
  ModelParams m;
  double tau_const;
  SolverParams sp;
  const double *geomC;       // GT_NCOMP * n2d
  const double *geomF[3];    // lower faces
  const double *conn;        // CONN_NCOMP * n2d
  int flux_ct;               // flux-CT averaging of the B-field fluxes
  int reduced;               // reduced solve: B^i explicit, Newton on the other N - 3 primitives
  double *emf;               // 3 * zg edge fields (flux_ct only)
  int nsm;                   // multiprocessors of the device
  int koff;                  // launches over a range of X^3 planes (pipelined host path): the interior zones are
                             // those of planes [koff, koff + n[2]) of the grid; sz, zg, n2d keep the full extents
};

// per-call device counters
struct Counters {
  unsigned long long n_active;     // zones left without a terminal status
  unsigned long long backtracks;   // rejected line-search trials
  unsigned long long list_count;   // compaction: entries appended to the next active list
  unsigned long long speeds[4];    // max wave-speed figures, non-negative doubles compared as integers
};

struct StatsDev {
  unsigned long long hist[16];
  unsigned long long unconverged;
  unsigned long long max_rel;      // double bits (non-negative)
};

// interior zone t (i fastest) -> padded coordinates and index
__host__ __device__ inline void zone_coords(const GridView &gv, long long t, int &i, int &j, int &k) {
  i = (int)(t % gv.n[0]) + gv.ngd[0];
  long long r = t / gv.n[0];
  j = (int)(r % gv.n[1]) + gv.ngd[1];
  k = (int)(r / gv.n[1]) + gv.ngd[2] + gv.koff;
}
__host__ __device__ inline long long zone_index(const GridView &gv, int i, int j, int k) {
  return ((long long)k * gv.sz[1] + j) * gv.sz[0] + i;
}

#ifdef __CUDACC__
// loads the geometry record of padded 2-D zone id from a table; DIR = 0: centre (no g^.. entries), 1..3: face
template <int DIR>
__device__ __forceinline__ void load_geom(const double *__restrict__ tab, long long n2d, long long id, GeomGen &g,
                                          double &tau) {
#pragma unroll
  for (int c = 0; c < 10; c++) g.g[c] = tab[(GT_GCOV + c) * n2d + id];
#pragma unroll
  for (int c = 0; c < 3; c++) g.bfac[c] = tab[(GT_BFAC + c) * n2d + id];
  g.alpha = tab[GT_ALPHA * n2d + id];
  g.sg = tab[GT_SQRTMG * n2d + id];
  tau = tab[GT_TAU * n2d + id];
  if constexpr (DIR > 0) {
    g.gcon00 = tab[(GT_GCON + sym4(0, 0)) * n2d + id];
    g.gcon0d = tab[(GT_GCON + sym4(0, DIR)) * n2d + id];
    g.gcondd = tab[(GT_GCON + sym4(DIR, DIR)) * n2d + id];
  } else {
    g.gcon00 = g.gcon0d = g.gcondd = 0.0;
  }
}
#endif

// ---- kernel launchers (defined in the kernels_*.cu files); all enqueue on `s` and return the launch count ----
int launch_newton_stage(const GridView &gv, const double *Pn, const double *PE, const double *C, const double *G,
                        const double *Pguess, int fresh, double dt_stage, int max_iters, double *Piter, double *resnorm, int32_t *status,
                        int32_t *iters, Counters *cnt, cudaStream_t s, const long long *list = nullptr,
                        long long nlist = 0, long long *next_list = nullptr);
int launch_invert(const GridView &gv, long long nz, long long nlist, const long long *list, const double *Ustar,
                  const double *geom, double *P, int32_t *iters, int32_t *status, double *resnorm, int max_iters, int first,
                  long long *next_list, Counters *cnt, cudaStream_t s);
int launch_prim_to_conserved(const GridView &gv, long long nz, const double *P, double *U, cudaStream_t s);
// what: bit 0 = face fluxes and speeds (a1, a2), bit 1 = stage constant and gradient terms (a3) from the face arrays
int launch_fluxes(const GridView &gv, const double *PE, const double *Pn, double dt_stage, double *C, double *G,
                  double *Fface, double *cface, Counters *cnt, cudaStream_t s, int what = 3);
int launch_speeds(const GridView &gv, const double *cface, Counters *cnt, cudaStream_t s);
// dirs: bit a set = fill the ghosts of direction a; planes [klo, klo + kcnt) of the padded X^3 extent (kcnt < 0: all)
// for the directions other than X^3
int launch_fill_ghosts(const GridView &gv, const int32_t bc[3][2], double *P, cudaStream_t s, int dirs = 7,
                       int klo = 0, int kcnt = -1);
int launch_metric_kerr(const GridView &gv, double a, double h, int tau_mode, double *geomC, double *geomF0,
                       double *geomF1, double *geomF2, double *conn, cudaStream_t s);
int launch_metric_flat(const GridView &gv, double *geomC, double *geomF0, double *geomF1, double *geomF2,
                       double *conn, cudaStream_t s);
int launch_stats(const GridView &gv, const double *Pn, double dt_stage, const double *resnorm,
                 const int32_t *status, const int32_t *iters, StatsDev *out, cudaStream_t s);
int launch_copy_interior(const GridView &gv, const double *src, double *dst, cudaStream_t s);
int launch_arith_selftest(unsigned long long n, unsigned long long seed, int wide, unsigned long long *out,
                          cudaStream_t s);
int launch_fp64_probe(int fma, int iters, double *sink, int blocks, int threads, cudaStream_t s);

}  // namespace grim
