// kernels_misc.cu -- geometry precompute (step a0), ghost fill, per-stage statistics, fp64 pipe probe.
#include "grim_internal.h"
#include "problems.cuh"

namespace grim {

// ---------------------------------------------------------------------------------------------------------
// a0  Geometry (L68-89 eqs 5-8; C-10).  Kerr-Schild (t,r,theta,phi), M = 1, transformed to X^mu by
// g_X = L^T g L, L = diag(1, r, pi(1 + (1-h) cos(2 pi X2)), 1) (eq 8).  Derivatives for the connection are
// exact: the metric function is evaluated on forward-mode dual numbers carrying d/dX1 and d/dX2.
// ---------------------------------------------------------------------------------------------------------
struct Dual {
  double v, d1, d2;
};
__device__ __forceinline__ Dual dmake(double v, double d1 = 0.0, double d2 = 0.0) { return Dual{v, d1, d2}; }
__device__ __forceinline__ Dual operator+(Dual a, Dual b) { return {a.v + b.v, a.d1 + b.d1, a.d2 + b.d2}; }
__device__ __forceinline__ Dual operator-(Dual a, Dual b) { return {a.v - b.v, a.d1 - b.d1, a.d2 - b.d2}; }
__device__ __forceinline__ Dual operator-(Dual a) { return {-a.v, -a.d1, -a.d2}; }
__device__ __forceinline__ Dual operator*(Dual a, Dual b) {
  return {a.v * b.v, a.d1 * b.v + a.v * b.d1, a.d2 * b.v + a.v * b.d2};
}
__device__ __forceinline__ Dual operator*(double s, Dual a) { return {s * a.v, s * a.d1, s * a.d2}; }
__device__ __forceinline__ Dual operator+(double s, Dual a) { return {s + a.v, a.d1, a.d2}; }
__device__ __forceinline__ Dual operator/(Dual a, Dual b) {
  double iv = 1.0 / b.v;
  double q = a.v * iv;
  return {q, (a.d1 - q * b.d1) * iv, (a.d2 - q * b.d2) * iv};
}
__device__ __forceinline__ Dual dexp(Dual a) {
  double e = exp(a.v);
  return {e, e * a.d1, e * a.d2};
}
__device__ __forceinline__ Dual dsin(Dual a) {
  double s = sin(a.v), c = cos(a.v);
  return {s, c * a.d1, c * a.d2};
}
__device__ __forceinline__ Dual dcos(Dual a) {
  double s = sin(a.v), c = cos(a.v);
  return {c, -s * a.d1, -s * a.d2};
}

// covariant metric in X coordinates with its X1, X2 derivatives; returns sqrt(-g) = Sigma sin(theta) |det L|
__device__ void kerr_mks_gcov(double a, double h, double X1, double X2, Dual (&g)[4][4], double &sqrtmg, double &r_out) {
  const double pi = 3.14159265358979323846;
  Dual x1 = dmake(X1, 1.0, 0.0), x2 = dmake(X2, 0.0, 1.0);
  Dual r = dexp(x1);                                                  // eq 5
  Dual th = pi * x2 + (0.5 * (1.0 - h)) * dsin((2.0 * pi) * x2);       // eq 6
  Dual sth = dsin(th), cth = dcos(th);
  if (fabs(sth.v) < 1e-20) sth = dmake(1e-20);  // C-21: faces on the polar axis; keeps g^{mu nu} finite, sqrt(-g) ~ 0
  Dual s2 = sth * sth;
  Dual Sig = r * r + (a * a) * (cth * cth);
  Dual f = (2.0 * r) / Sig;
  Dual L[4] = {dmake(1.0), r, pi * (1.0 + (1.0 - h) * dcos((2.0 * pi) * x2)), dmake(1.0)};  // eq 8
  Dual k[4][4];
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < 4; n++) k[m][n] = dmake(0.0);
  k[0][0] = -(1.0 + (-f));
  k[0][1] = k[1][0] = f;
  k[0][3] = k[3][0] = (-a) * (f * s2);
  k[1][1] = 1.0 + f;
  k[1][3] = k[3][1] = (-a) * (s2 * (1.0 + f));
  k[2][2] = Sig;
  k[3][3] = s2 * (Sig + (a * a) * (s2 * (1.0 + f)));
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < 4; n++) g[m][n] = k[m][n] * L[m] * L[n];
  Dual sg = Sig * sth * L[1] * L[2];
  sqrtmg = fabs(sg.v);
  r_out = r.v;
}

// inverse of a symmetric 4x4 by Gauss-Jordan elimination with partial pivoting
__device__ void invert_4x4(const double (&A)[4][4], double (&inv)[4][4]) {
  double w[4][8];
  for (int i = 0; i < 4; i++)
    for (int j = 0; j < 4; j++) {
      w[i][j] = A[i][j];
      w[i][4 + j] = (i == j) ? 1.0 : 0.0;
    }
  for (int c = 0; c < 4; c++) {
    int p = c;
    for (int rr = c + 1; rr < 4; rr++)
      if (fabs(w[rr][c]) > fabs(w[p][c])) p = rr;
    if (p != c)
      for (int j = 0; j < 8; j++) {
        double t = w[c][j];
        w[c][j] = w[p][j];
        w[p][j] = t;
      }
    const double d = 1.0 / w[c][c];
    for (int j = 0; j < 8; j++) w[c][j] *= d;
    for (int rr = 0; rr < 4; rr++)
      if (rr != c) {
        const double fac = w[rr][c];
        for (int j = 0; j < 8; j++) w[rr][j] -= fac * w[c][j];
      }
  }
  for (int i = 0; i < 4; i++)
    for (int j = 0; j < 4; j++) inv[i][j] = w[i][4 + j];
}

__device__ void store_geom(double *tab, long long n2d, long long id, const double (&gcov)[4][4],
                           const double (&gcon)[4][4], double sqrtmg, double tau) {
  for (int m = 0; m < 4; m++)
    for (int n = m; n < 4; n++) {
      tab[(GT_GCOV + sym4(m, n)) * n2d + id] = gcov[m][n];
      tab[(GT_GCON + sym4(m, n)) * n2d + id] = gcon[m][n];
    }
  const double alpha = 1.0 / sqrt(-gcon[0][0]);
  tab[GT_SQRTMG * n2d + id] = sqrtmg;
  tab[GT_ALPHA * n2d + id] = alpha;
  tab[GT_TAU * n2d + id] = tau;
  for (int i = 1; i < 4; i++) tab[(GT_BFAC + i - 1) * n2d + id] = alpha * gcon[0][i];
}

__global__ void metric_kerr_kernel(GridView gv, double a, double h, int tau_mode, double *geomC, double *geomF0,
                                   double *geomF1, double *geomF2, double *conn) {
  const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= gv.n2d) return;
  const int i = (int)(id % gv.sz[0]), j = (int)(id / gv.sz[0]);
  const double X1 = gv.xstart[0] + (i - gv.ngd[0] + 0.5) * gv.dx[0];
  const double X2 = gv.xstart[1] + (j - gv.ngd[1] + 0.5) * gv.dx[1];
  const double X1f = gv.xstart[0] + (i - gv.ngd[0]) * gv.dx[0];
  const double X2f = gv.xstart[1] + (j - gv.ngd[1]) * gv.dx[1];
  const double Xs[3][2] = {{X1, X2}, {X1f, X2}, {X1, X2f}};
  double *tabs[3] = {geomC, geomF0, geomF1};
  for (int loc = 0; loc < 3; loc++) {
    Dual g[4][4];
    double sqrtmg, r;
    kerr_mks_gcov(a, h, Xs[loc][0], Xs[loc][1], g, sqrtmg, r);
    double gcov[4][4], gcon[4][4];
    for (int m = 0; m < 4; m++)
      for (int n = 0; n < 4; n++) gcov[m][n] = g[m][n].v;
    invert_4x4(gcov, gcon);
    const double tau = (tau_mode == 1) ? r * sqrt(r) : gv.tau_const;  // C-11: tau_R = r^{3/2}
    store_geom(tabs[loc], gv.n2d, id, gcov, gcon, sqrtmg, tau);
    if (loc == 0) {
      store_geom(geomF2, gv.n2d, id, gcov, gcon, sqrtmg, tau);  // metric independent of X3
      // Gamma^l_{mn} = 1/2 g^{lk} (d_m g_{kn} + d_n g_{km} - d_k g_{mn}); d_t = d_X3 = 0
      for (int l = 0; l < 4; l++)
        for (int m = 0; m < 4; m++)
          for (int n = 0; n < 4; n++) {
            double s = 0.0;
            for (int k = 0; k < 4; k++) {
              const double dm = (m == 1) ? g[k][n].d1 : (m == 2) ? g[k][n].d2 : 0.0;
              const double dn = (n == 1) ? g[k][m].d1 : (n == 2) ? g[k][m].d2 : 0.0;
              const double dk = (k == 1) ? g[m][n].d1 : (k == 2) ? g[m][n].d2 : 0.0;
              s += gcon[l][k] * (dm + dn - dk);
            }
            conn[(l * 16 + m * 4 + n) * gv.n2d + id] = 0.5 * s;
          }
    }
  }
}

__global__ void metric_flat_kernel(GridView gv, double *geomC, double *geomF0, double *geomF1, double *geomF2,
                                   double *conn) {
  const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= gv.n2d) return;
  double gcov[4][4], gcon[4][4];
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < 4; n++) gcov[m][n] = gcon[m][n] = (m == n) ? (m == 0 ? -1.0 : 1.0) : 0.0;
  double *tabs[4] = {geomC, geomF0, geomF1, geomF2};
  for (int loc = 0; loc < 4; loc++) store_geom(tabs[loc], gv.n2d, id, gcov, gcon, 1.0, gv.tau_const);
  for (int c = 0; c < CONN_NCOMP; c++) conn[c * gv.n2d + id] = 0.0;
}

int launch_metric_kerr(const GridView &gv, double a, double h, int tau_mode, double *geomC, double *geomF0,
                       double *geomF1, double *geomF2, double *conn, cudaStream_t s) {
  const int tb = 128;
  metric_kerr_kernel<<<(unsigned)((gv.n2d + tb - 1) / tb), tb, 0, s>>>(gv, a, h, tau_mode, geomC, geomF0, geomF1,
                                                                       geomF2, conn);
  return 1;
}
int launch_metric_flat(const GridView &gv, double *geomC, double *geomF0, double *geomF1, double *geomF2,
                       double *conn, cudaStream_t s) {
  const int tb = 128;
  metric_flat_kernel<<<(unsigned)((gv.n2d + tb - 1) / tb), tb, 0, s>>>(gv, geomC, geomF0, geomF1, geomF2, conn);
  return 1;
}

// ---------------------------------------------------------------------------------------------------------
// Ghost fill (C-11): one launch per active direction, in the order 1, 2, 3; each covers the full padded extent
// of the other directions, so that corners end up filled.
// ---------------------------------------------------------------------------------------------------------
template <int DIR>
__global__ void fill_ghosts_kernel(GridView gv, int bc_lo, int bc_hi, double *__restrict__ P, int klo, int kcnt) {
  const int ng = gv.ngd[DIR], n = gv.n[DIR];
  // ghost layer index g in [0, 2 ng): lower side g < ng, upper side g >= ng
  const int e0 = (DIR == 0) ? 2 * ng : gv.sz[0];
  const int e1 = (DIR == 1) ? 2 * ng : gv.sz[1];
  const int e2 = (DIR == 2) ? 2 * ng : kcnt;
  const long long per_var = (long long)e0 * e1 * e2;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= per_var * gv.nvar) return;
  const int v = (int)(t / per_var);
  long long r = t % per_var;
  int c[3];
  c[0] = (int)(r % e0);
  r /= e0;
  c[1] = (int)(r % e1);
  c[2] = (int)(r / e1);
  const int gl = c[DIR];
  if (DIR != 2) c[2] += klo;
  const int side = (gl >= ng) ? 1 : 0;
  const int gz = side ? gl - ng : gl;
  const int bc = side ? bc_hi : bc_lo;
  if (bc == 3) return;  // GRIM_BC_NONE: caller fills
  const int dst = side == 0 ? (ng - 1 - gz) : (ng + n + gz);
  int src;
  if (bc == 0) src = side == 0 ? (ng + n - 1 - gz) : (ng + gz);          // periodic
  else if (bc == 1) src = side == 0 ? ng : (ng + n - 1);                  // outflow: copy the edge zone
  else src = side == 0 ? (ng + gz) : (ng + n - 1 - gz);                   // polar reflection
  int cd[3] = {c[0], c[1], c[2]}, cs[3] = {c[0], c[1], c[2]};
  cd[DIR] = dst;
  cs[DIR] = src;
  double val = P[v * gv.zg + zone_index(gv, cs[0], cs[1], cs[2])];
  if (bc == 2 && (v == U1 + DIR || v == B1 + DIR)) val = -val;
  P[v * gv.zg + zone_index(gv, cd[0], cd[1], cd[2])] = val;
}

int launch_fill_ghosts(const GridView &gv, const int32_t bc[3][2], double *P, cudaStream_t s, int dirs, int klo,
                       int kcnt) {
  int launches = 0;
  const int tb = 256;
  if (kcnt < 0) {
    klo = 0;
    kcnt = gv.sz[2];
  }
  for (int a = 0; a < 3; a++) {
    if (gv.ngd[a] == 0 || !(dirs & (1 << a))) continue;
    long long cnt = (long long)gv.nvar;
    for (int b = 0; b < 3; b++) cnt *= (b == a) ? 2 * gv.ngd[a] : (b == 2 ? kcnt : gv.sz[b]);
    if (cnt <= 0) continue;
    const unsigned blocks = (unsigned)((cnt + tb - 1) / tb);
    if (a == 0) fill_ghosts_kernel<0><<<blocks, tb, 0, s>>>(gv, bc[0][0], bc[0][1], P, klo, kcnt);
    if (a == 1) fill_ghosts_kernel<1><<<blocks, tb, 0, s>>>(gv, bc[1][0], bc[1][1], P, klo, kcnt);
    if (a == 2) fill_ghosts_kernel<2><<<blocks, tb, 0, s>>>(gv, bc[2][0], bc[2][1], P, klo, kcnt);
    launches++;
  }
  return launches;
}

// ---------------------------------------------------------------------------------------------------------
// Per-stage statistics: iteration histogram, unconverged count, max ||R||/scale
// ---------------------------------------------------------------------------------------------------------
template <int N, class G>
__global__ void stats_kernel(GridView gv, const double *__restrict__ Pn, double dt_stage,
                             const double *__restrict__ resnorm, const int32_t *__restrict__ status,
                             const int32_t *__restrict__ iters, StatsDev *out) {
  // per-block histogram in shared memory, one global atomic per non-empty bin and block (the per-thread global
  // atomics of the first version serialised 16.8 M updates on a handful of addresses: 18.6 ms at 256^3)
  __shared__ unsigned int s_hist[16];
  __shared__ unsigned int s_unconv;
  __shared__ unsigned long long s_max;
  if (threadIdx.x < 16) s_hist[threadIdx.x] = 0;
  if (threadIdx.x == 16) s_unconv = 0;
  if (threadIdx.x == 17) s_max = 0;
  __syncthreads();
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  double rel = 0.0;
  int unconv = 0;
  if (t < gv.nint) {
    int i, j, k;
    zone_coords(gv, t, i, j, k);
    const long long z = zone_index(gv, i, j, k);
    int it = iters[z];
    it = it > 15 ? 15 : it;
    atomicAdd(&s_hist[it], 1u);
    unconv = (status[z] & ST_CONVERGED) ? 0 : 1;
    G g;
    double tau = gv.tau_const;
    if constexpr (!G::flat) load_geom<0>(gv.geomC, gv.n2d, (long long)j * gv.sz[0] + i, g, tau);
    double P[N], U[N];
#pragma unroll
    for (int v = 0; v < N; v++) P[v] = Pn[v * gv.zg + z];
    Pieces pc;
    ExactArith ar;
    full_state<N>(ar, gv.m, g, tau, P, pc.th, pc.v, pc.b, pc.h);
    flux_vector<N>(g, 0, P, pc.th, pc.v, pc.b, pc.h, U);
    const double sc = sqrt(norm2sq<N>(U)) / dt_stage;
    rel = resnorm[z] / sc;
    if (!(rel > 0.0)) rel = 0.0;
  }
  const unsigned nun = __reduce_add_sync(0xffffffffu, (unsigned)unconv);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) rel = fmax(rel, __shfl_xor_sync(0xffffffffu, rel, o));
  if ((threadIdx.x & 31) == 0) {
    if (nun) atomicAdd(&s_unconv, nun);
    if (rel > 0.0) atomicMax(&s_max, (unsigned long long)__double_as_longlong(rel));
  }
  __syncthreads();
  if (threadIdx.x < 16 && s_hist[threadIdx.x]) atomicAdd(&out->hist[threadIdx.x], (unsigned long long)s_hist[threadIdx.x]);
  if (threadIdx.x == 16 && s_unconv) atomicAdd(&out->unconverged, (unsigned long long)s_unconv);
  if (threadIdx.x == 17 && s_max) atomicMax(&out->max_rel, s_max);
}

int launch_stats(const GridView &gv, const double *Pn, double dt_stage, const double *resnorm,
                 const int32_t *status, const int32_t *iters, StatsDev *out, cudaStream_t s) {
  const int tb = 256;
  const unsigned blocks = (unsigned)((gv.nint + tb - 1) / tb);
  const bool flat = gv.metric == 0;
  if (gv.nvar == 10) {
    if (flat) stats_kernel<10, GeomFlat><<<blocks, tb, 0, s>>>(gv, Pn, dt_stage, resnorm, status, iters, out);
    else stats_kernel<10, GeomGen><<<blocks, tb, 0, s>>>(gv, Pn, dt_stage, resnorm, status, iters, out);
  } else {
    if (flat) stats_kernel<8, GeomFlat><<<blocks, tb, 0, s>>>(gv, Pn, dt_stage, resnorm, status, iters, out);
    else stats_kernel<8, GeomGen><<<blocks, tb, 0, s>>>(gv, Pn, dt_stage, resnorm, status, iters, out);
  }
  return 1;
}

// copies the interior zones of every variable (the stage result) from src to dst
__global__ void copy_interior_kernel(GridView gv, const double *__restrict__ src, double *__restrict__ dst) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= gv.nint * gv.nvar) return;
  const int v = (int)(t / gv.nint);
  int i, j, k;
  zone_coords(gv, t % gv.nint, i, j, k);
  const long long z = v * gv.zg + zone_index(gv, i, j, k);
  dst[z] = src[z];
}

int launch_copy_interior(const GridView &gv, const double *src, double *dst, cudaStream_t s) {
  const int tb = 256;
  const long long cnt = gv.nint * gv.nvar;
  copy_interior_kernel<<<(unsigned)((cnt + tb - 1) / tb), tb, 0, s>>>(gv, src, dst);
  return 1;
}

// ---------------------------------------------------------------------------------------------------------
// fp64 pipe probe: 8 independent accumulator chains per thread
// ---------------------------------------------------------------------------------------------------------
template <int FMA>
__global__ void fp64_probe_kernel(int iters, double *sink) {
  double a0 = threadIdx.x * 1e-9, a1 = a0 + 1.0, a2 = a0 + 2.0, a3 = a0 + 3.0, a4 = a0 + 4.0, a5 = a0 + 5.0,
         a6 = a0 + 6.0, a7 = a0 + 7.0;
  const double m = 1.0000001, c = 1e-9;
  for (int i = 0; i < iters; i++) {
    if (FMA) {
      a0 = __fma_rn(a0, m, c); a1 = __fma_rn(a1, m, c); a2 = __fma_rn(a2, m, c); a3 = __fma_rn(a3, m, c);
      a4 = __fma_rn(a4, m, c); a5 = __fma_rn(a5, m, c); a6 = __fma_rn(a6, m, c); a7 = __fma_rn(a7, m, c);
    } else {
      a0 = __dmul_rn(a0, m); a1 = __dadd_rn(a1, c); a2 = __dmul_rn(a2, m); a3 = __dadd_rn(a3, c);
      a4 = __dmul_rn(a4, m); a5 = __dadd_rn(a5, c); a6 = __dmul_rn(a6, m); a7 = __dadd_rn(a7, c);
    }
  }
  const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
  if (s == 123.456) sink[0] = s;
}

// ---------------------------------------------------------------------------------------------------------
// Arithmetic self-test: SpecArith against ExactArith (the IEEE operators), operation by operation, on
// pseudo-random operands.  Sample n of a launch: two 64-bit hashes (splitmix64 of the counter) give the
// mantissas; exponents cycle through the whole fp64 range in `wide` mode (the in-range guard must then reject
// what the straight-line code gets wrong) or stay within +-400 of 1.  A sample counts as a mismatch when the
// speculative result differs in any bit from the exact one while the policy still reports ok.
// out[0..4]: mismatches of div, rcp, sqrt, div60, div_z/sqrt_z; out[5]: samples the guard accepted.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long splitmix64(unsigned long long x) {
  x += 0x9E3779B97F4A7C15ULL;
  x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ULL;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBULL;
  return x ^ (x >> 31);
}
__device__ __forceinline__ bool same_bits(double a, double b) {
  return __double_as_longlong(a) == __double_as_longlong(b) || (a != a && b != b);
}
__global__ void arith_selftest_kernel(unsigned long long n, unsigned long long seed, int wide,
                                      unsigned long long *out) {
  unsigned long long bad[5] = {0, 0, 0, 0, 0}, accepted = 0;
  for (unsigned long long t = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; t < n;
       t += (unsigned long long)gridDim.x * blockDim.x) {
    const unsigned long long h1 = splitmix64(seed + 2 * t), h2 = splitmix64(seed + 2 * t + 1);
    unsigned long long ma = h1 & 0x000FFFFFFFFFFFFFULL, mb = h2 & 0x000FFFFFFFFFFFFFULL;
    // every 8th sample: mantissas at the ends of the binade (all zeros / all ones / one bit), the hard cases
    if ((t & 7) == 7) {
      const unsigned sel = (unsigned)(h1 >> 52) & 3;
      ma = sel == 0 ? 0 : sel == 1 ? 0x000FFFFFFFFFFFFFULL : sel == 2 ? (1ULL << ((h1 >> 54) % 52)) : ma;
      const unsigned sel2 = (unsigned)(h2 >> 52) & 3;
      mb = sel2 == 0 ? 0 : sel2 == 1 ? 0x000FFFFFFFFFFFFFULL : sel2 == 2 ? (0x000FFFFFFFFFFFFFULL ^ (1ULL << ((h2 >> 54) % 52))) : mb;
    }
    unsigned long long ea, eb;
    if (wide) {
      ea = (h1 >> 52) & 0x7FF;
      eb = (h2 >> 52) & 0x7FF;
    } else {
      ea = 1023 - 400 + ((h1 >> 52) & 0x7FF) % 801;
      eb = 1023 - 400 + ((h2 >> 52) & 0x7FF) % 801;
    }
    const unsigned long long sa = wide ? (h1 >> 63) << 63 : 0, sb = (h2 >> 63) << 63;
    const double a = __longlong_as_double((long long)(sa | (ea << 52) | ma));
    const double b = __longlong_as_double((long long)(sb | (eb << 52) | mb));
    const double az = ((t & 63) == 5) ? (wide && (t & 64) ? -0.0 : 0.0) : a;
    ExactArith ex;
    {
      SpecArith sp;
      const double r = sp.div(a, b);
      if (sp.ok) { accepted++; if (!same_bits(r, ex.div(a, b))) bad[0]++; }
    }
    {
      SpecArith sp;
      const double r = sp.rcp(b);
      if (sp.ok && !same_bits(r, ex.rcp(b))) bad[1]++;
    }
    {
      SpecArith sp;
      const double r = sp.sqrt(a);
      if (sp.ok && !same_bits(r, ex.sqrt(a))) bad[2]++;
    }
    {
      SpecArith sp;
      const double r = div60(sp, az);
      if (sp.ok && !same_bits(r, div60(ex, az))) bad[3]++;
    }
    {
      SpecArith sp;
      const double r = sp.div_z(az, b);
      if (sp.ok && !same_bits(r, ex.div_z(az, b))) bad[4]++;
      SpecArith sq;
      const double r2 = sq.sqrt_z(az);
      if (sq.ok && !same_bits(r2, ex.sqrt_z(az))) bad[4]++;
    }
  }
  for (int k = 0; k < 5; k++)
    if (bad[k]) atomicAdd(&out[k], bad[k]);
  if (accepted) atomicAdd(&out[5], accepted);
}

int launch_arith_selftest(unsigned long long n, unsigned long long seed, int wide, unsigned long long *out,
                          cudaStream_t s) {
  arith_selftest_kernel<<<148 * 8, 256, 0, s>>>(n, seed, wide, out);
  return 1;
}

int launch_fp64_probe(int fma, int iters, double *sink, int blocks, int threads, cudaStream_t s) {
  if (fma) fp64_probe_kernel<1><<<blocks, threads, 0, s>>>(iters, sink);
  else fp64_probe_kernel<0><<<blocks, threads, 0, s>>>(iters, sink);
  return 1;
}

}  // namespace grim
