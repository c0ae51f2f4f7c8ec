"""ctypes binding of the ORACLE (oracle/grim_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It marshals numpy arrays to the C functions and nothing else; all arithmetic is in grim_oracle.c.
"""
import ctypes as C
import os
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
if _HERE not in sys.path:
    sys.path.insert(0, _HERE)
import build as _build  # noqa: E402

NMAX = 10
MINKOWSKI, KERR_MKS = 0, 1
MINMOD, MP5 = 0, 1
LLF, HLLE = 0, 1
BC_PERIODIC, BC_OUTFLOW, BC_REFLECT_POLAR, BC_NONE = 0, 1, 2, 3
TAU_CONST, TAU_R32 = 0, 1
CLOSURE_CS2TAU, CLOSURE_CONST = 0, 1
ST_CONVERGED, ST_KMAX, ST_LS_EXHAUSTED, ST_SINGULAR, ST_NONFINITE = 1, 2, 4, 8, 16


class Geom(C.Structure):
    _fields_ = [("gcov", (C.c_double * 4) * 4), ("gcon", (C.c_double * 4) * 4),
                ("sqrtmg", C.c_double), ("alpha", C.c_double)]


class Model(C.Structure):
    _fields_ = [("nvar", C.c_int32), ("gam", C.c_double), ("phi", C.c_double), ("psi", C.c_double),
                ("closure", C.c_int32)]


class Solver(C.Structure):
    _fields_ = [("fd_eps", C.c_double), ("eps_bt", C.c_double), ("atol", C.c_double), ("rtol", C.c_double),
                ("kmax", C.c_int32), ("lsmax", C.c_int32)]


class GridDesc(C.Structure):
    _fields_ = [("n1", C.c_int32), ("n2", C.c_int32), ("n3", C.c_int32), ("ng", C.c_int32), ("dim", C.c_int32),
                ("xstart", C.c_double * 3), ("xend", C.c_double * 3), ("bc", (C.c_int32 * 2) * 3),
                ("nvar", C.c_int32), ("recon", C.c_int32), ("limiter_theta", C.c_double),
                ("riemann", C.c_int32), ("gam", C.c_double), ("phi", C.c_double), ("psi", C.c_double),
                ("tau_mode", C.c_int32), ("tau", C.c_double),
                ("fd_eps", C.c_double), ("eps_bt", C.c_double), ("atol", C.c_double), ("rtol", C.c_double),
                ("kmax", C.c_int32), ("lsmax", C.c_int32), ("cfl", C.c_double), ("flux_ct", C.c_int32),
                ("closure", C.c_int32), ("reduced", C.c_int32)]


class StepStats(C.Structure):
    _fields_ = [("zones", C.c_int64), ("iters_hist", (C.c_int64 * 16) * 2), ("backtracks", C.c_int64 * 2),
                ("unconverged", C.c_int64 * 2), ("max_resnorm", C.c_double * 2)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _declare(_lib)
    return _lib


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


def _declare(L):
    L.og_num_threads.restype = C.c_int
    L.og_geom_minkowski.argtypes = [C.POINTER(Geom)]
    L.og_geom_kerr_mks.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, C.POINTER(Geom)]
    L.og_conn_kerr_mks.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, _dp]
    L.og_prim_to_U.argtypes = [C.POINTER(Model), C.POINTER(Geom), C.c_double, _dp, _dp]
    L.og_prim_to_F.argtypes = [C.POINTER(Model), C.POINTER(Geom), C.c_double, C.c_int, _dp, _dp]
    L.og_vmax2.argtypes = [C.POINTER(Model), C.POINTER(Geom), C.c_double, _dp]
    L.og_vmax2.restype = C.c_double
    L.og_wave_speeds.argtypes = [C.POINTER(Model), C.POINTER(Geom), C.c_double, C.c_int, _dp, _dp, _dp]
    L.og_cmax.argtypes = [C.POINTER(Model), C.POINTER(Geom), C.c_double, C.c_int, _dp]
    L.og_cmax.restype = C.c_double
    L.og_derived.argtypes = [C.POINTER(Model), C.POINTER(Geom), _dp, _dp, _dp, _dp]
    L.og_emhd_targets.argtypes = [C.POINTER(Model), C.POINTER(Geom), _dp, C.c_double, _dp, _dp, _dp,
                                  C.c_double, _dp, _dp]
    L.og_rescale_factors.argtypes = [C.POINTER(Model), C.c_double, _dp, _dp, _dp]
    L.og_geometric_source.argtypes = [C.POINTER(Model), C.POINTER(Geom), _dp, _dp, _dp]
    L.og_stress_tensor.argtypes = [C.POINTER(Model), C.POINTER(Geom), _dp, _dp]
    L.og_minmod3.argtypes = [C.c_double] * 3
    L.og_minmod3.restype = C.c_double
    L.og_slope.argtypes = [C.c_double] * 4
    L.og_slope.restype = C.c_double
    L.og_reconstruct.argtypes = [C.c_int, C.c_double, _dp, _dp, _dp]
    L.og_mp5_face.argtypes = [C.c_double] * 5
    L.og_mp5_face.restype = C.c_double
    L.og_lu_solve.argtypes = [C.c_int, _dp, _dp, _ip]
    L.og_lu_solve.restype = C.c_int
    L.og_linesearch_lambda.argtypes = [C.c_double] * 3
    L.og_linesearch_lambda.restype = C.c_double
    L.og_llf.argtypes = [C.c_int, _dp, _dp, _dp, _dp, C.c_double, _dp]
    L.og_hlle.argtypes = [C.c_int, _dp, _dp, _dp, _dp, C.c_double, C.c_double, _dp]
    L.og_grid_create.argtypes = [C.POINTER(GridDesc)]
    L.og_grid_create.restype = C.c_void_p
    L.og_grid_free.argtypes = [C.c_void_p]
    L.og_grid_set_metric.argtypes = [C.c_void_p, C.c_int, _dp, C.c_int]
    L.og_grid_set_metric.restype = C.c_int
    L.og_grid_zones_padded.argtypes = [C.c_void_p]
    L.og_grid_zones_padded.restype = C.c_int64
    L.og_fill_ghosts.argtypes = [C.c_void_p, _dp]
    L.og_grid_get_geom.argtypes = [C.c_void_p, C.c_int, C.c_int64, C.POINTER(Geom)]
    L.og_grid_get_conn.argtypes = [C.c_void_p, C.c_int64, _dp]
    L.og_grid_get_tau.argtypes = [C.c_void_p, C.c_int, C.c_int64]
    L.og_grid_get_tau.restype = C.c_double
    L.og_stage_prepare.argtypes = [C.c_void_p, _dp, _dp, C.c_double, _dp, _dp, _dp]
    L.og_zone_residual.argtypes = [C.c_void_p, C.c_int64, _dp, _dp, _dp, _dp, C.c_double, _dp, _dp]
    L.og_newton.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, C.c_double, _dp, C.c_int, _dp, _ip, _ip,
                            C.POINTER(C.c_int64)]
    L.og_newton.restype = C.c_int64
    L.og_choose_dt.argtypes = [C.c_void_p, _dp]
    L.og_choose_dt.restype = C.c_double
    L.og_timestep.argtypes = [C.c_void_p, _dp, C.c_double, C.POINTER(StepStats)]
    L.og_invert.argtypes = [C.POINTER(Model), C.POINTER(Solver), C.c_double, C.c_int64, _dp, C.POINTER(Geom),
                            _dp, _ip, _ip, _dp, C.POINTER(C.c_int64)]


def _d(a):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def _i(a):
    assert a.dtype == np.int32 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_ip)


def num_threads():
    return lib().og_num_threads()


def minkowski():
    g = Geom()
    lib().og_geom_minkowski(C.byref(g))
    return g


def kerr_mks(a, h, X1, X2):
    g = Geom()
    lib().og_geom_kerr_mks(a, h, X1, X2, C.byref(g))
    return g


def kerr_mks_conn(a, h, X1, X2):
    out = np.zeros((4, 4, 4))
    lib().og_conn_kerr_mks(a, h, X1, X2, _d(out))
    return out


def geom_arrays(g):
    return (np.array([[g.gcov[i][j] for j in range(4)] for i in range(4)]),
            np.array([[g.gcon[i][j] for j in range(4)] for i in range(4)]), g.sqrtmg, g.alpha)


def model(nvar=10, gam=4.0 / 3.0, phi=1.0, psi=1.0, closure=0):
    return Model(nvar, gam, phi, psi, closure)


def solver(fd_eps=4e-8, eps_bt=1e-4, atol=0.0, rtol=1e-12, kmax=30, lsmax=8):
    return Solver(fd_eps, eps_bt, atol, rtol, kmax, lsmax)


def prim_to_U(m, g, tau, P):
    P = np.ascontiguousarray(P, dtype=np.float64)
    U = np.zeros(m.nvar)
    lib().og_prim_to_U(C.byref(m), C.byref(g), tau, _d(P), _d(U))
    return U


def prim_to_F(m, g, tau, d, P):
    P = np.ascontiguousarray(P, dtype=np.float64)
    F = np.zeros(m.nvar)
    lib().og_prim_to_F(C.byref(m), C.byref(g), tau, d, _d(P), _d(F))
    return F


def vmax2(m, g, tau, P):
    P = np.ascontiguousarray(P, dtype=np.float64)
    return lib().og_vmax2(C.byref(m), C.byref(g), tau, _d(P))


def wave_speeds(m, g, tau, d, P):
    P = np.ascontiguousarray(P, dtype=np.float64)
    vp, vm = C.c_double(), C.c_double()
    lib().og_wave_speeds(C.byref(m), C.byref(g), tau, d, _d(P), C.byref(vp), C.byref(vm))
    return vp.value, vm.value


def cmax(m, g, tau, d, P):
    P = np.ascontiguousarray(P, dtype=np.float64)
    return lib().og_cmax(C.byref(m), C.byref(g), tau, d, _d(P))


def derived(m, g, P):
    """Theta, u^mu, u_mu of state P."""
    P = np.ascontiguousarray(P, dtype=np.float64)
    th = C.c_double()
    ucon, ucov = np.zeros(4), np.zeros(4)
    lib().og_derived(C.byref(m), C.byref(g), _d(P), C.byref(th), _d(ucon), _d(ucov))
    return th.value, ucon, ucov


def emhd_targets(m, g, conn, tau, PE, dTheta, ducov, divu):
    PE = np.ascontiguousarray(PE, dtype=np.float64)
    conn = np.ascontiguousarray(conn, dtype=np.float64)
    dTheta = np.ascontiguousarray(dTheta, dtype=np.float64)
    ducov = np.ascontiguousarray(ducov, dtype=np.float64)
    q0, dP0 = C.c_double(), C.c_double()
    lib().og_emhd_targets(C.byref(m), C.byref(g), _d(conn), tau, _d(PE), _d(dTheta), _d(ducov), divu,
                          C.byref(q0), C.byref(dP0))
    return q0.value, dP0.value


def geometric_source(m, g, conn, P):
    """S_nu = sqrt(-g) T^k_l Gamma^l_{nu k}, nu = 0..3 (eq 31), as og_stage_prepare forms it."""
    P = np.ascontiguousarray(P, dtype=np.float64)
    conn = np.ascontiguousarray(conn, dtype=np.float64)
    S = np.zeros(4)
    lib().og_geometric_source(C.byref(m), C.byref(g), _d(conn), _d(P), _d(S))
    return S


def stress_tensor(m, g, P):
    """T^mu_nu [mu][nu] of state P."""
    P = np.ascontiguousarray(P, dtype=np.float64)
    T = np.zeros((4, 4))
    lib().og_stress_tensor(C.byref(m), C.byref(g), _d(P), _d(T))
    return T


def rescale_factors(m, tau, P):
    P = np.ascontiguousarray(P, dtype=np.float64)
    fq, fd = C.c_double(), C.c_double()
    lib().og_rescale_factors(C.byref(m), tau, _d(P), C.byref(fq), C.byref(fd))
    return fq.value, fd.value


def minmod3(a, b, c):
    return lib().og_minmod3(a, b, c)


def slope(theta, vm, v0, vp):
    return lib().og_slope(theta, vm, v0, vp)


def reconstruct(recon, theta, v5):
    v5 = np.ascontiguousarray(v5, dtype=np.float64)
    a, b = C.c_double(), C.c_double()
    lib().og_reconstruct(recon, theta, _d(v5), C.byref(a), C.byref(b))
    return a.value, b.value


def mp5_face(v5):
    return lib().og_mp5_face(*[float(x) for x in v5])


def lu_solve(A, b):
    """Returns (x, piv, info); A, b untouched."""
    A = np.array(A, dtype=np.float64, order="C")
    x = np.array(b, dtype=np.float64)
    n = A.shape[0]
    piv = np.zeros(n, dtype=np.int32)
    info = lib().og_lu_solve(n, _d(A), _d(x), _i(piv))
    return x, piv, info


def linesearch_lambda(f0, flam, lam):
    return lib().og_linesearch_lambda(f0, flam, lam)


def hlle(Fm, Fp, Um, Up, cR, cL):
    Fm, Fp, Um, Up = (np.ascontiguousarray(x, dtype=np.float64) for x in (Fm, Fp, Um, Up))
    F = np.zeros(len(Fm))
    lib().og_hlle(len(Fm), _d(Fm), _d(Fp), _d(Um), _d(Up), cR, cL, _d(F))
    return F


def llf(Fm, Fp, Um, Up, c):
    Fm, Fp, Um, Up = [np.ascontiguousarray(x, dtype=np.float64) for x in (Fm, Fp, Um, Up)]
    F = np.zeros_like(Fm)
    lib().og_llf(len(Fm), _d(Fm), _d(Fp), _d(Um), _d(Up), c, _d(F))
    return F


def invert(m, s, Ustar, Pguess, tau=1.0, geoms=None):
    """Flat SoA [v][z] standalone inversion (O-10); geoms: None (Minkowski) or one Geom per zone.
    Returns P, iters, status, resnorm, backtracks."""
    Ustar = np.ascontiguousarray(Ustar, dtype=np.float64)
    P = np.array(Pguess, dtype=np.float64, order="C")
    nz = P.shape[1]
    iters = np.zeros(nz, dtype=np.int32)
    status = np.zeros(nz, dtype=np.int32)
    resnorm = np.zeros(nz)
    bt = C.c_int64(0)
    garr = None
    if geoms is not None:
        assert len(geoms) == nz
        garr = (Geom * nz)(*geoms)
    lib().og_invert(C.byref(m), C.byref(s), tau, nz, _d(Ustar), garr, _d(P), _i(iters), _i(status),
                    _d(resnorm), C.byref(bt))
    return P, iters, status, resnorm, bt.value


class Grid:
    """Owns an og_grid.  Arrays are numpy float64 [nvar, s3, s2, s1] (ghosts included)."""

    def __init__(self, n1, n2=1, n3=1, ng=3, dim=2, xstart=(0, 0, 0), xend=(1, 1, 1),
                 bc=BC_PERIODIC, nvar=10, recon=MINMOD, limiter_theta=1.0, gam=4.0 / 3.0, phi=1.0, psi=1.0,
                 tau_mode=TAU_CONST, tau=1.0, fd_eps=4e-8, eps_bt=1e-4, atol=0.0, rtol=1e-14, kmax=8,
                 lsmax=5, cfl=0.5, metric=MINKOWSKI, metric_params=(), flux_ct=False, reduced=False, riemann=0,
                 closure=0):
        d = GridDesc()
        d.flux_ct = 1 if flux_ct else 0
        d.reduced = 1 if reduced else 0
        d.closure = closure
        d.n1, d.n2, d.n3, d.ng, d.dim = n1, n2, n3, ng, dim
        for a in range(3):
            d.xstart[a], d.xend[a] = float(xstart[a]), float(xend[a])
            for s in range(2):
                d.bc[a][s] = bc if np.isscalar(bc) else bc[a][s]
        d.nvar, d.recon, d.limiter_theta, d.riemann = nvar, recon, limiter_theta, riemann
        d.gam, d.phi, d.psi, d.tau_mode, d.tau = gam, phi, psi, tau_mode, tau
        d.fd_eps, d.eps_bt, d.atol, d.rtol, d.kmax, d.lsmax, d.cfl = fd_eps, eps_bt, atol, rtol, kmax, lsmax, cfl
        self.desc = d
        self.h = lib().og_grid_create(C.byref(d))
        mp = np.array(metric_params, dtype=np.float64)
        rc = lib().og_grid_set_metric(self.h, metric, _d(mp) if mp.size else None, int(mp.size))
        assert rc == 0
        self.nvar = nvar
        self.n = (n1, n2, n3)
        self.ngd = tuple(ng if a < dim else 0 for a in range(3))
        self.sz = tuple(self.n[a] + 2 * self.ngd[a] for a in range(3))
        self.shape = (nvar, self.sz[2], self.sz[1], self.sz[0])
        self.zg = self.sz[0] * self.sz[1] * self.sz[2]
        assert self.zg == lib().og_grid_zones_padded(self.h)
        self.dx = tuple((xend[a] - xstart[a]) / self.n[a] for a in range(3))
        self.xstart = tuple(xstart)

    def __del__(self):
        try:
            lib().og_grid_free(self.h)
        except Exception:
            pass

    def interior(self, A):
        g = self.ngd
        return A[..., g[2]:g[2] + self.n[2], g[1]:g[1] + self.n[1], g[0]:g[0] + self.n[0]]

    def centers(self):
        """Zone-centre coordinates X^1, X^2, X^3 of the padded grid, broadcast to [s3, s2, s1]."""
        ax = [self.xstart[a] + (np.arange(self.sz[a]) - self.ngd[a] + 0.5) * self.dx[a] for a in range(3)]
        X3, X2, X1 = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
        return X1, X2, X3

    def zeros(self):
        return np.zeros(self.shape)

    def fill_ghosts(self, P):
        lib().og_fill_ghosts(self.h, _d(P))

    def geom(self, loc, j, i):
        g = Geom()
        lib().og_grid_get_geom(self.h, loc, j * self.sz[0] + i, C.byref(g))
        return g

    def conn(self, j, i):
        out = np.zeros((4, 4, 4))
        lib().og_grid_get_conn(self.h, j * self.sz[0] + i, _d(out))
        return out

    def tau(self, loc, j, i):
        return lib().og_grid_get_tau(self.h, loc, j * self.sz[0] + i)

    def geometry_tables(self):
        """The grid's geometry as plain tables over the padded 2-D plane (idx2d = j*s1 + i), in the layout of
        include/grim.h grim_set_metric_tables: tab[loc][comp][idx2d] with comp 0..9 = g_mu_nu (00 01 02 03 11 12 13
        22 23 33), 10..19 = g^mu^nu, 20 = sqrt(-g), 21 = lapse, 22 = tau_R; conn[l*16 + m*4 + n][idx2d].  Copies
        of stored values only (no arithmetic)."""
        n2d = self.sz[0] * self.sz[1]
        tab = np.zeros((4, 23, n2d))
        conn = np.zeros((64, n2d))
        sym = [(0, 0), (0, 1), (0, 2), (0, 3), (1, 1), (1, 2), (1, 3), (2, 2), (2, 3), (3, 3)]
        for j in range(self.sz[1]):
            for i in range(self.sz[0]):
                id2 = j * self.sz[0] + i
                for loc in range(4):
                    g = self.geom(loc, j, i)
                    for c, (m, n) in enumerate(sym):
                        tab[loc, c, id2] = g.gcov[m][n]
                        tab[loc, 10 + c, id2] = g.gcon[m][n]
                    tab[loc, 20, id2] = g.sqrtmg
                    tab[loc, 21, id2] = g.alpha
                    tab[loc, 22, id2] = self.tau(loc, j, i)
                conn[:, id2] = self.conn(j, i).reshape(64)
        return tab, conn

    def stage_prepare(self, Pn, PE, dt_stage):
        Cc = np.zeros(self.shape)
        G = np.zeros((3,) + self.shape[1:])
        sp = np.zeros(4)
        lib().og_stage_prepare(self.h, _d(Pn), _d(PE), dt_stage, _d(Cc), _d(G), _d(sp))
        return Cc, G, sp

    def zone_residual(self, z, Pn, PE, Cc, G, dt_stage, P):
        P = np.ascontiguousarray(P, dtype=np.float64)
        R = np.zeros(self.nvar)
        lib().og_zone_residual(self.h, z, _d(Pn), _d(PE), _d(Cc), _d(G), dt_stage, _d(P), _d(R))
        return R

    def newton(self, Pn, PE, Cc, G, dt_stage, P_iter, max_iters=0, state=None):
        """Runs Newton iterations in place on P_iter.  state = (resnorm, status, iters) carried between calls."""
        if state is None:
            state = (np.zeros(self.shape[1:]), np.zeros(self.shape[1:], dtype=np.int32),
                     np.zeros(self.shape[1:], dtype=np.int32))
        rn, st, it = state
        bt = C.c_int64(0)
        nact = lib().og_newton(self.h, _d(Pn), _d(PE), _d(Cc), _d(G), dt_stage, _d(P_iter), max_iters,
                               _d(rn), _i(st), _i(it), C.byref(bt))
        return nact, state, bt.value

    def choose_dt(self, P):
        return lib().og_choose_dt(self.h, _d(P))

    def timestep(self, P, dt):
        st = StepStats()
        lib().og_timestep(self.h, _d(P), dt, C.byref(st))
        return st
