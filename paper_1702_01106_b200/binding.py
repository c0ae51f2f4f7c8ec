"""ctypes binding of libgrim_b200.so (include/grim.h).  Marshalling only; torch provides device memory/streams.

The `Grid` methods carry the names of the C entry points without the `grim_` prefix.  Tensor arguments must be
contiguous CUDA tensors of the stated dtype on the grid's device; they are passed as raw device pointers.
"""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))

IDEAL, EMHD = 8, 10
MINKOWSKI, KERR_MKS = 0, 1
MINMOD, MP5 = 0, 1
LLF, HLLE = 0, 1
BC_PERIODIC, BC_OUTFLOW, BC_REFLECT_POLAR, BC_NONE = 0, 1, 2, 3
TAU_CONST, TAU_R32 = 0, 1
ST_CONVERGED, ST_KMAX, ST_LS_EXHAUSTED, ST_SINGULAR, ST_NONFINITE = 1, 2, 4, 8, 16
ST_TERMINAL = ST_CONVERGED | ST_KMAX | ST_SINGULAR | ST_NONFINITE


class GrimError(RuntimeError):
    pass


class GridDesc(C.Structure):
    _fields_ = [("n1", C.c_int32), ("n2", C.c_int32), ("n3", C.c_int32), ("ng", C.c_int32), ("dim", C.c_int32),
                ("xstart", C.c_double * 3), ("xend", C.c_double * 3), ("bc", (C.c_int32 * 2) * 3),
                ("model", C.c_int32), ("recon", C.c_int32), ("limiter_theta", C.c_double), ("riemann", C.c_int32),
                ("gamma", C.c_double), ("phi", C.c_double), ("psi", C.c_double),
                ("tau_mode", C.c_int32), ("tau", C.c_double),
                ("fd_eps", C.c_double), ("eps_bt", C.c_double), ("atol", C.c_double), ("rtol", C.c_double),
                ("kmax", C.c_int32), ("lsmax", C.c_int32), ("cfl", C.c_double),
                ("device", C.c_int32), ("stream", C.c_void_p), ("flux_ct", C.c_int32), ("reduced_solve", C.c_int32),
                ("closure", C.c_int32)]


class StepStats(C.Structure):
    _fields_ = [("zones", C.c_int64), ("iters_hist", (C.c_int64 * 16) * 2), ("backtracks", C.c_int64 * 2),
                ("unconverged", C.c_int64 * 2), ("max_resnorm", C.c_double * 2)]


_vp, _dbl, _i32, _i64 = C.c_void_p, C.c_double, C.c_int32, C.c_int64
_pd, _pi32, _pi64 = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_int64)

# name -> (restype, argtypes): every symbol include/grim.h declares
_SIGNATURES = {
    "grim_init_grid": (C.c_int, [C.POINTER(_vp), C.POINTER(GridDesc)]),
    "grim_set_metric": (C.c_int, [_vp, _i32, _pd, _i32]),
    "grim_set_metric_tables": (C.c_int, [_vp, _pd, _pd]),
    "grim_compute_fluxes": (C.c_int, [_vp, _vp, _vp, _dbl, _vp, _vp, _vp]),
    "grim_newton_step": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _dbl, _i32, _vp, _vp, _vp, _vp, _pi64]),
    "grim_newton_solve": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _dbl, _vp, _vp, _vp, _vp, _vp]),
    "grim_invert_primitives": (C.c_int, [_vp, _i64, _vp, _vp, _vp, _vp, _vp, _vp]),
    "grim_timestep": (C.c_int, [_vp, _vp, _dbl, _pd, C.POINTER(StepStats)]),
    "grim_free": (None, [_vp]),
    "grim_last_error": (C.c_char_p, [_vp]),
    "grim_version": (C.c_int, []),
    "grim_zones_padded": (_i64, [_vp, _pi32]),
    "grim_fill_ghosts": (C.c_int, [_vp, _vp]),
    "grim_prim_to_conserved": (C.c_int, [_vp, _i64, _vp, _vp]),
    "grim_get_geometry": (C.c_int, [_vp, _i32, _i64, _pd, _pd, _pd, _pd, _pd, _pd]),
    "grim_fp64_probe": (C.c_int, [_vp, _i32, _i32, _pd]),
    "grim_arith_selftest": (C.c_int, [_vp, _i64, _i64, _i32, _pi64]),
    "grim_timestep_host": (C.c_int, [_vp, _vp, _i32, _dbl, _pd]),
    "grim_last_host_mode": (C.c_int, [_vp]),
    "grim_invert_primitives_host": (C.c_int, [_vp, _i64, _vp, _vp, _vp, _vp, _vp]),
    "grim_invert_primitives_static": (C.c_int, [C.POINTER(GridDesc), _i64, _vp, _vp, _vp, _vp, _vp, _vp]),
    "grim_launch_count": (_i64, [_vp]),
    "grim_set_timing": (C.c_int, [_vp, _i32]),
    "grim_get_timing": (C.c_int, [_vp, _pd, _pi64]),
}

KERNEL_CLASSES = ("ghosts", "flux", "newton", "invert", "other")
HOST_MODES = ("none", "whole", "pipelined")      # GRIM_HOST_MODE_*
ABI_VERSION = 101                                # GRIM_VERSION this file's ctypes layouts (GridDesc, StepStats) mirror


def exported_symbols():
    return sorted(_SIGNATURES)


def lib_path():
    return os.path.join(HERE, "libgrim_b200.so")


_lib = None


def lib():
    """Loads the CUDA library.  No fallback: a missing library is an error."""
    global _lib
    if _lib is None:
        p = lib_path()
        if not os.path.exists(p):
            raise GrimError("%s is missing: build it with `python -m paper_1702_01106_b200.build` "
                            "(there is no CPU fallback)" % p)
        L = C.CDLL(p)
        L.grim_version.restype = C.c_int
        if L.grim_version() != ABI_VERSION:
            raise GrimError("%s is version %d, this binding mirrors the structs of version %d: rebuild it with "
                            "`python -m paper_1702_01106_b200.build --force`" % (p, L.grim_version(), ABI_VERSION))
        for name, (res, args) in _SIGNATURES.items():
            f = getattr(L, name)
            f.restype = res
            f.argtypes = args
        _lib = L
    return _lib


def _ptr(t, dtype=None):
    """Raw device pointer of a contiguous CUDA tensor (None -> NULL)."""
    if t is None:
        return None
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()):
        raise GrimError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise GrimError("expected dtype %s, got %s" % (dtype, t.dtype))
    return C.c_void_p(t.data_ptr())


def _host_ptr(t, dtype=None):
    import torch
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.is_contiguous()):
        raise GrimError("expected a contiguous host tensor")
    if dtype is not None and t.dtype != dtype:
        raise GrimError("expected dtype %s, got %s" % (dtype, t.dtype))
    return C.c_void_p(t.data_ptr())


STATIC_MAX_ZONES = 1 << 20   # GRIM_STATIC_MAX_ZONES of include/grim.h


def invert_primitives_static(U_target, P_inout, iters, status, resnorm, geom=None, model=IDEAL, gamma=4.0 / 3.0,
                             phi=1.0, psi=1.0, closure=0, tau=1.0, fd_eps=4e-8, eps_bt=1e-4, rtol=1e-14, kmax=8,
                             lsmax=5, device=0, stream=None):
    """grim_invert_primitives_static: the standalone inversion for a caller that must not allocate device memory.

    A `Grid` cannot be used by code that runs inside an application whose memory pool already holds the device's
    memory, or inside a loop that cannot afford the device-wide stall of cudaMalloc/cudaFree: creating a `Grid`
    allocates its scratch, and `Grid.invert_primitives` allocates its zone lists.  This function needs no `Grid` and
    allocates nothing, on any call: its scratch is a fixed 8 MiB array inside the library's device image, which is why
    at most STATIC_MAX_ZONES (2^20) zones fit in one call (more raises GrimError) and why two calls must never run on
    the same GPU at the same time (they would share, and corrupt, that array).  Make the first call on a device during
    set-up: that call looks up the array's device address.  Arguments and results are those of
    `Grid.invert_primitives`, bit for bit; the model and solver parameters are passed here instead of coming from a
    grid.  Returns after the stream is synchronised."""
    import torch
    d = GridDesc()
    d.n1 = d.n2 = d.n3 = 1
    d.dim = 1
    d.model, d.gamma, d.phi, d.psi, d.closure = model, gamma, phi, psi, closure
    d.tau_mode, d.tau = TAU_CONST, tau
    d.fd_eps, d.eps_bt, d.atol, d.rtol, d.kmax, d.lsmax = fd_eps, eps_bt, 0.0, rtol, kmax, lsmax
    d.device = device
    if stream is None:
        stream = torch.cuda.current_stream(device).cuda_stream
    d.stream = stream
    nz = P_inout.shape[1]
    if geom is not None and tuple(geom.shape) != (15, nz):
        raise GrimError("invert_primitives_static: geom must have shape (15, %d)" % nz)
    L = lib()
    f64, i32 = torch.float64, torch.int32
    rc = L.grim_invert_primitives_static(C.byref(d), nz, _ptr(U_target, f64), _ptr(geom, f64), _ptr(P_inout, f64),
                                         _ptr(iters, i32), _ptr(status, i32), _ptr(resnorm, f64))
    if rc != 0:
        msg = L.grim_last_error(None)
        raise GrimError("grim_invert_primitives_static failed (%d): %s" % (rc, msg.decode() if msg else ""))


class Grid:
    """Owns a grim_ctx.  Grid arrays are torch.float64 CUDA tensors of shape [nvar, s3, s2, s1]."""

    def __init__(self, n1, n2=1, n3=1, ng=3, dim=2, xstart=(0.0, 0.0, 0.0), xend=(1.0, 1.0, 1.0), bc=BC_PERIODIC,
                 model=EMHD, recon=MINMOD, limiter_theta=1.0, gamma=4.0 / 3.0, phi=1.0, psi=1.0, tau_mode=TAU_CONST,
                 tau=1.0, fd_eps=4e-8, eps_bt=1e-4, atol=0.0, rtol=1e-14, kmax=8, lsmax=5, cfl=0.5,
                 metric=MINKOWSKI, metric_params=(), device=0, stream=None, flux_ct=False, reduced=False, riemann=LLF,
                 closure=0):
        import torch
        self.torch = torch
        d = GridDesc()
        d.n1, d.n2, d.n3, d.ng, d.dim = n1, n2, n3, ng, dim
        for a in range(3):
            d.xstart[a], d.xend[a] = float(xstart[a]), float(xend[a])
            for s in range(2):
                d.bc[a][s] = bc if isinstance(bc, int) else bc[a][s]
        d.model, d.recon, d.limiter_theta, d.riemann = model, recon, limiter_theta, riemann
        d.gamma, d.phi, d.psi, d.tau_mode, d.tau = gamma, phi, psi, tau_mode, tau
        d.fd_eps, d.eps_bt, d.atol, d.rtol, d.kmax, d.lsmax, d.cfl = fd_eps, eps_bt, atol, rtol, kmax, lsmax, cfl
        d.device = device
        d.flux_ct = 1 if flux_ct else 0
        d.reduced_solve = 1 if reduced else 0
        d.closure = closure
        if stream is None and torch.cuda.is_available():
            stream = torch.cuda.current_stream(device).cuda_stream
        d.stream = stream
        self.desc = d
        self.h = _vp()
        self._L = lib()
        rc = self._L.grim_init_grid(C.byref(self.h), C.byref(d))
        if rc != 0:
            msg = self._L.grim_last_error(None)
            self.h = None
            raise GrimError("grim_init_grid failed (%d): %s" % (rc, msg.decode() if msg else ""))
        self.device = torch.device("cuda", device)
        self.nvar = model
        self.n = (n1, n2, n3)
        self.ngd = tuple(ng if a < dim else 0 for a in range(3))
        self.sz = tuple(self.n[a] + 2 * self.ngd[a] for a in range(3))
        self.shape = (model, self.sz[2], self.sz[1], self.sz[0])
        self.zg = self.sz[0] * self.sz[1] * self.sz[2]
        self.zones = n1 * n2 * n3
        self.set_metric(metric, metric_params)

    # -- plumbing ------------------------------------------------------------------------------------------
    def _check(self, rc, what):
        if rc != 0:
            msg = self._L.grim_last_error(self.h)
            raise GrimError("%s failed (%d): %s" % (what, rc, msg.decode() if msg else ""))

    def close(self):
        if getattr(self, "h", None):
            self._L.grim_free(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def zeros(self, nvar=None, dtype=None):
        t = self.torch
        shape = ((nvar,) if nvar else ()) + self.shape[1:]
        return t.zeros(shape, dtype=dtype or t.float64, device=self.device)

    def interior(self, A):
        g = self.ngd
        return A[..., g[2]:g[2] + self.n[2], g[1]:g[1] + self.n[1], g[0]:g[0] + self.n[0]]

    def launch_count(self):
        return int(self._L.grim_launch_count(self.h))

    def set_timing(self, on=True):
        self._check(self._L.grim_set_timing(self.h, 1 if on else 0), "grim_set_timing")

    def get_timing(self):
        """{class: (device ms, launches)} accumulated since set_timing(True)."""
        ms = (C.c_double * len(KERNEL_CLASSES))()
        n = (C.c_int64 * len(KERNEL_CLASSES))()
        self._check(self._L.grim_get_timing(self.h, ms, n), "grim_get_timing")
        return {k: (ms[i], n[i]) for i, k in enumerate(KERNEL_CLASSES)}

    # -- the entry points ----------------------------------------------------------------------------------
    def set_metric(self, kind, params=()):
        arr = (C.c_double * max(len(params), 1))(*[float(x) for x in params])
        self._check(self._L.grim_set_metric(self.h, kind, arr, len(params)), "grim_set_metric")

    def set_metric_tables(self, tab, conn):
        """tab: numpy float64 [4, 23, n2d]; conn: [64, n2d] (layout: include/grim.h)."""
        import numpy as np
        n2d = self.sz[0] * self.sz[1]
        tab = np.ascontiguousarray(tab, dtype=np.float64)
        conn = np.ascontiguousarray(conn, dtype=np.float64)
        if tab.shape != (4, 23, n2d) or conn.shape != (64, n2d):
            raise GrimError("set_metric_tables: expected shapes (4, 23, %d) and (64, %d)" % (n2d, n2d))
        self._check(self._L.grim_set_metric_tables(self.h, tab.ctypes.data_as(_pd), conn.ctypes.data_as(_pd)),
                    "grim_set_metric_tables")

    def fill_ghosts(self, P):
        self._check(self._L.grim_fill_ghosts(self.h, _ptr(P, self.torch.float64)), "grim_fill_ghosts")

    def compute_fluxes(self, P_E, P_n, dt_stage, C_out=None, G_out=None, speeds_out=None):
        f64 = self.torch.float64
        self._check(self._L.grim_compute_fluxes(self.h, _ptr(P_E, f64), _ptr(P_n, f64), dt_stage, _ptr(C_out, f64),
                                                _ptr(G_out, f64), _ptr(speeds_out, f64)), "grim_compute_fluxes")

    def newton_step(self, P_n, P_E, C_, G_, dt_stage, max_iters, P_iter, resnorm, status, iters, want_active=True):
        t = self.torch
        na = C.c_int64(0)
        self._check(self._L.grim_newton_step(self.h, _ptr(P_n, t.float64), _ptr(P_E, t.float64), _ptr(C_, t.float64),
                                             _ptr(G_, t.float64), dt_stage, max_iters, _ptr(P_iter, t.float64),
                                             _ptr(resnorm, t.float64), _ptr(status, t.int32), _ptr(iters, t.int32),
                                             C.byref(na) if want_active else None), "grim_newton_step")
        return na.value if want_active else None

    def newton_solve(self, P_n, P_E, C_, G_, dt_stage, P_guess, P_out, resnorm=None, status=None, iters=None):
        t = self.torch
        self._check(self._L.grim_newton_solve(self.h, _ptr(P_n, t.float64), _ptr(P_E, t.float64), _ptr(C_, t.float64),
                                              _ptr(G_, t.float64), dt_stage, _ptr(P_guess, t.float64),
                                              _ptr(P_out, t.float64), _ptr(resnorm, t.float64),
                                              _ptr(status, t.int32), _ptr(iters, t.int32)), "grim_newton_solve")

    def invert_primitives(self, U_target, P_inout, iters, status, resnorm, geom=None):
        """geom: None (Minkowski) or a [15, nz] CUDA tensor of per-zone geometry (layout: include/grim.h)."""
        t = self.torch
        nz = P_inout.shape[1]
        if geom is not None and tuple(geom.shape) != (15, nz):
            raise GrimError("invert_primitives: geom must have shape (15, %d)" % nz)
        self._check(self._L.grim_invert_primitives(self.h, nz, _ptr(U_target, t.float64), _ptr(geom, t.float64),
                                                   _ptr(P_inout, t.float64), _ptr(iters, t.int32),
                                                   _ptr(status, t.int32), _ptr(resnorm, t.float64)),
                    "grim_invert_primitives")

    def invert_primitives_host(self, U_host, P_host, iters_host=None, status_host=None, resnorm_host=None):
        t = self.torch
        nz = P_host.shape[1]
        self._check(self._L.grim_invert_primitives_host(self.h, nz, _host_ptr(U_host, t.float64),
                                                        _host_ptr(P_host, t.float64), _host_ptr(iters_host, t.int32),
                                                        _host_ptr(status_host, t.int32),
                                                        _host_ptr(resnorm_host, t.float64)),
                    "grim_invert_primitives_host")

    def prim_to_conserved(self, P, U):
        t = self.torch
        self._check(self._L.grim_prim_to_conserved(self.h, P.shape[1], _ptr(P, t.float64), _ptr(U, t.float64)),
                    "grim_prim_to_conserved")

    def timestep(self, P, dt=0.0, want_dt=False, want_stats=False):
        """One time step in place.  Returns (dt_used or None, StepStats or None)."""
        dtu = C.c_double(0.0)
        st = StepStats()
        self._check(self._L.grim_timestep(self.h, _ptr(P, self.torch.float64), dt, C.byref(dtu) if want_dt else None,
                                          C.byref(st) if want_stats else None), "grim_timestep")
        return (dtu.value if want_dt else None), (st if want_stats else None)

    def timestep_host(self, P_host, nsteps, dt=0.0):
        dtu = C.c_double(0.0)
        self._check(self._L.grim_timestep_host(self.h, _host_ptr(P_host, self.torch.float64), nsteps, dt,
                                               C.byref(dtu)), "grim_timestep_host")
        return dtu.value

    def last_host_mode(self):
        """'none' | 'whole' | 'pipelined': the form the last timestep_host call took (grim_last_host_mode)."""
        return HOST_MODES[self._L.grim_last_host_mode(self.h)]

    def get_geometry(self, loc, j, i):
        import numpy as np
        gcov, gcon, conn = np.zeros(16), np.zeros(16), np.zeros(64)
        sg, al, tau = C.c_double(), C.c_double(), C.c_double()
        dp = lambda a: a.ctypes.data_as(_pd)  # noqa: E731
        self._check(self._L.grim_get_geometry(self.h, loc, j * self.sz[0] + i, dp(gcov), dp(gcon), C.byref(sg),
                                              C.byref(al), C.byref(tau), dp(conn)), "grim_get_geometry")
        return gcov.reshape(4, 4), gcon.reshape(4, 4), sg.value, al.value, tau.value, conn.reshape(4, 4, 4)

    def fp64_probe(self, fma=True, iters=1 << 16):
        out = C.c_double(0.0)
        self._check(self._L.grim_fp64_probe(self.h, 1 if fma else 0, iters, C.byref(out)), "grim_fp64_probe")
        return out.value

    def arith_selftest(self, n, seed=0, wide=False):
        """-> (mismatches of [a/b, 1/b, sqrt, a/60, zero-tolerant variants], accepted a/b samples)"""
        out = (C.c_int64 * 6)()
        self._check(self._L.grim_arith_selftest(self.h, int(n), int(seed), 1 if wide else 0, out),
                    "grim_arith_selftest")
        return [int(x) for x in out[:5]], int(out[5])
