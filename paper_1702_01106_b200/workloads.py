"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs; recipes in DESIGN.md).

numpy only.  This module holds none of the method's arithmetic: it produces primitive-variable arrays (initial
data), guesses and grid descriptions, and serves both the oracle (tests, cpu_baseline) and the CUDA library
(tests, bench.py).  The linear-mode eigenvectors come from data/linear_modes.json, written by
oracle/write_mode_tables.py.  No public dataset is involved: the paper's tests are analytic initial data.
"""
import json
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))

_modes = None


def mode_tables():
    global _modes
    if _modes is None:
        with open(os.path.join(HERE, "data", "linear_modes.json")) as f:
            _modes = json.load(f)
    return _modes


def padded_centres(n, ngd, xstart, xend):
    """Zone-centre coordinates X^1, X^2, X^3 of the padded grid, each of shape [s3, s2, s1]."""
    ax = []
    for a in range(3):
        dx = (xend[a] - xstart[a]) / n[a]
        ax.append(xstart[a] + (np.arange(n[a] + 2 * ngd[a]) - ngd[a] + 0.5) * dx)
    X3, X2, X1 = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    return X1, X2, X3


def linear_mode_state(P0, modes, amp, X1, X2, X3):
    """P = P0 + amp * sum_m Re[dP_m exp(i (k_m . x + phase_m))]."""
    P0 = np.asarray(P0, dtype=np.float64)
    P = np.repeat(P0[:, None], X1.size, axis=1).reshape((len(P0),) + X1.shape).copy()
    for md in modes:
        k = md["k"]
        dP = np.asarray(md["dP_re"]) + 1j * np.asarray(md["dP_im"])
        ph = np.exp(1j * (k[0] * X1 + k[1] * X2 + k[2] * X3 + md.get("phase", 0.0)))
        P += amp * (dP[:, None, None, None] * ph[None]).real
    return P


def config1(n=64, amp=1e-4):
    """Ideal MHD, 2-D Minkowski, n x n periodic on [0,1]^2, fast mode k = (2 pi, 2 pi), minmod, LLF, cfl 0.5."""
    t = mode_tables()["config1"]
    grid = dict(n1=n, n2=n, n3=1, ng=3, dim=2, xstart=(0.0, 0.0, 0.0), xend=(1.0, 1.0, 1.0), nvar=8, recon=0,
                limiter_theta=1.0, gam=t["gamma"], rtol=1e-14, kmax=8, lsmax=5, cfl=0.5)
    X = padded_centres((n, n, 1), (3, 3, 0), grid["xstart"], grid["xend"])
    return grid, linear_mode_state(t["P0"], t["modes"], amp, *X)


def config3(n=128, amp=1e-4, dim=3, recon=1, ranks=1, rank=0):
    """EMHD, 3-D Minkowski, n^3 periodic on [0,1]^3, four seeded random-phase linear modes, MP5, LLF, cfl 0.5.
    The headline run is the same generator at n = 256.  ranks > 1: rank's slab of the n x n x (ranks n) grid on
    [0,1]^2 x [0,ranks] (dim = 2: of the n x (ranks n) grid on [0,1] x [0,ranks]; the modes have period 1, so the
    stacked grid is periodic too)."""
    t = mode_tables()["config3"]
    nn = (n, n, n if dim == 3 else 1)
    xs, xe = [0.0, 0.0, 0.0], [1.0, 1.0, 1.0]
    xs[dim - 1], xe[dim - 1] = float(rank), float(rank + 1)      # slabs along the slowest active direction
    grid = dict(n1=nn[0], n2=nn[1], n3=nn[2], ng=3, dim=dim, xstart=tuple(xs),
                xend=tuple(xe), nvar=10, recon=recon, limiter_theta=1.0, gam=t["gamma"],
                phi=t["phi"], psi=t["psi"], tau=t["tau"], rtol=1e-14, kmax=8, lsmax=5, cfl=0.5)
    ngd = (3, 3, 3 if dim == 3 else 0)
    X = padded_centres(nn, ngd, grid["xstart"], grid["xend"])
    return grid, linear_mode_state(t["P0"], t["modes"], amp, *X)


def config2(nz, seed=1702, nvar=8):
    """Standalone primitive recovery (BASELINE config 2): rho, u log-uniform in [1e-4, 1e2]; Lorentz factor
    uniform in [1, 10], isotropic direction; |B|^2/rho log-uniform in [1e-3, 1e2], isotropic; guess = P (1 + 0.1 xi),
    xi ~ U[-1,1] per component (C-20).  For nvar = 10, q and dP are small seeded fractions of rho Theta^{3/2} and
    of the pressure.  Returns (P_true, P_guess), each [nvar, nz]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    P = np.zeros((nvar, nz))
    P[0] = np.exp(rng.uniform(np.log(1e-4), np.log(1e2), nz))
    P[1] = np.exp(rng.uniform(np.log(1e-4), np.log(1e2), nz))
    W = rng.uniform(1.0, 10.0, nz)
    d = rng.standard_normal((3, nz))
    d /= np.linalg.norm(d, axis=0, keepdims=True)
    P[2:5] = np.sqrt(W * W - 1.0) * d
    Bsq = P[0] * np.exp(rng.uniform(np.log(1e-3), np.log(1e2), nz))
    d = rng.standard_normal((3, nz))
    d /= np.linalg.norm(d, axis=0, keepdims=True)
    P[5:8] = np.sqrt(Bsq) * d
    xi = rng.uniform(-1.0, 1.0, (nvar, nz))
    if nvar == 10:
        pg = P[1] / 3.0
        P[8] = 0.1 * rng.uniform(-1.0, 1.0, nz) * P[0] * (pg / P[0]) ** 1.5
        P[9] = 0.1 * rng.uniform(-1.0, 1.0, nz) * pg
    guess = P * (1.0 + 0.1 * xi)
    return P, guess


def kerr_synthetic(n1=256, n2=256, n3=128, nvar=10, seed=9375, a=0.9375, h=0.3):
    """Stand-in for BASELINE configs 4-5 (the Fishbone-Moncrief closed form is not in PAPER.md): a smooth seeded
    EMHD state on the same grid -- Kerr a = 0.9375 in modified Kerr-Schild coordinates (h = 0.3), X^1 = ln r in
    [ln 1.3, ln 40], X^2 in [0, 1], X^3 = phi in [0, 2 pi) (n3 = 1: 2-D), outflow / polar reflection / periodic
    boundaries, tau_R = r^{3/2}, closure coefficients 1, MP5 -- with power-law radial profiles, a poloidal-angle
    modulation and 0.1 % white noise.  Returns (grid description, P[nvar, s3, s2, s1]); ghosts are not filled."""
    dim = 3 if n3 > 1 else 2
    grid = dict(n1=n1, n2=n2, n3=n3, ng=3, dim=dim, nvar=nvar, recon=1, limiter_theta=1.0,
                xstart=(float(np.log(1.3)), 0.0, 0.0), xend=(float(np.log(40.0)), 1.0, float(2 * np.pi)),
                bc=[[1, 1], [2, 2], [0, 0]], tau_mode=1, metric=1, metric_params=(a, h), gam=4.0 / 3.0,
                phi=1.0, psi=1.0, rtol=1e-12, kmax=8, lsmax=5, cfl=0.5)
    ngd = (3, 3, 3 if dim == 3 else 0)
    X1, X2, _ = padded_centres((n1, n2, n3), ngd, grid["xstart"], grid["xend"])
    X1, X2 = X1[:1], X2[:1]
    r = np.exp(X1)
    s3 = n3 + 2 * ngd[2]
    P = np.zeros((nvar, s3) + X1.shape[1:])
    P[0] = r ** -1.5 * (1 + 0.1 * np.sin(3 * X1) * np.cos(2 * np.pi * X2))
    P[1] = 0.1 * r ** -2.5 * (1 + 0.1 * np.cos(2 * X1 + 1.0))
    P[2] = -0.05 / r * (1 + 0.2 * np.sin(2 * np.pi * X2))
    P[3] = 0.002 * np.sin(2 * np.pi * X2) / r
    P[4] = 0.05 * r ** -1.5
    P[5] = 0.02 * r ** -3 * (1 + 0.3 * np.cos(np.pi * X2))
    P[6] = 0.002 * r ** -3 * np.sin(2 * np.pi * X2)
    P[7] = 0.01 * r ** -3
    if nvar == 10:
        P[8] = 1e-3 * P[0] * (P[1] / (3 * P[0])) ** 1.5 * np.sin(2 * np.pi * X2 + 0.3)
        P[9] = 1e-2 * P[1] / 3 * np.cos(X1)
    rng = np.random.Generator(np.random.PCG64(seed))
    P *= 1 + 1e-3 * rng.standard_normal(P.shape)
    return grid, P


def firehose(n=64, alpha=1e-6):
    """Firehose-instability test of the paper (L583-601, eqs 58-65): 1-D Minkowski, periodic on [0,1], EMHD,
    rho = 1, u = 2, B^1 = 0.1, dP = -0.011 < -b^2, tau_R = 1e6, u^2 = 0.1628 alpha sin(2 pi x^1),
    B^2 = 0.9867 alpha cos(2 pi x^1) (eq 63 prints x^2, a misprint: the mode varies along B^1; reading G-12) --
    the linearly unstable Alfven mode with growth rate 0.1036.  Returns (grid description, P)."""
    grid = dict(n1=n, n2=1, n3=1, ng=3, dim=1, xstart=(0.0, 0.0, 0.0), xend=(1.0, 1.0, 1.0), nvar=10, recon=1,
                limiter_theta=1.0, gam=4.0 / 3.0, phi=1.0, psi=1.0, tau=1e6, rtol=1e-13, kmax=10, lsmax=5, cfl=0.5)
    X1, _, _ = padded_centres((n, 1, 1), (3, 0, 0), grid["xstart"], grid["xend"])
    P = np.zeros((10,) + X1.shape)
    P[0], P[1], P[5], P[9] = 1.0, 2.0, 0.1, -0.011
    P[3] = 0.1628 * alpha * np.sin(2 * np.pi * X1)
    P[6] = 0.9867 * alpha * np.cos(2 * np.pi * X1)
    return grid, P


def conduction(n=64, A=0.2, R2=0.005, B0=1e-4, k=4, chi=0.01, nu=0.01, tau=0.1):
    """Anisotropic-conduction test of the paper (L538-572, eqs 53-57): 2-D Minkowski, periodic on [0,1]^2, EMHD with
    the CONSTANT thermal diffusivity chi = 0.01 and tau_R = 0.1 the paper prescribes (closure = 1: chi = phi, nu = psi
    as constants; the paper gives no viscosity for this test, reading C-24: nu = chi), gamma = 4/3:
    rho = 1 - A exp(-r^2/R^2) about the centre of the box, u = 1 (pressure equilibrium), fluid at rest,
    B^1 = B0, B^2 = B0 sin(2 pi k x^1), q = dP = 0.  Returns (grid description, P)."""
    grid = dict(n1=n, n2=n, n3=1, ng=3, dim=2, xstart=(0.0, 0.0, 0.0), xend=(1.0, 1.0, 1.0), nvar=10, recon=1,
                limiter_theta=2.0, gam=4.0 / 3.0, phi=chi, psi=nu, closure=1, tau=tau, rtol=1e-13, kmax=10, lsmax=5,
                cfl=0.5)
    X1, X2, _ = padded_centres((n, n, 1), (3, 3, 0), grid["xstart"], grid["xend"])
    # periodic images of the blob are exp(-1/0.005) away: the nearest image only
    d1 = (X1 - 0.5 + 0.5) % 1.0 - 0.5
    d2 = (X2 - 0.5 + 0.5) % 1.0 - 0.5
    P = np.zeros((10,) + X1.shape)
    P[0] = 1.0 - A * np.exp(-(d1 * d1 + d2 * d2) / R2)
    P[1] = 1.0
    P[5] = B0
    P[6] = B0 * np.sin(2 * np.pi * k * X1)
    return grid, P


# ------------------------------------------------------------------------------------------------------------
# BASELINE configs 4-5: equilibrium torus around a Kerr black hole (Fishbone & Moncrief 1976; PAPER.md L645 item 6,
# L712).  PAPER.md prints no formula; the solution is re-derived here from what it is: a stationary, axisymmetric,
# purely rotating perfect fluid with constant l = u^t u_phi.  For u = u^t (d_t + Omega d_phi) the acceleration is
# a_mu = -d_mu ln u^t + l d_mu Omega (normalisation differentiated), and the relativistic Euler equation
# d_mu ln h = -a_mu integrates, for constant l, to
#     ln h = ln u^t - l Omega + const                                      (h = specific enthalpy),
# with Omega(r, theta) the root of  l (g_tt + 2 Omega g_tphi + Omega^2 g_phiphi) + g_tphi + Omega g_phiphi = 0
# (Boyer-Lindquist components) and l the value of u^t u_phi of the circular geodesic at the pressure maximum.
# ------------------------------------------------------------------------------------------------------------
def _bl_circular(a, l, r, th):
    """Boyer-Lindquist g_tt, g_tphi, g_phiphi at (r, theta); angular velocity and u^t of the flow with u^t u_phi = l.
    Returns (Omega, ut2) with ut2 = (u^t)^2 (non-positive or nan where no such time-like flow exists)."""
    s2 = np.sin(th) ** 2
    Sig = r * r + a * a * np.cos(th) ** 2
    Del = r * r - 2.0 * r + a * a
    AA = (r * r + a * a) ** 2 - Del * a * a * s2
    gtt, gtp, gpp = -(1.0 - 2.0 * r / Sig), -2.0 * a * r * s2 / Sig, AA * s2 / Sig
    qa, qb, qc = l * gpp, 2.0 * l * gtp + gpp, l * gtt + gtp
    with np.errstate(invalid="ignore", divide="ignore"):
        Om = -2.0 * qc / (qb + np.sqrt(qb * qb - 4.0 * qa * qc))       # the root that tends to -qc/qb for small l
        ut2 = -1.0 / (gtt + 2.0 * Om * gtp + Om * Om * gpp)
    return Om, ut2


def _mks_theta(X2, h):
    return np.pi * X2 + 0.5 * (1.0 - h) * np.sin(2.0 * np.pi * X2), np.pi * (1.0 + (1.0 - h) * np.cos(2.0 * np.pi * X2))


def _mks_gcov(a, h, X1, X2):
    """Covariant Kerr-Schild metric in the modified coordinates (t, X1 = ln r, X2, phi) (eqs 5-8), [4,4,...]."""
    r = np.exp(X1)
    th, dth = _mks_theta(X2, h)
    s2, Sig = np.sin(th) ** 2, r * r + a * a * np.cos(th) ** 2
    f = 2.0 * r / Sig
    g = np.zeros((4, 4) + np.shape(r))
    g[0, 0] = -(1.0 - f)
    g[0, 1] = g[1, 0] = f
    g[0, 3] = g[3, 0] = -a * f * s2
    g[1, 1] = 1.0 + f
    g[1, 3] = g[3, 1] = -a * s2 * (1.0 + f)
    g[2, 2] = Sig
    g[3, 3] = s2 * (Sig + a * a * s2 * (1.0 + f))
    L = [np.ones_like(r), r, dth, np.ones_like(r)]
    for m in range(4):
        for n in range(4):
            g[m, n] = g[m, n] * L[m] * L[n]
    return g, Sig * np.abs(np.sin(th)) * r * np.abs(dth)          # sqrt(-g)


def fm_torus(n1=256, n2=256, n3=1, nvar=10, a=0.9375, h=0.3, r_in=6.0, r_max=12.0, kappa=1e-3, gam=4.0 / 3.0,
             beta=100.0, seed_field=1e-5, noise=0.04, noise_phi=0.02, seed=9375, rho_floor=1e-4, u_floor=1e-6):
    """BASELINE config 4 (n3 = 1) / config 5 (n3 > 1): the equilibrium torus of the derivation above with inner edge
    r_in and pressure maximum r_max on an MKS grid (h = 0.3), X1 = ln r in [ln 1.3, ln 40], X2 in [0, 1], outflow /
    polar reflection / periodic boundaries, tau_R = r^{3/2}, closure coefficients 1, generalised minmod (theta = 1; reading
    C-25: an MP5 torus run waits for floors and limiters the paper does not print, see below); polytrope p = kappa rho^gam
    normalised to rho = 1 at the pressure maximum; outside it a static atmosphere rho_floor r^{-3/2}, u_floor r^{-5/2};
    single poloidal field loop A_phi = max(rho - 0.2, 0) scaled to 2 max(P_g) / max(b^2) = beta, plus a weak uniform
    vertical seed field (A_phi += seed_field r^2 sin^2 theta / 2) so that bhat (eqs 33-34) is defined everywhere;
    u <- u (1 + noise (xi - 1/2)), xi ~ U[0,1) seeded, drawn per (X1, X2) zone and extended axisymmetrically, times
    (1 + noise_phi (eta - 1/2)) per 3-D zone when n3 > 1.  noise = 0, beta = inf, seed_field = 0: the exact hydrodynamic
    equilibrium (oracle pin P-12(b)).  Returns (grid description, P[nvar, s3, s2, s1]); ghosts are not filled."""
    dim = 3 if n3 > 1 else 2
    # Reconstruction: generalised minmod, the paper's limiter for its nonlinear tests (L651).  BASELINE does not name one
    # for configs 4-5, and MP5 as read (C-6: acceptance test with the absolute eps = 1e-10) passes unlimited values for
    # data << 1e-5 -- negative internal energies on the faces of the torus edge, which the paper's (unprinted) floors
    # would catch.
    grid = dict(n1=n1, n2=n2, n3=n3, ng=3, dim=dim, nvar=nvar, recon=0, limiter_theta=1.0,
                xstart=(float(np.log(1.3)), 0.0, 0.0), xend=(float(np.log(40.0)), 1.0, float(2 * np.pi)),
                bc=[[1, 1], [2, 2], [0, 0]], tau_mode=1, metric=1, metric_params=(a, h), gam=gam,
                phi=1.0, psi=1.0, rtol=1e-12, kmax=8, lsmax=5, cfl=0.5)
    ngd = (3, 3, 3 if dim == 3 else 0)
    dx1 = (grid["xend"][0] - grid["xstart"][0]) / n1
    dx2 = 1.0 / n2
    x1c = grid["xstart"][0] + (np.arange(n1 + 6) - 3 + 0.5) * dx1
    x2c = (np.arange(n2 + 6) - 3 + 0.5) * dx2
    X2, X1 = np.meshgrid(x2c, x1c, indexing="ij")                   # [s2, s1]
    # l of the circular geodesic at the pressure maximum (equatorial, prograde: Omega = 1/(r^{3/2} + a))
    OmK = 1.0 / (r_max ** 1.5 + a)
    gtt, gtp, gpp = -(1.0 - 2.0 / r_max), -2.0 * a / r_max, (r_max ** 2 + a * a) + 2.0 * a * a / r_max
    l = (gtp + OmK * gpp) / -(gtt + 2.0 * OmK * gtp + OmK * OmK * gpp)

    def torus(X1_, X2_):
        """rho, u (normalised), Omega, u^t at MKS points; zero density outside the torus."""
        r = np.exp(X1_)
        th, _ = _mks_theta(X2_, h)
        Om, ut2 = _bl_circular(a, l, r, th)
        Om0, ut20 = _bl_circular(a, l, np.float64(r_in), np.float64(0.5 * np.pi))
        Omx, ut2x = _bl_circular(a, l, np.float64(r_max), np.float64(0.5 * np.pi))
        with np.errstate(invalid="ignore", divide="ignore"):
            lnh = 0.5 * np.log(ut2) - l * Om - (0.5 * np.log(ut20) - l * Om0)
        lnhx = 0.5 * np.log(ut2x) - l * Omx - (0.5 * np.log(ut20) - l * Om0)
        inside = np.isfinite(lnh) & (lnh > 0.0) & (r >= r_in)
        hm1 = np.where(inside, np.expm1(np.where(inside, lnh, 0.0)), 0.0)
        rho = (hm1 * (gam - 1.0) / (kappa * gam)) ** (1.0 / (gam - 1.0))
        rhox = (np.expm1(lnhx) * (gam - 1.0) / (kappa * gam)) ** (1.0 / (gam - 1.0))
        u = kappa * rho ** gam / (gam - 1.0) / rhox
        return rho / rhox, u, np.where(inside, Om, 0.0), np.where(inside, np.sqrt(np.where(inside, ut2, 1.0)), 1.0), inside

    rho, u, Om, ut, inside = torus(X1, X2)
    r = np.exp(X1)
    th, dth = _mks_theta(X2, h)
    Sig = r * r + a * a * np.cos(th) ** 2
    P2 = np.zeros((nvar,) + X1.shape)
    P2[0] = np.maximum(rho, rho_floor * r ** -1.5)
    P2[1] = np.maximum(u, u_floor * r ** -2.5)
    # u^mu = u^t (1, 0, 0, Omega) is the same in Boyer-Lindquist, Kerr-Schild and MKS components (u^r = u^theta = 0);
    # u~^i = u^i + alpha^2 g^{ti} u^t (C-9) with alpha^2 = 1/(1 + 2r/Sigma), g^{t X1} = (2r/Sigma)/r, g^{t X2} = g^{t phi} = 0
    f = 2.0 * r / Sig
    P2[2] = np.where(inside, (f / (1.0 + f)) / r * ut, 0.0)
    P2[4] = np.where(inside, ut * Om, 0.0)
    # magnetic field from A_phi at the zone corners (analytic density there): B^1 = -d_2 A / sqrt(-g), B^2 = d_1 A / sqrt(-g)
    if np.isfinite(beta) or seed_field != 0.0:
        x1f = grid["xstart"][0] + (np.arange(n1 + 7) - 3) * dx1
        x2f = (np.arange(n2 + 7) - 3) * dx2
        X2f, X1f = np.meshgrid(x2f, x1f, indexing="ij")
        gcov, sg = _mks_gcov(a, h, X1, X2)
        rf = np.exp(X1f)
        thf, _ = _mks_theta(X2f, h)

        def curl(A):
            B1 = -((A[1:, :-1] - A[:-1, :-1]) + (A[1:, 1:] - A[:-1, 1:])) / (2.0 * dx2 * sg)
            B2 = ((A[:-1, 1:] - A[:-1, :-1]) + (A[1:, 1:] - A[1:, :-1])) / (2.0 * dx1 * sg)
            return B1, B2

        B1s, B2s = curl(0.5 * seed_field * rf * rf * np.sin(thf) ** 2)
        if np.isfinite(beta):
            B1l, B2l = curl(np.maximum(torus(X1f, X2f)[0] - 0.2, 0.0))
            # b^2 of the loop field alone with the torus velocity: b^t = B^i u_i, b^i = (B^i + b^t u^i)/u^t (L248)
            ucon = np.stack([ut, np.zeros_like(ut), np.zeros_like(ut), ut * Om])
            ucov = np.einsum("mn...,n...->m...", gcov, ucon)
            bt = B1l * ucov[1] + B2l * ucov[2]
            bcon = np.stack([bt, (B1l + bt * ucon[1]) / ut, (B2l + bt * ucon[2]) / ut, bt * ucon[3] / ut])
            bsq = np.einsum("m...,mn...,n...->...", bcon, gcov, bcon)
            scale = np.sqrt(2.0 * (gam - 1.0) * u.max() / (beta * bsq.max()))
            B1s, B2s = B1s + scale * B1l, B2s + scale * B2l
        P2[5], P2[6] = B1s, B2s
    rng = np.random.Generator(np.random.PCG64(seed))
    if noise:
        P2[1] *= 1.0 + noise * (rng.uniform(size=X1.shape) - 0.5)
    s3 = n3 + 2 * ngd[2]
    P = np.repeat(P2[:, None], s3, axis=1)
    if dim == 3 and noise_phi:
        P[1] *= 1.0 + noise_phi * (rng.uniform(size=P[1].shape) - 0.5)
    return grid, np.ascontiguousarray(P)
