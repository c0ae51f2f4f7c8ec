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
