"""Shared helpers of the parity tests: build the oracle grid and the CUDA-library grid from one description."""
import numpy as np

import oracle as og


def oracle_grid(gk, **over):
    k = dict(gk)
    k.update(over)
    return og.Grid(k["n1"], k.get("n2", 1), k.get("n3", 1), ng=k.get("ng", 3), dim=k.get("dim", 2),
                   xstart=k.get("xstart", (0, 0, 0)), xend=k.get("xend", (1, 1, 1)), bc=k.get("bc", og.BC_PERIODIC),
                   nvar=k.get("nvar", 10), recon=k.get("recon", 0), limiter_theta=k.get("limiter_theta", 1.0),
                   gam=k.get("gam", 4.0 / 3.0), phi=k.get("phi", 1.0), psi=k.get("psi", 1.0),
                   tau_mode=k.get("tau_mode", 0), tau=k.get("tau", 1.0), fd_eps=k.get("fd_eps", 4e-8),
                   eps_bt=k.get("eps_bt", 1e-4), atol=k.get("atol", 0.0), rtol=k.get("rtol", 1e-14),
                   kmax=k.get("kmax", 8), lsmax=k.get("lsmax", 5), cfl=k.get("cfl", 0.5),
                   metric=k.get("metric", 0), metric_params=k.get("metric_params", ()),
                   flux_ct=k.get("flux_ct", False), reduced=k.get("reduced", False),
                   riemann=k.get("riemann", 0), closure=k.get("closure", 0))


def cuda_grid(gk, **over):
    import paper_1702_01106_b200 as gb
    k = dict(gk)
    k.update(over)
    return gb.Grid(k["n1"], k.get("n2", 1), k.get("n3", 1), ng=k.get("ng", 3), dim=k.get("dim", 2),
                   xstart=k.get("xstart", (0, 0, 0)), xend=k.get("xend", (1, 1, 1)), bc=k.get("bc", 0),
                   model=k.get("nvar", 10), recon=k.get("recon", 0), limiter_theta=k.get("limiter_theta", 1.0),
                   gamma=k.get("gam", 4.0 / 3.0), phi=k.get("phi", 1.0), psi=k.get("psi", 1.0),
                   tau_mode=k.get("tau_mode", 0), tau=k.get("tau", 1.0), fd_eps=k.get("fd_eps", 4e-8),
                   eps_bt=k.get("eps_bt", 1e-4), atol=k.get("atol", 0.0), rtol=k.get("rtol", 1e-14),
                   kmax=k.get("kmax", 8), lsmax=k.get("lsmax", 5), cfl=k.get("cfl", 0.5),
                   metric=k.get("metric", 0), metric_params=k.get("metric_params", ()),
                   flux_ct=k.get("flux_ct", False), reduced=k.get("reduced", False), riemann=k.get("riemann", 0),
                   closure=k.get("closure", 0))


def to_dev(a, dtype=None):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t if dtype is None else t.to(dtype)


def rel_err_per_primitive(A, B, interior=None, gam=None):
    """north_star metric: max over zones of |A-B| / max(|B|, floor_v), floor_v = 1e-12 max_z|B_v|; velocity and
    field components relative to the norm of their vector.  With gam given, q and dP (which change
    sign and pass through zero inside the domain) are measured against max(|q|, 1e-3 rho Theta^{3/2}) and
    max(|dP|, 1e-3 P_g): a thousandth of their free-streaming / isotropic-pressure scale."""
    if interior is not None:
        A, B = interior(A), interior(B)
    nv = A.shape[0]
    out = np.zeros(nv)
    if gam is not None and nv == 10:
        pg = (gam - 1.0) * abs(B[1])
        nat = {8: 1e-3 * abs(B[0]) * (pg / abs(B[0])) ** 1.5, 9: 1e-3 * pg}
    else:
        nat = {}
    def vecnorm(X, lo):
        return np.sqrt((X[lo:lo + 3] ** 2).sum(axis=0))
    for v in range(nv):
        if 2 <= v <= 4:
            ref = vecnorm(B, 2)
        elif 5 <= v <= 7:
            ref = vecnorm(B, 5)
        else:
            ref = abs(B[v])
        floor = 1e-12 * max(ref.max(), 1e-300)
        if v in nat:
            ref = np.maximum(ref, nat[v])
        out[v] = (abs(A[v] - B[v]) / np.maximum(ref, floor)).max()
    return out


def random_smooth_state(g, nvar, rng, amp=0.05):
    """Smooth-ish positive random primitives on the padded grid of oracle grid g (ghosts NOT yet consistent)."""
    X1, X2, X3 = g.centers()
    P = np.zeros(g.shape)
    base = [1.0, 2.0, 0.1, -0.2, 0.15, 0.1, 0.3, -0.2, 0.01, 0.02][:nvar]
    for v in range(nvar):
        ph = rng.uniform(0, 2 * np.pi, 3)
        P[v] = base[v] + amp * (np.sin(2 * np.pi * X1 + ph[0]) + np.cos(2 * np.pi * X2 + ph[1])
                                + np.sin(2 * np.pi * X3 + ph[2])) * (abs(base[v]) + 0.1)
        P[v] += 0.01 * amp * rng.standard_normal(P[v].shape)
    return P
