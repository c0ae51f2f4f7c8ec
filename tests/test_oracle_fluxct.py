"""Pins of the oracle's flux-CT (NEXT-1; section 4.2: Toth 2000's flux-CT "as in harm": face fluxes
of B averaged to the edges and back).  The paper prints no formula, so the pins are what the scheme is FOR and what a
wrong sign, a wrong neighbour or a missing factor would break:

* the cell-corner-centred div B (the representation flux-CT preserves, L329: "violations are at machine tolerance") is
  unchanged by time steps to round-off in 2-D and 3-D, while without flux-CT it drifts at truncation level;
* the summed conserved variables on a periodic grid are still unchanged (the averaged fluxes are still fluxes);
* in 1-D the scheme reduces to F^1(B^1) = 0: B^1 does not change at all;
* a uniform state is still a fixed point, bit for bit.
"""
import numpy as np
import pytest

import oracle as og
from common import oracle_grid, random_smooth_state


def corner_divb(P, g):
    """Toth's cell-corner div B on the padded grid: the X^d difference of B^d averaged over the 2^(dim-1) zones that
    share the corner in the transverse directions.  Returned on corners (i-1/2, j-1/2[, k-1/2]), shape sz-1."""
    dim = sum(1 for a in range(3) if g.ngd[a] > 0)
    out = 0.0
    for d in range(dim):
        B = P[5 + d]
        ax = 2 - d                                  # array axes are (k, j, i)
        D = np.diff(B, axis=ax) / g.dx[d]
        for t in range(dim):
            if t == d:
                continue
            at = 2 - t
            lo = [slice(None)] * 3
            hi = [slice(None)] * 3
            lo[at], hi[at] = slice(0, -1), slice(1, None)
            D = 0.5 * (D[tuple(lo)] + D[tuple(hi)])
        out = out + D
    return out


def interior_corners(d, g):
    sl = tuple(slice(g.ngd[a], g.ngd[a] + g.n[a]) if g.ngd[a] else slice(None) for a in (2, 1, 0))
    return d[sl]


@pytest.mark.parametrize("dim,nvar,recon", [(2, 8, og.MINMOD), (2, 10, og.MP5), (3, 10, og.MINMOD), (3, 8, og.MP5)])
def test_corner_divb_preserved_only_with_flux_ct(dim, nvar, recon):
    n = (14, 11, 9 if dim == 3 else 1)
    drift = {}
    for ct in (False, True):
        g = oracle_grid(dict(n1=n[0], n2=n[1], n3=n[2], dim=dim, nvar=nvar, recon=recon, flux_ct=ct))
        P = random_smooth_state(g, nvar, np.random.default_rng(11), amp=0.05)
        g.fill_ghosts(P)
        d0 = interior_corners(corner_divb(P, g), g)
        dt = g.choose_dt(P)
        for _ in range(4):
            st = g.timestep(P, dt)
            assert st.unconverged[1] == 0
        g.fill_ghosts(P)
        d1 = interior_corners(corner_divb(P, g), g)
        drift[ct] = abs(d1 - d0).max()
        scale = abs(P[5:8]).max() / min(g.dx[:dim])
    assert drift[True] < 1e-13 * scale, drift
    assert drift[False] > 1e-4 * scale, drift          # the same steps without flux-CT move it at truncation level


def test_conservation_with_flux_ct():
    g = oracle_grid(dict(n1=12, n2=10, n3=8, dim=3, nvar=8, recon=og.MP5, flux_ct=True, kmax=10))
    P = random_smooth_state(g, 8, np.random.default_rng(3), amp=0.05)
    g.fill_ghosts(P)
    m, geo = og.model(nvar=8), og.minkowski()

    def total(P):
        Pi = g.interior(P).reshape(8, -1)
        return sum(og.prim_to_U(m, geo, 1.0, Pi[:, z]) for z in range(Pi.shape[1]))

    U0 = total(P)
    g.timestep(P, g.choose_dt(P))
    U1 = total(P)
    assert np.max(abs(U1 - U0)) < 1e-11 * abs(U0).max()


def test_one_dimension_keeps_b1_exactly():
    g = oracle_grid(dict(n1=40, n2=1, n3=1, dim=1, nvar=10, recon=og.MP5, flux_ct=True))
    P = random_smooth_state(g, 10, np.random.default_rng(5), amp=0.05)
    P[5] = 0.3                                           # div B = 0 in 1-D means B^1 uniform
    g.fill_ghosts(P)
    P0 = P.copy()
    for _ in range(3):
        g.timestep(P, 0.004)
    assert np.array_equal(g.interior(P)[5], g.interior(P0)[5])
    assert not np.array_equal(g.interior(P)[6], g.interior(P0)[6])


def test_uniform_state_is_a_fixed_point():
    g = oracle_grid(dict(n1=8, n2=7, n3=6, dim=3, nvar=10, recon=og.MP5, flux_ct=True))
    P = g.zeros()
    for v, x in enumerate([1.0, 2.0, 0.1, -0.2, 0.15, 0.1, 0.3, -0.2, 0.0, 0.0]):
        P[v] = x
    P0 = P.copy()
    g.timestep(P, 0.01)
    # q, dP relax towards their (zero-gradient) targets = 0 and stay 0; everything else is untouched
    assert np.array_equal(g.interior(P), g.interior(P0))
