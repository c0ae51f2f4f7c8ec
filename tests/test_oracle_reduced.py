"""Pins of the oracle's reduced solve (NEXT-2; "equations without implicitly coupled source terms are
treated explicitly, and do not require the nonlinear solver"; L643: a 5 x 5 Jacobian for ideal MHD, 7 x 7 for EMHD).
B^i is advanced explicitly from the flux divergence, Newton runs on the other nvar - 3 primitives.

* It solves the same equations: after time steps the result agrees with the full nvar-unknown solve to the Newton
  tolerance (both converge to the root of the same residual; the B^i rows are linear and exact either way).
* The B^i update is exactly the discrete induction equation: U(B) changes by -dt times the flux divergence, so the
  summed conserved variables are unchanged on a periodic grid and, with flux-CT, the corner div B stays at round-off.
* The iteration counts do not exceed those of the full solve on smooth data (fewer unknowns, same contraction).
"""
import numpy as np
import pytest

import oracle as og
from common import oracle_grid, random_smooth_state
from test_oracle_fluxct import corner_divb, interior_corners


@pytest.mark.parametrize("dim,nvar,recon", [(2, 8, og.MINMOD), (2, 10, og.MP5), (3, 10, og.MINMOD)])
def test_reduced_solve_reaches_the_root_of_the_full_solve(dim, nvar, recon):
    n = (14, 11, 9 if dim == 3 else 1)
    out, iters = {}, {}
    for red in (False, True):
        g = oracle_grid(dict(n1=n[0], n2=n[1], n3=n[2], dim=dim, nvar=nvar, recon=recon, reduced=red))
        P = random_smooth_state(g, nvar, np.random.default_rng(21), amp=0.05)
        g.fill_ghosts(P)
        dt = g.choose_dt(P)
        tot = 0
        for _ in range(3):
            st = g.timestep(P, dt)
            assert st.unconverged[0] == 0 and st.unconverged[1] == 0
            tot += sum(i * st.iters_hist[s][i] for s in range(2) for i in range(16))
        out[red], iters[red] = g.interior(P).copy(), tot
    scale = abs(out[False]).reshape(nvar, -1).max(axis=1)
    err = abs(out[True] - out[False]).reshape(nvar, -1).max(axis=1)
    assert (err < 1e-12 * np.maximum(scale, 1.0)).all(), err
    assert iters[True] <= iters[False]


def test_reduced_solve_conserves_and_keeps_divb_with_flux_ct():
    g = oracle_grid(dict(n1=12, n2=10, n3=8, dim=3, nvar=10, recon=og.MP5, reduced=True, flux_ct=True))
    P = random_smooth_state(g, 10, np.random.default_rng(8), amp=0.05)
    g.fill_ghosts(P)
    m, geo = og.model(nvar=10), og.minkowski()

    def total(P):
        Pi = g.interior(P).reshape(10, -1)
        return sum(og.prim_to_U(m, geo, 1.0, Pi[:, z]) for z in range(Pi.shape[1]))

    U0, d0 = total(P), interior_corners(corner_divb(P, g), g)
    dt = g.choose_dt(P)
    for _ in range(3):
        g.timestep(P, dt)
    g.fill_ghosts(P)
    U1, d1 = total(P), interior_corners(corner_divb(P, g), g)
    assert np.max(abs(U1[:8] - U0[:8])) < 1e-11 * abs(U0).max()
    assert abs(d1 - d0).max() < 1e-13 * abs(P[5:8]).max() / min(g.dx)


def test_reduced_b_update_is_the_explicit_induction_step():
    """One stage by hand: B_new = B_n - dt' divF_B, with divF_B read off the stage constant of the full path."""
    g = oracle_grid(dict(n1=10, n2=9, n3=1, dim=2, nvar=8, recon=og.MINMOD, reduced=True))
    P = random_smooth_state(g, 8, np.random.default_rng(2), amp=0.05)
    g.fill_ghosts(P)
    dts = 0.003
    C, G, _ = g.stage_prepare(P, P, dts)
    Pit = P.copy()
    nact, (rn, st, it), _ = g.newton(P, P, C, G, dts, Pit)
    assert nact == 0
    divF_B = g.interior(C)[5:8] + g.interior(P)[5:8] / dts          # C = -U(P_n)/dt' + divF, U(B) = B (Minkowski)
    expect = g.interior(P)[5:8] - dts * divF_B
    assert np.allclose(g.interior(Pit)[5:8], expect, rtol=0, atol=1e-14)
    assert (g.interior(st) & og.ST_CONVERGED).all()
