"""GPU parity of the general-metric path in THREE dimensions and at BASELINE's full sizes (configs 4 and 5: Kerr
a = 0.9375 in modified Kerr-Schild coordinates, 256 x 256 and 256 x 256 x 128), VERDICT r1 items 3-4.

The oracle's geometry tables are uploaded through grim_set_metric_tables, so every kernel sees the oracle's inputs
and the bar is bit equality: face_flux_kernel<.., GeomGen, dir 2>, the X^3 terms of the curved stage-constant
kernel, the connection source, the curved EMHD gradient terms and the Newton kernel with g_mu_nu.  The full-size
runs use the in-place, no-statistics branch of grim_timestep that bench.py times, and compare EVERY interior zone
with the oracle run on the whole grid (the Kerr grids are small enough for that: 6.6e4 and 8.4e6 zones).
"""
import numpy as np
import pytest

import oracle as og
from common import cuda_grid, oracle_grid, to_dev

pytestmark = pytest.mark.gpu

BC_KERR = [[og.BC_OUTFLOW, og.BC_OUTFLOW], [og.BC_REFLECT_POLAR, og.BC_REFLECT_POLAR],
           [og.BC_PERIODIC, og.BC_PERIODIC]]
KERR3D = dict(n1=20, n2=18, n3=12, ng=3, dim=3, xstart=(np.log(1.3), 0.0, 0.0), xend=(np.log(40.0), 1.0, 2 * np.pi),
              bc=BC_KERR, nvar=10, recon=og.MP5, limiter_theta=1.0, tau_mode=og.TAU_R32, metric=og.KERR_MKS,
              metric_params=(0.9375, 0.3), rtol=1e-13, kmax=8, lsmax=5)


def kerr_state_3d(go, seed, phi_amp=0.02):
    """The smooth admissible EMHD state of the 2-D Kerr tests with a phi-dependent modulation and seeded noise."""
    rng = np.random.default_rng(seed)
    X1, X2, X3 = go.centers()
    r = np.exp(X1)
    mod = 1 + phi_amp * np.sin(X3 + 0.4) * np.cos(2 * X3 + 2 * np.pi * X2)
    P = np.zeros(go.shape)
    P[0] = r ** -1.5 * (1 + 0.1 * np.sin(3 * X1) * np.cos(2 * np.pi * X2)) * mod
    P[1] = 0.1 * r ** -2.5 * (1 + 0.1 * np.cos(2 * X1 + 1.0)) * (2 - mod)
    P[2] = -0.05 / r * (1 + 0.2 * np.sin(2 * np.pi * X2))
    P[3] = 0.002 * np.sin(2 * np.pi * X2) / r * mod
    P[4] = 0.05 * r ** -1.5 * (1 + phi_amp * np.cos(X3))
    P[5] = 0.02 * r ** -3 * (1 + 0.3 * np.cos(np.pi * X2))
    P[6] = 0.002 * r ** -3 * np.sin(2 * np.pi * X2)
    P[7] = 0.01 * r ** -3 * (1 + phi_amp * np.sin(2 * X3))
    if go.nvar == 10:
        P[8] = 1e-3 * P[0] * (P[1] / (3 * P[0])) ** 1.5 * np.sin(2 * np.pi * X2 + 0.3 + X3)
        P[9] = 1e-2 * P[1] / 3 * np.cos(X1 + X3)
    P *= 1 + 1e-3 * rng.standard_normal(P.shape)
    go.fill_ghosts(P)
    return P


@pytest.mark.parametrize("opts", [dict(), dict(nvar=8, recon=og.MINMOD), dict(recon=og.MINMOD, limiter_theta=2.0),
                                  dict(flux_ct=True), dict(reduced=True), dict(riemann=1),
                                  dict(flux_ct=True, reduced=True, riemann=1, nvar=8, recon=og.MINMOD)])
def test_kerr_3d_timestep_bitwise_with_oracle_tables(opts):
    gk = dict(KERR3D, **opts)
    go, gc = oracle_grid(gk), cuda_grid(gk)
    gc.set_metric_tables(*go.geometry_tables())
    P0 = kerr_state_3d(go, 5)[:gk["nvar"]].copy()
    go.fill_ghosts(P0)
    dt = go.choose_dt(P0)
    Po, dP = P0.copy(), to_dev(P0)
    for _ in range(2):
        so = go.timestep(Po, dt)
        _, sc = gc.timestep(dP, dt, want_stats=True)
        for s in range(2):
            assert list(so.iters_hist[s]) == list(sc.iters_hist[s])
            assert so.unconverged[s] == sc.unconverged[s]
    assert np.isfinite(go.interior(Po)).all()
    assert np.array_equal(go.interior(dP.cpu().numpy()), go.interior(Po))


def test_kerr_3d_stage_pieces_bitwise():
    """grim_compute_fluxes (C, G, speeds) and per-iteration Newton in 3-D curved space, oracle tables."""
    import torch
    gk = dict(KERR3D)
    go, gc = oracle_grid(gk), cuda_grid(gk)
    gc.set_metric_tables(*go.geometry_tables())
    P0 = kerr_state_3d(go, 8)
    dt = 0.5 * go.choose_dt(P0)
    Co, Go, spo = go.stage_prepare(P0, P0, dt)
    dPn = to_dev(P0)
    dC, dG, dsp = gc.zeros(10), gc.zeros(3), torch.zeros(4, dtype=torch.float64, device="cuda")
    gc.compute_fluxes(dPn, dPn, dt, dC, dG, dsp)
    assert np.array_equal(go.interior(dC.cpu().numpy()), go.interior(Co))
    assert np.array_equal(go.interior(dG.cpu().numpy()), go.interior(Go))
    assert np.array_equal(dsp.cpu().numpy(), spo)
    Po = P0.copy()
    state = None
    dP = dPn.clone()
    drn, dst, dit = gc.zeros(), gc.zeros(dtype=torch.int32), gc.zeros(dtype=torch.int32)
    for it in range(3):
        nact, state, _ = go.newton(P0, P0, Co, Go, dt, Po, max_iters=1, state=state)
        nact_c = gc.newton_step(dPn, dPn, dC, dG, dt, 1, dP, drn, dst, dit)
        assert nact == nact_c
        assert np.array_equal(go.interior(dP.cpu().numpy()), go.interior(Po))
        assert np.array_equal(go.interior(dit.cpu().numpy()), go.interior(state[2]))
        assert np.array_equal(go.interior(dst.cpu().numpy()), go.interior(state[1]))
        assert np.array_equal(go.interior(drn.cpu().numpy()), go.interior(state[0]))


def _fullsize(n1, n2, n3, steps):
    from paper_1702_01106_b200 import workloads
    gk, P0 = workloads.kerr_synthetic(n1=n1, n2=n2, n3=n3)
    go, gc = oracle_grid(gk), cuda_grid(gk)
    gc.set_metric_tables(*go.geometry_tables())
    go.fill_ghosts(P0)
    dt = go.choose_dt(P0)
    dP = to_dev(P0)
    Po = P0
    for _ in range(steps):
        gc.timestep(dP, dt)                      # bench.py's branch: no statistics, P_{n+1} written in place
        go.timestep(Po, dt)
    got = gc.interior(dP).cpu().numpy()
    exp = go.interior(Po)
    assert np.isfinite(exp).all()
    assert np.array_equal(got, exp)


def test_config4_shape_fullsize_every_zone():
    """256 x 256 Kerr (BASELINE config 4's grid), smooth synthetic state with MP5, 3 time steps, every interior zone
    bit-equal to the oracle.  (Config 4 itself -- the torus, 100 steps -- is tests/test_gpu_torus.py.)"""
    _fullsize(256, 256, 1, 3)
