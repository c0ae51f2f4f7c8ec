"""Grid-level oracle pins: Table 1 evolution converges at 2nd order (P-2), conservation (P-7), round-trip
inversion (P-8), Newton behaviour (P-11), ghost fill.  CPU only."""
import numpy as np
import pytest

import oracle as og


def table1_state(grid, table1, A, t):
    P0, dP, w, k = table1
    X1, X2, X3 = grid.centers()
    ph = np.exp(1j * (k[0] * X1 + k[1] * X2) + w * t)
    return P0[:, None, None, None] + A * (dP[:, None, None, None] * ph[None]).real


def run_table1(N, table1, theta, A=1e-8, tfinal=0.5, recon=og.MINMOD):
    g = og.Grid(N, N, 1, ng=3, dim=2, nvar=10, recon=recon, limiter_theta=theta, rtol=1e-14, kmax=8)
    P = table1_state(g, table1, A, 0.0)
    dt0 = g.choose_dt(P)
    nsteps = int(np.ceil(tfinal / dt0))
    dt = tfinal / nsteps
    hist = np.zeros(16, dtype=np.int64)
    for _ in range(nsteps):
        st = g.timestep(P, dt)
        hist += np.array(st.iters_hist[0][:]) + np.array(st.iters_hist[1][:])
        assert st.unconverged[0] == 0 and st.unconverged[1] == 0
    err = abs(g.interior(P) - g.interior(table1_state(g, table1, A, tfinal))).mean(axis=(1, 2, 3)) / A
    return err, hist


def test_table1_evolution_second_order(table1):
    """PAPER.md L499-507 (Fig 4): L1 error of the evolved Table-1 mode at t = 0.5 falls at 2nd order.
    theta = 2 (monotonised-central end of the generalised minmod family, L115) because strict minmod clips
    the extrema of a sinusoid and is only ~1st order there (SURVEY hard part 6)."""
    e = [run_table1(N, table1, 2.0)[0].sum() for N in (16, 32, 64)]
    o1, o2 = np.log2(e[0] / e[1]), np.log2(e[1] / e[2])
    assert e[2] < 0.03 and o1 > 1.8 and o2 > 1.9, (e, o1, o2)


def test_table1_evolution_mp5_converges_faster(table1):
    e = [run_table1(N, table1, 2.0, recon=og.MP5)[0].sum() for N in (16, 32)]
    assert np.log2(e[0] / e[1]) > 1.9 and e[1] < 0.06, e


def test_table1_decay_rate(table1):
    """The mode both propagates and decays (L499): amplitude of u at t=0.5 is exp(Re w t) of the initial."""
    P0, dP, w, k = table1
    N, A = 64, 1e-8
    g = og.Grid(N, N, 1, ng=3, dim=2, nvar=10, recon=og.MP5, limiter_theta=2.0, rtol=1e-14, kmax=8)
    P = table1_state(g, table1, A, 0.0)
    dt = 0.5 / int(np.ceil(0.5 / g.choose_dt(P)))
    for _ in range(int(round(0.5 / dt))):
        g.timestep(P, dt)
    amp = np.sqrt(2 * np.mean((g.interior(P)[1] - 2.0) ** 2)) / (A * abs(dP[1]))
    assert abs(amp - np.exp(w.real * 0.5)) < 5e-3


@pytest.mark.parametrize("nvar,recon,dim", [(8, og.MINMOD, 2), (10, og.MP5, 2), (10, og.MINMOD, 3)])
def test_conservation_periodic(nvar, recon, dim):
    """P-7 (L19, L536): on a periodic Minkowski grid the summed conserved variables of rows 0-7 are unchanged
    by a step, to Newton tolerance + round-off."""
    rng = np.random.default_rng(7)
    n = (12, 10, 8 if dim == 3 else 1)
    g = og.Grid(*n, ng=3, dim=dim, nvar=nvar, recon=recon, limiter_theta=1.5, rtol=1e-14, kmax=10)
    P = g.zeros()
    X1, X2, X3 = g.centers()
    P[0] = 1 + 0.3 * np.sin(2 * np.pi * X1) * np.cos(2 * np.pi * X2)
    P[1] = 2 + 0.5 * np.cos(2 * np.pi * (X1 + X2 + (X3 if dim == 3 else 0)))
    P[2] = 0.2 * np.sin(2 * np.pi * X2); P[3] = -0.1 * np.cos(2 * np.pi * X1); P[4] = 0.05
    P[5] = 0.3; P[6] = 0.2 + 0.1 * np.sin(2 * np.pi * X1); P[7] = 0.1
    if nvar == 10:
        P[8] = 0.01 * np.sin(2 * np.pi * X1); P[9] = 0.02 * np.cos(2 * np.pi * X2)
    m, geo = og.model(nvar=nvar), og.minkowski()

    def total(P):
        Pi = g.interior(P).reshape(nvar, -1)
        return sum(og.prim_to_U(m, geo, 1.0, Pi[:, z]) for z in range(Pi.shape[1]))

    U0 = total(P)
    dt = g.choose_dt(P)
    st = g.timestep(P, dt)
    assert st.unconverged[1] == 0
    U1 = total(P)
    scale = abs(U0).max()
    assert np.max(abs(U1[:8] - U0[:8])) < 1e-11 * scale
    if nvar == 10:   # rows 8-9 have sources: they do change
        assert np.max(abs(U1[8:] - U0[8:])) > 1e-8


def _cfg2_like(rng, nz, nvar=8):
    P = np.zeros((nvar, nz))
    P[0] = np.exp(rng.uniform(np.log(1e-4), np.log(1e2), nz))
    P[1] = np.exp(rng.uniform(np.log(1e-4), np.log(1e2), nz))
    W = rng.uniform(1, 10, nz)
    n = rng.standard_normal((3, nz)); n /= np.linalg.norm(n, axis=0)
    P[2:5] = np.sqrt(W * W - 1) * n
    B2 = P[0] * np.exp(rng.uniform(np.log(1e-3), np.log(1e2), nz))
    n = rng.standard_normal((3, nz)); n /= np.linalg.norm(n, axis=0)
    P[5:8] = np.sqrt(B2) * n
    return P


def test_round_trip_inversion():
    """P-8: P -> U(P) -> Newton from a +-10% guess -> P' ; converged zones reproduce U to rtol, and the
    primitives to 1e-9 where the problem is well conditioned."""
    rng = np.random.default_rng(1702)
    nz = 4000
    P = _cfg2_like(rng, nz)
    m, geo = og.model(nvar=8), og.minkowski()
    U = np.stack([og.prim_to_U(m, geo, 1.0, P[:, z]) for z in range(nz)], axis=1)
    guess = P * (1 + 0.1 * rng.uniform(-1, 1, P.shape))
    s = og.solver(rtol=1e-12, kmax=30, lsmax=8)
    Pr, iters, status, resnorm, bt = og.invert(m, s, U, guess)
    conv = (status & og.ST_CONVERGED) != 0
    assert conv.mean() > 0.9
    assert np.all(resnorm[conv] < 1e-12) and np.all(iters[conv] >= 1) and np.all(iters <= 30)
    assert np.all(((status & og.ST_KMAX) != 0) == (~conv & ((status & (og.ST_SINGULAR | og.ST_NONFINITE)) == 0)))
    U2 = np.stack([og.prim_to_U(m, geo, 1.0, Pr[:, z]) for z in range(nz)], axis=1)
    rel = np.linalg.norm(U2 - U, axis=0) / np.linalg.norm(U, axis=0)
    assert np.all(rel[conv] < 1.01e-12)
    # B is recovered exactly-ish (linear rows); the rest where magnetisation and W are moderate
    assert np.max(abs(Pr[5:8, conv] - P[5:8, conv]) / np.linalg.norm(P[5:8, conv], axis=0)) < 1e-11
    W = np.sqrt(1 + (P[2:5] ** 2).sum(0))
    well = conv & (W < 3) & ((P[5:8] ** 2).sum(0) / P[0] < 1) & (P[1] / P[0] > 1e-2)
    assert well.sum() > 50
    assert np.max(abs(Pr[:2, well] - P[:2, well]) / P[:2, well]) < 1e-9


def test_round_trip_inversion_kerr_point_geometry():
    """O-10 with geom_or_null given: every zone has its own Kerr (MKS, a = 0.9375) geometry.  P -> U(P) with
    og_prim_to_U in that zone's geometry (itself pinned by the trace / Eckart-frame identities in Kerr) -> Newton from
    a +-5 % guess -> P'.  A zone solved with another zone's geometry (or the Minkowski one) misses U by O(1)."""
    rng = np.random.default_rng(9375)
    nz = 600
    P = _cfg2_like(rng, nz)
    P[2:5] *= 0.2 / np.maximum(1.0, np.sqrt((P[2:5] ** 2).sum(0)))[None]      # moderate velocities: well conditioned
    X1 = rng.uniform(np.log(1.5), np.log(40.0), nz)
    X2 = rng.uniform(0.05, 0.95, nz)
    geoms = [og.kerr_mks(0.9375, 0.3, X1[z], X2[z]) for z in range(nz)]
    m = og.model(nvar=8)
    U = np.stack([og.prim_to_U(m, geoms[z], 1.0, P[:, z]) for z in range(nz)], axis=1)
    guess = P * (1 + 0.05 * rng.uniform(-1, 1, P.shape))
    s = og.solver(rtol=1e-12, kmax=30, lsmax=8)
    Pr, iters, status, resnorm, bt = og.invert(m, s, U, guess, geoms=geoms)
    conv = (status & og.ST_CONVERGED) != 0
    assert conv.mean() > 0.9
    U2 = np.stack([og.prim_to_U(m, geoms[z], 1.0, Pr[:, z]) for z in range(nz)], axis=1)
    rel = np.linalg.norm(U2 - U, axis=0) / np.linalg.norm(U, axis=0)
    assert np.all(rel[conv] < 1.01e-12)
    well = conv & ((P[5:8] ** 2).sum(0) / P[0] < 1) & (P[1] / P[0] > 1e-2) & (P[1] / P[0] < 1e2)
    assert well.sum() > 30
    assert np.max(abs(Pr[:2, well] - P[:2, well]) / P[:2, well]) < 1e-6      # conditioning x the 1e-12 residual
    # negative control: the same targets solved in the wrong geometry (zone z+1's) do not reproduce P
    Pw, _, stw, _, _ = og.invert(m, s, U, guess, geoms=geoms[1:] + geoms[:1])
    bad = abs(Pw[:2, well] - P[:2, well]) / P[:2, well]
    assert np.nanmedian(bad.max(axis=0)) > 1e-3


def test_inversion_hydro_against_bisection():
    """P-11(iv): brute force.  B = 0 hydrodynamics reduces to a scalar equation for the pressure; solve it by
    bisection in numpy and compare with the oracle's Newton result."""
    rng = np.random.default_rng(5)
    gam = 4.0 / 3.0
    nz = 200
    P = _cfg2_like(rng, nz)
    P[5:8] = 0
    P[0] = np.exp(rng.uniform(-2, 2, nz)); P[1] = np.exp(rng.uniform(-2, 2, nz))
    m, geo = og.model(nvar=8, gam=gam), og.minkowski()
    U = np.stack([og.prim_to_U(m, geo, 1.0, P[:, z]) for z in range(nz)], axis=1)
    Pr, iters, status, resnorm, bt = og.invert(m, og.solver(rtol=1e-13, kmax=40), U, P * (1 + 0.1 * rng.uniform(-1, 1, P.shape)))
    for z in range(nz):
        if not status[z] & og.ST_CONVERGED:
            continue
        D, E, S = U[0, z], -U[1, z], U[2:5, z]          # D = rho W, E = -T^t_t = w W^2 - p, S_i = w W u_i
        S2 = S @ S

        def f(p):                                      # textbook 1-D reduction: unknown pressure
            v2 = S2 / (E + p) ** 2
            W = 1 / np.sqrt(1 - v2)
            rho = D / W
            eps_u = (E + p) / W ** 2 - rho - p          # u = w - rho - p with w = (E+p)/W^2
            return (gam - 1) * eps_u - p

        lo, hi = max(0.0, np.sqrt(S2) - E) * (1 + 1e-14) + 1e-300, 10 * (E + 1)
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            lo, hi = (mid, hi) if f(mid) > 0 else (lo, mid)
        p = 0.5 * (lo + hi)
        assert abs((gam - 1) * Pr[1, z] - p) < 1e-8 * p


def test_newton_linear_problem_one_iteration_and_jacobian_accuracy():
    """P-11(i,ii): B rows of the step residual are linear, R_B = (B - B_n)/dt' + C_B: one Newton iteration
    leaves them at round-off; and the residual function's FD Jacobian matches a central-difference one."""
    g = og.Grid(8, 8, 1, ng=2, dim=2, nvar=10, recon=og.MINMOD, limiter_theta=1.0, rtol=0.0, atol=0.0, kmax=1)
    X1, X2, X3 = g.centers()
    P = g.zeros()
    P[0] = 1 + 0.2 * np.sin(2 * np.pi * X1); P[1] = 2 + 0.2 * np.cos(2 * np.pi * X2)
    P[2] = 0.1 * np.sin(2 * np.pi * X2); P[5] = 0.1; P[6] = 0.3 + 0.05 * np.sin(2 * np.pi * X1)
    P[8] = 0.01; P[9] = -0.01
    g.fill_ghosts(P)
    dt = 0.5 * g.choose_dt(P)
    C, G, sp = g.stage_prepare(P, P, dt)
    Pit = P.copy()
    nact, (rn, st, it), bt = g.newton(P, P, C, G, dt, Pit, max_iters=1)
    z = (0 * g.sz[1] + 5) * g.sz[0] + 4
    R = g.zone_residual(z, P, P, C, G, dt, Pit.reshape(10, -1)[:, z])
    R0 = g.zone_residual(z, P, P, C, G, dt, P.reshape(10, -1)[:, z])
    # linear rows: solved by one iteration up to the FD Jacobian's rounding (~eps_machine/fd_eps ~ 3e-9)
    assert np.max(abs(R[5:8])) < 1e-7 * np.max(abs(R0[5:8]))
    assert np.linalg.norm(R) < 1e-2 * np.linalg.norm(R0)     # nonlinear rows: one Newton step of a 20% amplitude problem
    # FD Jacobian (eq 22-23) vs central differences
    Pz = P.reshape(10, -1)[:, z].copy()
    eps = 4e-8
    J = np.zeros((10, 10)); Jc = np.zeros((10, 10))
    for j in range(10):
        pe = Pz.copy(); pe[j] = eps if abs(Pz[j]) < 5 * eps else (1 + eps) * Pz[j]
        J[:, j] = (g.zone_residual(z, P, P, C, G, dt, pe) - R0) / (pe[j] - Pz[j])
        h = 1e-5 * max(abs(Pz[j]), 1e-2)
        pp, pm = Pz.copy(), Pz.copy(); pp[j] += h; pm[j] -= h
        Jc[:, j] = (g.zone_residual(z, P, P, C, G, dt, pp) - g.zone_residual(z, P, P, C, G, dt, pm)) / (2 * h)
    assert np.max(abs(J - Jc)) < 2e-5 * np.max(abs(Jc))
    # B block: J_BB = I/dt', J_B,other = 0 (C-1)
    assert np.allclose(J[5:8, 5:8], np.eye(3) / dt, rtol=1e-6) and np.max(abs(J[5:8, :5])) < 1e-6


def test_newton_quadratic_convergence_and_stepwise_equals_whole():
    """P-11(iii): residual falls ~quadratically to the FD floor; running k single-iteration calls gives the
    same bits as one whole solve (C-13 / SURVEY 7.2 'both must give bit-identical results')."""
    g = og.Grid(8, 6, 1, ng=2, dim=2, nvar=10, recon=og.MINMOD, rtol=1e-14, kmax=6)
    X1, X2, X3 = g.centers()
    P = g.zeros()
    P[0] = 1 + 0.3 * np.sin(2 * np.pi * X1); P[1] = 2 + 0.3 * np.cos(2 * np.pi * X2)
    P[2] = 0.2 * np.sin(2 * np.pi * X2); P[3] = 0.1; P[5] = 0.1; P[6] = 0.3; P[8] = 0.02; P[9] = 0.01
    g.fill_ghosts(P)
    dt = g.choose_dt(P)
    C, G, sp = g.stage_prepare(P, P, dt)
    Pa = P.copy()
    nact, (rna, sta, ita), bta = g.newton(P, P, C, G, dt, Pa, max_iters=0)
    Pb = P.copy()
    state = None
    hist = []
    for k in range(10):
        nact, state, bt = g.newton(P, P, C, G, dt, Pb, max_iters=1, state=state)
        hist.append(g.interior(state[0]).max())
        if nact == 0:
            break
    assert np.array_equal(Pa, Pb) and np.array_equal(ita, state[2]) and np.array_equal(sta, state[1])
    assert np.array_equal(rna, state[0])
    assert g.interior(sta).min() & og.ST_CONVERGED
    assert hist[1] < 1e-3 * hist[0] and hist[2] < 1e-3 * hist[1], hist


def test_fill_ghosts():
    g = og.Grid(6, 5, 4, ng=2, dim=3, nvar=8, bc=[[og.BC_PERIODIC] * 2, [og.BC_REFLECT_POLAR] * 2, [og.BC_OUTFLOW] * 2])
    rng = np.random.default_rng(0)
    P = g.zeros()
    g.interior(P)[...] = rng.standard_normal((8, 4, 5, 6))
    g.fill_ghosts(P)
    assert np.array_equal(P[:, 2:6, 2:7, 0:2], P[:, 2:6, 2:7, 6:8])          # periodic X1
    assert np.array_equal(P[:, 2:6, 2:7, 8:10], P[:, 2:6, 2:7, 2:4])
    sgn = np.ones(8); sgn[3] = -1; sgn[6] = -1                              # u~2, B2 flip at the pole
    assert np.array_equal(P[:, 2:6, 1, :], sgn[:, None, None] * P[:, 2:6, 2, :])
    assert np.array_equal(P[:, 2:6, 0, :], sgn[:, None, None] * P[:, 2:6, 3, :])
    assert np.array_equal(P[:, 2:6, 8, :], sgn[:, None, None] * P[:, 2:6, 5, :])
    assert np.array_equal(P[:, 0, :, :], P[:, 2, :, :]) and np.array_equal(P[:, 7, :, :], P[:, 5, :, :])
