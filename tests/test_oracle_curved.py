"""Pins of the oracle's CURVED-SPACE path (readings C-5, C-8, C-9, C-11).
CPU only.  What is pinned and by what:

  * og_geometric_source (the routine og_stage_prepare calls per zone; eq 31) -- the identity
    T^k_l Gamma^l_{nu k} = (1/2) T^{kl} d_nu g_kl for the Levi-Civita connection, with d g taken by 4th-order
    differences of og_geom_kerr_mks (no Gamma on the right-hand side): rows nu = t, phi vanish (stationary,
    axisymmetric), rows r, theta match; the transposed contraction T^k_l Gamma^k_{nu l} fails (negative control).
  * emhd_space_part / og_emhd_targets with a non-zero connection (eqs 37-38) -- brute force
    nabla_mu u_nu = d_mu u_nu - Gamma^l_{mu nu} u_l written out with numpy, Gamma from the Christoffel formula on
    differenced metrics; a connection with the upper index misplaced fails.
  * og_stage_prepare + og_zone_residual on a Kerr grid, all ten rows (geometric source, face-centre geometry,
    the Gamma terms and limited slopes of the EMHD targets, tau_R = r^{3/2}, and the terms (1/2) q~ div u,
    (1/2) dP~ div u, which vanish in every linear test) -- a MANUFACTURED SOLUTION: for a smooth analytic
    field P(t, X) the grid residual must converge, at second order, to the continuum operator
    d_t U + d_i F^i - S evaluated independently from the paper's equations (eqs 30-31, 37-40) with high-order
    differences of the oracle's pinned point functions.  Dropping (1/2) q~ div u from the continuum side, or
    evaluating the fluxes with zone-centre geometry, is shown to be resolved (sensitivity checks).
  * an exact stationary solution: static Tolman atmosphere (Theta sqrt(-g_tt) = const) threaded by a monopole
    field in Schwarzschild, Kerr-Schild coordinates, with polar reflection -- the residual of all ten rows
    vanishes at second order (pressure gradient against the geometric source; q_0 = dP_0 = 0 only because the
    connection terms cancel the gradients), and og_timestep leaves it stationary.
  * og_fill_ghosts polar reflection -- an axisymmetric analytic field evaluated at the mirrored coordinates.
"""
import numpy as np
import pytest

import oracle as og

A_SPIN, H_MKS = 0.9375, 0.3
GAM = 4.0 / 3.0


def gcov_of(a, h, X1, X2):
    return og.geom_arrays(og.kerr_mks(a, h, X1, X2))[0]


def d4(f, x, d):
    """4th-order central difference of an array-valued function of one variable."""
    return (8.0 * (f(x + d) - f(x - d)) - (f(x + 2 * d) - f(x - 2 * d))) / (12.0 * d)


def dg_fd(a, h, X1, X2, d=1e-3):
    """dg[l][m][n] = d_l g_mn of the MKS Kerr metric by 4th-order differences (zero for l = t, phi)."""
    dg = np.zeros((4, 4, 4))
    dg[1] = d4(lambda x: gcov_of(a, h, x, X2), X1, d)
    dg[2] = d4(lambda x: gcov_of(a, h, X1, x), X2, d)
    return dg


def christoffel_fd(a, h, X1, X2, d=1e-3):
    g = og.kerr_mks(a, h, X1, X2)
    gcon = og.geom_arrays(g)[1]
    dg = dg_fd(a, h, X1, X2, d)
    # Gamma^l_mn = 1/2 g^lk (d_m g_kn + d_n g_km - d_k g_mn)
    return 0.5 * (np.einsum("lk,mkn->lmn", gcon, dg) + np.einsum("lk,nkm->lmn", gcon, dg)
                  - np.einsum("lk,kmn->lmn", gcon, dg))


def rand_prims(rng, n, nvar):
    P = np.zeros((n, nvar))
    P[:, 0] = 10 ** rng.uniform(-1, 0.5, n)
    P[:, 1] = 10 ** rng.uniform(-1, 0.5, n)
    P[:, 2:5] = rng.standard_normal((n, 3)) * np.array([0.3, 0.3, 0.05])
    P[:, 5:8] = rng.standard_normal((n, 3)) * np.array([0.3, 0.3, 0.05])
    if nvar == 10:
        P[:, 8:10] = rng.standard_normal((n, 2)) * 0.05
    return P


POINTS = ((np.log(1.5), 0.13), (np.log(3.0), 0.31), (np.log(12.0), 0.5), (np.log(30.0), 0.82))


# ------------------------------------------------------------------------------------------- geometric source
@pytest.mark.parametrize("nvar", [8, 10])
def test_geometric_source_is_half_T_dg(nvar):
    rng = np.random.default_rng(31)
    m = og.model(nvar=nvar, gam=GAM)
    worst_t, worst_x, worst_neg = 0.0, 0.0, np.inf
    for X1, X2 in POINTS:
        g = og.kerr_mks(A_SPIN, H_MKS, X1, X2)
        gcov, gcon, sg, _ = og.geom_arrays(g)
        conn = og.kerr_mks_conn(A_SPIN, H_MKS, X1, X2)
        dg = dg_fd(A_SPIN, H_MKS, X1, X2)
        for P in rand_prims(rng, 12, nvar):
            S = og.geometric_source(m, g, conn, P)
            T = og.stress_tensor(m, g, P)                    # T^mu_nu
            Tup = T @ gcon                                   # T^{mu nu}
            assert abs(Tup - Tup.T).max() < 1e-11 * abs(Tup).max()      # symmetric: eq 27 lowered correctly
            ref = 0.5 * sg * np.einsum("kl,nkl->n", Tup, dg)
            scale = sg * abs(T).max() * abs(conn).max()
            worst_t = max(worst_t, abs(S[0]) / scale, abs(S[3]) / scale)
            worst_x = max(worst_x, abs(S[1] - ref[1]) / scale, abs(S[2] - ref[2]) / scale)
            # negative control: the index of Gamma contracted with the UPPER index of T
            wrong = sg * np.einsum("kl,knl->n", T, conn)
            worst_neg = min(worst_neg, abs(wrong - ref).max() / scale)
    assert worst_t < 1e-13          # nu = t, phi: stationarity and axisymmetry
    assert worst_x < 1e-9           # nu = r, theta: against the differenced metric
    assert worst_neg > 1e-3         # the transposed contraction does not satisfy the identity


def test_stress_tensor_entry_point_is_the_flux_rows():
    rng = np.random.default_rng(32)
    m = og.model(nvar=10, gam=GAM)
    g = og.kerr_mks(A_SPIN, H_MKS, np.log(4.0), 0.4)
    for P in rand_prims(rng, 5, 10):
        T = og.stress_tensor(m, g, P)
        assert np.array_equal(g.sqrtmg * T[0], og.prim_to_U(m, g, 1.0, P)[1:5])
        for d in (1, 2, 3):
            assert np.array_equal(g.sqrtmg * T[d], og.prim_to_F(m, g, 1.0, d, P)[1:5])


# ------------------------------------------------------------------------------------------- EMHD targets with Gamma
def state_np(P, gcov, gcon, alpha):
    """u^mu, u_mu, b^mu, bhat^mu, b^2 from the paper's definitions (L41, L248; C-9), numpy."""
    ut = P[2:5]
    W = np.sqrt(1.0 + ut @ gcov[1:, 1:] @ ut)
    ucon = np.concatenate([[W / alpha], ut - W * alpha * gcon[0, 1:]])
    ucov = gcov @ ucon
    bt = P[5:8] @ ucov[1:]
    bcon = np.concatenate([[bt], (P[5:8] + bt * ucon[1:]) / ucon[0]])
    bsq = bcon @ gcov @ bcon
    return ucon, ucov, bcon, bcon / np.sqrt(bsq), bsq


def targets_np(P, gcov, gcon, alpha, conn, tau, dTheta, ducov, divu, phi=1.0, psi=1.0, gam=GAM):
    """q_0 = -rho chi bhat^mu (d_mu Theta + Theta a_mu), a_mu = u^nu nabla_nu u_mu (eq 37);
    dP_0 = 3 rho nu (bhat^mu bhat^nu nabla_mu u_nu - div u / 3) (eq 38, G-5);
    nabla_mu u_nu = d_mu u_nu - Gamma^l_{mu nu} u_l;  chi = phi cs^2 tau, nu = psi cs^2 tau (L299)."""
    ucon, ucov, _, bh, _ = state_np(P, gcov, gcon, alpha)
    rho, u = P[0], P[1]
    Pg = (gam - 1.0) * u
    Th = Pg / rho
    cs2 = gam * Pg / (rho + gam * u)
    nab = ducov - np.einsum("lmn,l->mn", conn, ucov)          # nabla_mu u_nu
    acc = ucon @ nab                                          # a_nu
    q0 = -rho * (phi * cs2 * tau) * (bh @ (dTheta + Th * acc))
    dP0 = 3.0 * rho * (psi * cs2 * tau) * (bh @ nab @ bh - divu / 3.0)
    return q0, dP0


def test_emhd_targets_with_connection_against_brute_force():
    rng = np.random.default_rng(33)
    m = og.model(nvar=10, gam=GAM, phi=0.8, psi=1.3)
    worst, worst_neg = 0.0, np.inf
    for X1, X2 in POINTS:
        g = og.kerr_mks(A_SPIN, H_MKS, X1, X2)
        gcov, gcon, sg, alpha = og.geom_arrays(g)
        conn_o = og.kerr_mks_conn(A_SPIN, H_MKS, X1, X2)
        conn_fd = christoffel_fd(A_SPIN, H_MKS, X1, X2)
        assert abs(conn_o - conn_fd).max() < 1e-8 * abs(conn_fd).max()
        tau = np.exp(1.5 * X1)
        for P in rand_prims(rng, 10, 10):
            dTheta = rng.standard_normal(4)
            ducov = rng.standard_normal((4, 4))
            divu = rng.standard_normal()
            q0, dP0 = og.emhd_targets(m, g, conn_o, tau, P, dTheta, ducov, divu)
            rq, rd = targets_np(P, gcov, gcon, alpha, conn_fd, tau, dTheta, ducov, divu, phi=0.8, psi=1.3)
            sc_q = abs(rq) + P[0] * tau * abs(conn_fd).max()
            sc_d = abs(rd) + P[0] * tau * abs(conn_fd).max()
            worst = max(worst, abs(q0 - rq) / sc_q, abs(dP0 - rd) / sc_d)
            # negative control: the upper index of Gamma exchanged with a lower one
            wq, wd = targets_np(P, gcov, gcon, alpha, conn_fd.transpose(1, 0, 2), tau, dTheta, ducov, divu,
                                phi=0.8, psi=1.3)
            worst_neg = min(worst_neg, max(abs(wq - q0) / sc_q, abs(wd - dP0) / sc_d))
    assert worst < 1e-8
    assert worst_neg > 1e-4


# ------------------------------------------------------------------------------------------- manufactured solution
class Field:
    """Smooth analytic primitives P(t, X) = base + amp sin(phase), phase = k.(X - X_mid) + w t + phi kept inside
    (-pi/2, pi/2) over the whole box and the time of the test, so that every primitive is monotone in every
    coordinate: the limited slopes of the EMHD gradient terms (L115) then equal the central differences, as they do
    for resolved smooth data, and the limiter's clipping at extrema (a local O(dX) effect that belongs to the scheme,
    not to the equations) does not blur the convergence order."""

    def __init__(self, nvar, seed, lo, hi, amp=0.25):
        rng = np.random.default_rng(seed)
        self.nvar = nvar
        lo, hi = np.asarray(lo, float), np.asarray(hi, float)
        self.mid = 0.5 * (lo + hi)
        half = 0.5 * (hi - lo)
        self.base = np.array([1.0, 1.5, 0.12, -0.08, 0.05, 0.25, 0.35, -0.15, 0.03, -0.04][:nvar])
        self.amp = amp * np.array([1.0, 1.5, 0.5, 0.5, 0.3, 0.4, 0.4, 0.3, 0.3, 0.3][:nvar])
        # each active direction swings the phase by +-(0.2 .. 0.3) rad across the box; |phi| <= 0.3
        self.k = rng.choice([-1.0, 1.0], (nvar, 3)) * rng.uniform(0.2, 0.3, (nvar, 3)) / np.where(half > 0, half, 1.0)
        self.k[:, half <= 0] = 0.0
        self.w = rng.uniform(0.5, 1.5, nvar)
        self.ph = rng.uniform(-0.3, 0.3, nvar)

    def __call__(self, t, X1, X2, X3):
        X1, X2, X3 = np.broadcast_arrays(np.asarray(X1, float), np.asarray(X2, float), np.asarray(X3, float))
        out = np.empty((self.nvar,) + X1.shape)
        for v in range(self.nvar):
            out[v] = self.base[v] + self.amp[v] * np.sin(self.k[v, 0] * (X1 - self.mid[0]) + self.k[v, 1] * (X2 - self.mid[1])
                                                         + self.k[v, 2] * (X3 - self.mid[2]) + self.w[v] * t + self.ph[v])
        return out


def continuum_operator(field, m, kerr, tau_mode, tau_const, t, X, d=2e-3, drop_half_div=False, phi=1.0, psi=1.0):
    """L[P](t, X) = d_t U + d_i F^i - S from the paper's equations: eq 30 (rows 0, 5-7: no source), eq 31 (rows
    1-4: S_nu = (1/2) sqrt(-g) T^{kl} d_nu g_kl), eqs 39-40 with eqs 37-38, 41-42 (rows 8, 9).  Derivatives by
    4th-order differences of og_prim_to_U / og_prim_to_F / og_derived along t, X1, X2, X3."""
    nvar = m.nvar
    X = np.asarray(X, float)

    def geom(x):
        return og.kerr_mks(A_SPIN, H_MKS, x[0], x[1]) if kerr else og.minkowski()

    def tau(x):
        return np.exp(1.5 * x[0]) if tau_mode == og.TAU_R32 else tau_const

    def prim(tt, x):
        return field(tt, x[0], x[1], x[2])

    def shifted(mu, s):
        x = X.copy()
        tt = t
        if mu == 0:
            tt = t + s
        else:
            x[mu - 1] += s
        return tt, x

    def dmu(fun, mu):
        return d4(lambda s: fun(*shifted(mu, s)), 0.0, d)

    L = dmu(lambda tt, x: og.prim_to_U(m, geom(x), tau(x), prim(tt, x)), 0)
    for dd in (1, 2, 3):
        L = L + dmu(lambda tt, x, dd=dd: og.prim_to_F(m, geom(x), tau(x), dd, prim(tt, x)), dd)
    g = geom(X)
    gcov, gcon, sg, alpha = og.geom_arrays(g)
    P = prim(t, X)
    terms = abs(L).copy()
    if kerr:
        T = np.zeros((4, 4))
        T[0] = og.prim_to_U(m, g, tau(X), P)[1:5]
        for dd in (1, 2, 3):
            T[dd] = og.prim_to_F(m, g, tau(X), dd, P)[1:5]
        Tup = (T / sg) @ gcon
        dg = dg_fd(A_SPIN, H_MKS, X[0], X[1])
        S = 0.5 * sg * np.einsum("kl,nkl->n", Tup, dg)
        L[1:5] -= S
        terms[1:5] += abs(S)
        conn = christoffel_fd(A_SPIN, H_MKS, X[0], X[1])
    else:
        conn = np.zeros((4, 4, 4))
    if nvar == 10:
        def der(tt, x):
            th, ucon, ucov = og.derived(m, geom(x), prim(tt, x))
            sgx = geom(x).sqrtmg
            return np.concatenate([[th], ucov, sgx * ucon])
        D = np.array([dmu(der, mu) for mu in range(4)])          # D[mu] = d_mu (Theta, u_nu, sqrt(-g) u^nu)
        dTheta, ducov = D[:, 0], D[:, 1:5]
        divu = sum(D[mu, 5 + mu] for mu in range(4)) / sg
        q0, dP0 = targets_np(P, gcov, gcon, alpha, conn, tau(X), dTheta, ducov, divu, phi=phi, psi=psi)
        fq, fd = og.rescale_factors(m, tau(X), P)
        qt, dpt = P[8] * fq, P[9] * fd
        hq = 0.0 if drop_half_div else 0.5 * qt * divu
        hd = 0.0 if drop_half_div else 0.5 * dpt * divu
        Sq = sg * (-(qt - fq * q0) / tau(X) + hq)
        Sd = sg * (-(dpt - fd * dP0) / tau(X) + hd)
        L[8] -= Sq
        L[9] -= Sd
        terms[8] += abs(Sq)
        terms[9] += abs(Sd)
    return L, terms


def grid_residual(field, gk, t0, dts, sample):
    """Stage-1 residual (eq 19: P_E = P_n) of the oracle grid at the trial state field(t0 + dts) for the sampled
    interior zones; every ghost zone holds the analytic field (BC_NONE)."""
    g = og.Grid(**gk)
    X1, X2, X3 = g.centers()
    Pn = np.ascontiguousarray(field(t0, X1, X2, X3))
    P = np.ascontiguousarray(field(t0 + dts, X1, X2, X3))
    C, G, _ = g.stage_prepare(Pn, Pn, dts)
    out = []
    for (k, j, i) in sample(g):
        z = (k * g.sz[1] + j) * g.sz[0] + i
        R = g.zone_residual(z, Pn, Pn, C, G, dts, P[:, k, j, i])
        out.append(((X1[k, j, i], X2[k, j, i], X3[k, j, i]), R))
    return out


def mms_errors(field, m, gk_of_n, ns, kerr, tau_mode, tau_const, t0=0.05, dts=1e-5, per_dir=12, **kw):
    """|R_grid - L| / (size of the terms of that row) over a regular sub-lattice of about per_dir zones per active
    direction, per resolution: returns (mean over the zones, max over the zones), each [resolution][row].  The mean
    is the L1 error the paper's convergence plots use (L507): where a derived quantity has an extremum the limited
    slope (L115) is clipped to zero, a local O(dX) error on a set of zones of measure O(dX)."""
    means, maxs = [], []
    for n in ns:
        gk = gk_of_n(n)

        def sample(g):
            ax = [range(g.ngd[a] + (max(g.n[a] // per_dir, 1)) // 2, g.ngd[a] + g.n[a], max(g.n[a] // per_dir, 1))
                  for a in range(3)]
            return [(k, j, i) for k in ax[2] for j in ax[1] for i in ax[0]]
        E = []
        for X, R in grid_residual(field, gk, t0, dts, sample):
            L, terms = continuum_operator(field, m, kerr, tau_mode, tau_const, t0, X, **kw)
            E.append(abs(R - L) / terms.max())
        E = np.array(E)
        means.append(E.mean(axis=0))
        maxs.append(E.max(axis=0))
    return np.array(means), np.array(maxs)


KERR_LO, KERR_HI = (np.log(3.0), 0.12, 0.0), (np.log(6.0), 0.44, 1.0)   # one hemisphere: the metric is even about X2 = 1/2


def kerr_gk(n, nvar=10, recon=og.MP5, dim=2, n3=1):
    return dict(n1=n, n2=n, n3=n3, ng=3, dim=dim, xstart=KERR_LO, xend=KERR_HI,
                bc=og.BC_NONE, nvar=nvar, recon=recon, limiter_theta=2.0, gam=GAM, tau_mode=og.TAU_R32,
                metric=og.KERR_MKS, metric_params=(A_SPIN, H_MKS))


def test_manufactured_solution_kerr_2d_converges_at_second_order():
    m = og.model(nvar=10, gam=GAM)
    field = Field(10, 5, KERR_LO[:2] + (0.0,), KERR_HI[:2] + (0.0,))
    mean, mx = mms_errors(field, m, kerr_gk, (16, 32, 64), True, og.TAU_R32, 1.0)
    assert mean[2].max() < 2e-4, mean
    # second order in L1, every row on its own: mass, the four geometric-source rows, induction, q, dP
    assert (mean[0] / mean[1] > 3.3).all() and (mean[1] / mean[2] > 3.3).all(), mean
    # rows without limited slopes also pointwise
    assert (mx[0, :8] / mx[1, :8] > 3.3).all() and (mx[1, :8] / mx[2, :8] > 3.3).all(), mx


def test_manufactured_solution_resolves_the_half_div_terms():
    """Sensitivity of the pin: dropping (1/2) q~ div u, (1/2) dP~ div u from the continuum side moves rows 8, 9 by
    far more than the error reached at 64^2, so an oracle that dropped them would fail the test above."""
    m = og.model(nvar=10, gam=GAM)
    field = Field(10, 5, KERR_LO[:2] + (0.0,), KERR_HI[:2] + (0.0,))
    full = mms_errors(field, m, kerr_gk, (64,), True, og.TAU_R32, 1.0, per_dir=6)[0][0]
    dropped = mms_errors(field, m, kerr_gk, (64,), True, og.TAU_R32, 1.0, per_dir=6, drop_half_div=True)[0][0]
    assert dropped[8] > 20 * full[8] and dropped[9] > 20 * full[9], (full, dropped)


def test_manufactured_solution_kerr_3d_minmod():
    """3-D general-metric path (config 5's shape): X3 fluxes and slopes, minmod(theta = 2), ideal and EMHD."""
    for nvar in (8, 10):
        m = og.model(nvar=nvar, gam=GAM)
        field = Field(nvar, 9, KERR_LO, KERR_HI)
        mean, mx = mms_errors(field, m, lambda n: kerr_gk(n, nvar=nvar, recon=og.MINMOD, dim=3, n3=n), (12, 24), True,
                              og.TAU_R32, 1.0, per_dir=6)
        assert (mean[0] / mean[1] > 3.0).all(), mean


def test_manufactured_solution_minkowski_3d():
    m = og.model(nvar=10, gam=GAM, phi=0.7, psi=1.4)
    field = Field(10, 6, (0.0, 0.0, 0.0), (1.0, 1.0, 1.0))

    def gk(n):
        # limiter_theta = 2: with theta = 1 the limited slope of monotone data is the smaller one-sided difference,
        # a first-order gradient
        return dict(n1=n, n2=n, n3=n, ng=3, dim=3, bc=og.BC_NONE, nvar=10, recon=og.MP5, limiter_theta=2.0, gam=GAM,
                    phi=0.7, psi=1.4, tau=0.5, metric=og.MINKOWSKI)
    mean, mx = mms_errors(field, m, gk, (12, 24), False, og.TAU_CONST, 0.5, dts=1e-6, per_dir=6, phi=0.7, psi=1.4)
    # rows 0-7 are MP5 fluxes only: already at the O(dt') floor of the time difference; rows 8, 9 carry the 3-point slopes
    assert (mean[1, :8] < 1e-6).all() and (mean[0, 8:] / mean[1, 8:] > 3.3).all(), mean
    dropped = mms_errors(field, m, gk, (24,), False, og.TAU_CONST, 0.5, dts=1e-6, per_dir=6, phi=0.7, psi=1.4,
                         drop_half_div=True)[0][0]
    assert dropped[8] > 10 * mean[1][8] and dropped[9] > 10 * mean[1][9]


# ------------------------------------------------------------------------------------------- exact stationary solution
def tolman_atmosphere(g, K=0.05, Theta_inf=1.0, Bmono=0.4):
    """Static fluid u^mu = xi^mu/|xi| in Schwarzschild (a = 0), Kerr-Schild coordinates, in thermal (Tolman:
    Theta chi = Theta_inf, chi = sqrt(1 - 2/r)) and hydrostatic equilibrium (d P_g = -(rho + u + P_g) d ln chi):
        ln P_g = ln K - chi/Theta_inf - gam/(gam-1) ln chi,   rho = P_g/Theta,   u = P_g/(gam-1),
    threaded by the monopole B^{X1} = Bmono / r^3 (sqrt(-g) B^1 independent of X1: div B = 0, current-free).
    Then q_0 = 0 (eq 37: d_mu Theta + Theta a_mu = 0), dP_0 = 0 (eq 38: rigid Killing flow), and q = dP = 0 is an
    exact stationary solution of all ten equations."""
    X1, X2, X3 = g.centers()
    r = np.exp(X1)
    chi = np.sqrt(1.0 - 2.0 / r)
    Th = Theta_inf / chi
    Pg = K * np.exp(-chi / Theta_inf) * chi ** (-GAM / (GAM - 1.0))
    P = np.zeros(g.shape)
    P[0] = Pg / Th
    P[1] = Pg / (GAM - 1.0)
    # u^i = 0, u^t = 1/chi  ->  W = alpha u^t,  u~^i = u^i + W alpha g^{ti} (C-9)
    for j in range(g.sz[1]):
        for i in range(g.sz[0]):
            gcov, gcon, sg, alpha = og.geom_arrays(g.geom(0, j, i))
            W = alpha / np.sqrt(-gcov[0, 0])
            P[2:5, :, j, i] = (W * alpha * gcon[0, 1:4])[:, None]
    P[5] = Bmono / r ** 3
    return P


def atmosphere_gk(n, nvar):
    bc = [[og.BC_NONE, og.BC_NONE], [og.BC_REFLECT_POLAR, og.BC_REFLECT_POLAR], [og.BC_PERIODIC, og.BC_PERIODIC]]
    return dict(n1=n, n2=n, ng=3, dim=2, xstart=(np.log(3.0), 0.0, 0.0), xend=(np.log(9.0), 1.0, 1.0), bc=bc,
                nvar=nvar, recon=og.MP5, limiter_theta=2.0, gam=GAM, tau_mode=og.TAU_R32, metric=og.KERR_MKS,
                metric_params=(0.0, H_MKS))


@pytest.mark.parametrize("nvar", [8, 10])
def test_tolman_atmosphere_is_stationary_at_second_order(nvar):
    errs = []
    for n in (16, 32, 64):
        g = og.Grid(**atmosphere_gk(n, nvar))
        P = tolman_atmosphere(g)[:nvar].copy()
        g.fill_ghosts(P)
        dts = 1e3
        C, G, _ = g.stage_prepare(P, P, dts)
        Ci = g.interior(C)
        # R(P_n) = C + U(P_n)/dt' = div F - S (the U terms cancel to round-off / dt'); size of the balancing terms of
        # the radial momentum row: sqrt(-g) P_g / dX1
        X1, X2, _ = g.centers()
        R = np.zeros((nvar, g.n[1], g.n[0]))
        scale = 0.0
        for jj in range(g.n[1]):
            for ii in range(g.n[0]):
                j, i = jj + g.ngd[1], ii + g.ngd[0]
                R[:, jj, ii] = g.zone_residual(j * g.sz[0] + i, P, P, C, G, dts, P[:, 0, j, i])
                scale = max(scale, g.geom(0, j, i).sqrtmg * (GAM - 1.0) * P[1, 0, j, i])
        errs.append(abs(R).max(axis=(1, 2)) / scale)
    errs = np.array(errs)
    assert errs[2].max() < 1e-2, errs
    # second order: cleanly in the theta-momentum row (pressure gradient against the geometric source all the way to
    # the axis) and in the EMHD rows; on average over the two doublings in the rows whose coarse-grid error is the
    # MP5 limiter's on the steep inner atmosphere
    assert errs[0][3] / errs[1][3] > 3.5 and errs[1][3] / errs[2][3] > 3.5, errs
    assert (errs[0][:3] / errs[2][:3] > 12.0).all(), errs
    assert (errs[:, 4] == 0).all() and (errs[:, 6:8] == 0).all()        # u_phi = B^2 = B^3 = 0 exactly
    if nvar == 10:   # q_0 = dP_0 = 0 needs the connection terms to cancel the gradients
        assert (errs[0][8:] / errs[1][8:] > 3.5).all() and (errs[1][8:] / errs[2][8:] > 3.5).all(), errs


def test_tolman_atmosphere_needs_the_geometric_source():
    """Sensitivity: the same atmosphere with the pressure scale height halved (a force imbalance of order one, which
    is what a wrong Gamma contraction in the radial source row would be) does not converge."""
    g = og.Grid(**atmosphere_gk(32, 8))
    P = tolman_atmosphere(g, Theta_inf=0.5)[:8].copy()       # Theta_inf halved in P_g only below
    P_ok = tolman_atmosphere(g, Theta_inf=1.0)[:8]
    P[0] = P_ok[0] * P[1] / P_ok[1]                          # P_g profile of Theta_inf = 0.5 at the temperature of 1.0
    g.fill_ghosts(P)
    C, G, _ = g.stage_prepare(P, P, 1e3)
    j, i = g.ngd[1] + 16, g.ngd[0] + 16
    R = g.zone_residual(j * g.sz[0] + i, P, P, C, G, 1e3, P[:, 0, j, i])
    assert abs(R[2]) / (g.geom(0, j, i).sqrtmg * (GAM - 1.0) * P[1, 0, j, i]) > 0.1


def test_tolman_atmosphere_time_step_is_stationary():
    drift = []
    for n in (16, 32):
        g = og.Grid(**atmosphere_gk(n, 10))
        P0 = tolman_atmosphere(g)
        g.fill_ghosts(P0)
        P = P0.copy()
        dt = 0.2 * g.dx[0] * 3.0            # a fraction of the light-crossing time of the innermost zone
        for _ in range(4):
            g.timestep(P, dt)
        d = g.interior(P) - g.interior(P0)
        rel = [abs(d[0]).max() / abs(g.interior(P0)[0]).max(), abs(d[1]).max() / abs(g.interior(P0)[1]).max(),
               abs(d[8]).max() / abs(g.interior(P0)[1]).max(), abs(d[9]).max() / abs(g.interior(P0)[1]).max()]
        drift.append(max(rel) / (4 * dt))
    assert drift[1] < 2e-3 and drift[0] / drift[1] > 2.5, drift


# ------------------------------------------------------------------------------------------- polar reflection
def test_polar_reflection_is_the_field_at_the_mirrored_coordinates():
    """A smooth axisymmetric field continued through the axis: scalars and the X1, X3 components are even in theta,
    the X2 components (u~^2, B^2) odd.  og_fill_ghosts(REFLECT_POLAR) must reproduce the analytic field evaluated
    at the ghost coordinates (theta(X2) is odd about X2 = 0 and about X2 = 1)."""
    bc = [[og.BC_OUTFLOW, og.BC_OUTFLOW], [og.BC_REFLECT_POLAR, og.BC_REFLECT_POLAR], [og.BC_PERIODIC, og.BC_PERIODIC]]
    g = og.Grid(n1=8, n2=12, ng=3, dim=2, xstart=(0.0, 0.0, 0.0), xend=(1.0, 1.0, 1.0), bc=bc, nvar=10)
    X1, X2, _ = g.centers()
    th = np.pi * X2 + 0.5 * (1 - H_MKS) * np.sin(2 * np.pi * X2)
    even = lambda c: 1.0 + 0.3 * np.cos(th) * c + 0.1 * np.cos(2 * th) * X1
    odd = lambda c: 0.2 * np.sin(th) * c + 0.05 * np.sin(2 * th) * X1
    P = np.zeros(g.shape)
    for v in range(10):
        P[v] = odd(v + 1.0) if v in (3, 6) else even(v + 1.0)
    Q = P.copy()
    ng = g.ngd[1]
    Q[:, :, :ng, :] = np.nan
    Q[:, :, ng + g.n[1]:, :] = np.nan
    g.fill_ghosts(Q)
    i0, i1 = g.ngd[0], g.ngd[0] + g.n[0]
    assert np.allclose(Q[:, :, :, i0:i1], P[:, :, :, i0:i1], rtol=0, atol=1e-14)
    # outflow in X1: copies of the nearest interior zone, X2 ghosts included
    assert np.array_equal(Q[:, :, :, 0], Q[:, :, :, i0]) and np.array_equal(Q[:, :, :, -1], Q[:, :, :, i1 - 1])
