"""Element-level oracle pins: line search (P-5), LU vs LAPACK (P-9), reconstruction (P-10), wave speeds,
stress-tensor invariants, geometry identities (P-12a).  CPU only."""
import numpy as np
import pytest

import oracle as og

RNG = np.random.default_rng(20170201)


# ---------------------------------------------------------------- P-5 line search (eq 25)
def test_linesearch_is_quadratic_minimiser():
    # f(l) = f0 - 2 f0 l + c l^2 has f(0) = f0, f'(0) = -2 f0 and its minimiser is f0/c
    for f0, c, lam in ((3.0, 40.0, 1.0), (1e-6, 5e-5, 0.37), (2.0, 9.0, 0.5)):
        fl = f0 - 2 * f0 * lam + c * lam * lam
        assert abs(og.linesearch_lambda(f0, fl, lam) - f0 / c) < 1e-14 * f0 / c * 10


def test_linesearch_shrinks_when_rejected():
    # rejected trial: sqrt(f(l)) >= sqrt(f0) (1 - eps l)  =>  0 < l_new <= l / (2 (1 - eps))   (C-14)
    eps = 1e-4
    for _ in range(1000):
        f0 = 10 ** RNG.uniform(-12, 6)
        lam = RNG.uniform(1e-3, 1.0)
        fl = f0 * (1 - eps * lam) ** 2 * (1 + 10 ** RNG.uniform(-8, 4))
        ln = og.linesearch_lambda(f0, fl, lam)
        assert 0 < ln <= lam / (2 * (1 - eps)) * (1 + 1e-12)


# ---------------------------------------------------------------- P-9 LU vs LAPACK
@pytest.mark.parametrize("n", [5, 7, 8, 10])
def test_lu_matches_lapack(n):
    import scipy.linalg as sla
    for trial in range(200):
        A = RNG.standard_normal((n, n))
        if trial % 3 == 1:   # graded rows/columns, as a Jacobian in mixed units
            A = A * 10.0 ** RNG.uniform(-6, 6, (n, 1)) * 10.0 ** RNG.uniform(-3, 3, (1, n))
        b = RNG.standard_normal(n)
        x, piv, info = og.lu_solve(A, b)
        assert info == 0
        lu, lpiv = sla.lu_factor(A)
        assert np.array_equal(piv, lpiv)                      # identical pivot sequence (dgetrf)
        xr = sla.lu_solve((lu, lpiv), b)
        cond = np.linalg.cond(A)
        assert np.max(abs(x - xr)) <= 1e-13 * cond * np.max(abs(xr)) + 1e-300


def test_lu_flags_singular():
    A = np.array([[1.0, 2.0, 3.0], [2.0, 4.0, 6.0], [1.0, 0.0, 1.0]])
    A[:, 1] = 0.0                                # exact zero column -> zero pivot at step 2 (C-19)
    x, piv, info = og.lu_solve(A, np.ones(3))
    assert info == 2
    A = np.eye(3); A[1, 1] = np.nan
    assert og.lu_solve(A, np.ones(3))[2] != 0


def test_lu_first_max_tie_break():
    A = np.array([[1.0, 2.0, 0.0], [-1.0, 1.0, 1.0], [1.0, 0.0, 3.0]])   # |a_i0| all equal: LAPACK keeps row 0
    x, piv, info = og.lu_solve(A, np.array([1.0, 2.0, 3.0]))
    assert piv[0] == 0 and np.allclose(A @ x, [1, 2, 3])


# ---------------------------------------------------------------- P-10 reconstruction
def test_minmod_cases():
    assert og.minmod3(1.0, 2.0, 3.0) == 1.0
    assert og.minmod3(-1.0, -2.0, -0.5) == -0.5
    assert og.minmod3(1.0, -2.0, 3.0) == 0.0
    assert og.minmod3(0.0, 2.0, 3.0) == 0.0
    # generalised minmod slope: theta=1 picks the smaller one-sided difference, theta=2 the central one
    assert og.slope(1.0, 0.0, 1.0, 3.0) == 1.0
    assert og.slope(2.0, 0.0, 1.0, 3.0) == 1.5
    assert og.slope(1.0, 0.0, 1.0, 0.5) == 0.0           # extremum


def test_minmod_reconstructs_linear_data_exactly():
    v = np.array([0.0, 0.25, 0.5, 0.75, 1.0]) * 3.0 + 1.0
    lu, rl = og.reconstruct(og.MINMOD, 1.0, v)
    assert lu == (v[2] + v[3]) / 2 and rl == (v[1] + v[2]) / 2


def test_mp5_exact_for_quartics_and_mirror_symmetric():
    # cell-centred POINT values of a degree-4 polynomial: the unlimited MP5 value is the 5th-order
    # interpolant of cell AVERAGES, so feed averages and compare with the exact face value
    from numpy.polynomial import polynomial as Pn
    for _ in range(50):
        c = RNG.standard_normal(5) * np.array([1, 0.0, 0.05, 0.01, 0.002]) + np.array([50, RNG.choice([-1.0, 1.0]), 0, 0, 0])  # monotone: limiter inactive
        ci = Pn.polyint(c)
        avg = np.array([Pn.polyval(i + 0.5, ci) - Pn.polyval(i - 0.5, ci) for i in range(-2, 3)])
        lu, rl = og.reconstruct(og.MP5, 1.0, avg)
        assert abs(lu - Pn.polyval(0.5, c)) < 1e-12 * 50
        assert abs(rl - Pn.polyval(-0.5, c)) < 1e-12 * 50
        lu2, rl2 = og.reconstruct(og.MP5, 1.0, avg[::-1].copy())
        assert lu2 == rl and rl2 == lu


def test_mp5_monotone_data_stays_bounded():
    for _ in range(500):
        v = np.cumsum(RNG.uniform(0, 1, 5) ** 3)       # monotone increasing, uneven jumps
        lu, rl = og.reconstruct(og.MP5, 1.0, v)
        t = 1e-14
        assert v[2] - t <= lu <= v[3] + t and v[1] - t <= rl <= v[2] + t
    v = np.array([0.0, 0.0, 0.0, 1.0, 1.0])             # step: limiter active
    lu, rl = og.reconstruct(og.MP5, 1.0, v)
    assert 0.0 <= lu <= 1.0 and rl == 0.0


# ---------------------------------------------------------------- wave speeds (eqs 43-48)
def _rand_prims(n, nvar=10):
    P = np.zeros((n, nvar))
    P[:, 0] = 10 ** RNG.uniform(-2, 1, n)
    P[:, 1] = 10 ** RNG.uniform(-2, 1, n)
    P[:, 2:5] = RNG.standard_normal((n, 3))
    P[:, 5:8] = RNG.standard_normal((n, 3)) * 0.5
    if nvar == 10:
        P[:, 8] = RNG.standard_normal(n) * 0.01
        P[:, 9] = RNG.standard_normal(n) * 0.01
    return P


def test_wave_speeds_rest_frame_and_boost():
    g = og.minkowski()
    for nvar in (8, 10):
        m = og.model(nvar=nvar)
        for P in _rand_prims(50, nvar):
            P0 = P.copy(); P0[2:5] = 0
            vm = np.sqrt(og.vmax2(m, g, 1.0, P0))
            for d in (1, 2, 3):
                vp, vn = og.wave_speeds(m, g, 1.0, d, P0)
                assert abs(vp - vm) < 1e-13 and abs(vn + vm) < 1e-13
            # motion along x only: relativistic velocity addition of +-vmax (b^2 is frame invariant)
            Pb = P.copy(); Pb[3:5] = 0
            v = Pb[2] / np.sqrt(1 + Pb[2] ** 2)
            vmb = np.sqrt(og.vmax2(m, g, 1.0, Pb))
            vp, vn = og.wave_speeds(m, g, 1.0, 1, Pb)
            assert abs(vp - (v + vmb) / (1 + v * vmb)) < 1e-12
            assert abs(vn - (v - vmb) / (1 - v * vmb)) < 1e-12
            assert abs(og.cmax(m, g, 1.0, 1, Pb) - max(abs(vp), abs(vn))) == 0
            assert og.cmax(m, g, 1.0, 2, P) < 1.0


def test_vmax_ideal_closed_form():
    g = og.minkowski()
    m = og.model(nvar=8)
    P = np.array([1.0, 2.0, 0, 0, 0, 0.1, 0.3, 0.0])
    gam = 4.0 / 3.0
    cs2 = gam * (gam - 1) * 2 / (1 + gam * 2)
    va2 = 0.1 / (1 + gam * 2 + 0.1)
    assert abs(og.vmax2(m, g, 1.0, P) - (cs2 + va2 - cs2 * va2)) < 1e-15
    assert abs(np.sqrt(og.vmax2(m, g, 1.0, P)) - 0.512383522) < 1e-9      # SURVEY P-3


# ---------------------------------------------------------------- stress tensor invariants (eqs 27, 33-34)
def _full_T(m, g, P):
    T = np.zeros((4, 4))
    T[0] = og.prim_to_U(m, g, 1.0, P)[1:5]
    for d in (1, 2, 3):
        T[d] = og.prim_to_F(m, g, 1.0, d, P)[1:5]
    return T / g.sqrtmg


@pytest.mark.parametrize("curved", [False, True])
def test_stress_tensor_trace_and_eckart_frame(curved):
    g = og.kerr_mks(0.9375, 0.3, np.log(3.0), 0.31) if curved else og.minkowski()
    gam = 4.0 / 3.0
    for nvar in (8, 10):
        m = og.model(nvar=nvar, gam=gam)
        for P in _rand_prims(40, nvar):
            T = _full_T(m, g, P)
            rho, u = P[0], P[1]
            # trace: q and dP terms are traceless, b-terms cancel: T^mu_mu = -(rho+u) + 3 P_g
            assert abs(np.trace(T) - (-(rho + u) + 3 * (gam - 1) * u)) < 1e-11 * (abs(T).max())
            # T^mu_nu u^nu = -(rho + u + b^2/2) u^mu - q bhat^mu   (Eckart frame, L248)
            th, ucon, ucov = og.derived(m, g, P)
            lhs = T @ ucon
            D = og.prim_to_U(m, g, 1.0, P)[0] / g.sqrtmg
            assert abs(D - rho * ucon[0]) < 1e-13 * abs(D)
            assert abs(ucon @ ucov + 1) < 1e-12 * ucon[0] ** 2
            if nvar == 8:
                # lhs parallel to u^mu; the coefficient gives b^2 >= 0
                coef = lhs[0] / ucon[0]
                assert np.max(abs(lhs - coef * ucon)) < 1e-10 * abs(lhs).max()
                bsq = -2 * (coef + rho + u)
                assert bsq > -1e-10
            else:
                # remove the part along u: remainder = -q bhat, whose norm^2 is q^2
                gcov = np.array([[g.gcov[i][j] for j in range(4)] for i in range(4)])
                # lhs + (u_nu lhs^nu) u^mu projects out the part along u (u.u = -1)
                rem = lhs + (lhs @ gcov @ ucon) * ucon
                assert abs(rem @ gcov @ rem - P[8] ** 2) < 1e-9 * max(1.0, abs(T).max() ** 2)


def test_conserved_B_is_sqrtmg_B_and_induction_flux_antisymmetric():
    g = og.kerr_mks(0.5, 0.3, np.log(5.0), 0.4)
    m = og.model(nvar=8)
    for P in _rand_prims(20, 8):
        U = og.prim_to_U(m, g, 1.0, P)
        assert np.array_equal(U[5:8], g.sqrtmg * P[5:8])
        F = [og.prim_to_F(m, g, 1.0, d, P) for d in (1, 2, 3)]
        for i in range(3):
            assert F[i][5 + i] == 0.0                      # F^i(B^i) = 0
            for j in range(3):
                assert abs(F[j][5 + i] + F[i][5 + j]) < 1e-13 * (abs(F[j][5 + i]) + 1e-300) + 1e-15
        # non-relativistic limit of F^j(B^i) = B^i v^j - B^j v^i  (d_t B = curl(v x B)), G-3
    Ps = np.array([1.0, 1.0, 1e-6, 2e-6, 0, 0.3, 0.7, 0.0])
    F1 = og.prim_to_F(m, og.minkowski(), 1.0, 1, Ps)
    assert abs(F1[6] - (0.7 * 1e-6 - 0.3 * 2e-6)) < 1e-15


def test_rescale_factors_closed_form():
    # eqs 41-42 with chi = phi cs^2 tau: tau cancels
    m = og.model(nvar=10, gam=5.0 / 3.0, phi=0.7, psi=1.9)
    P = np.array([0.3, 1.7, 0, 0, 0, 1, 0, 0, 0.1, 0.2])
    cs2 = (5 / 3) * (2 / 3) * 1.7 / (0.3 + 5 / 3 * 1.7)
    Th = (2 / 3) * 1.7 / 0.3
    for tau in (1.0, 0.1, 37.0):
        fq, fd = og.rescale_factors(m, tau, P)
        assert abs(fq - 1 / np.sqrt(0.7 * cs2 * 0.3 * Th * Th)) < 1e-14 * fq
        assert abs(fd - 1 / np.sqrt(1.9 * cs2 * 0.3 * Th)) < 1e-14 * fd


# ---------------------------------------------------------------- P-12a geometry identities (C-10)
def test_kerr_mks_identities():
    a, h = 0.9375, 0.3
    for X1, X2 in ((np.log(1.3), 0.05), (np.log(2.0), 0.5), (np.log(12.0), 0.27), (np.log(40.0), 0.93)):
        g = og.kerr_mks(a, h, X1, X2)
        gcov, gcon, sg, alpha = og.geom_arrays(g)
        assert np.max(abs(gcov @ gcon - np.eye(4))) < 1e-12
        assert np.allclose(gcov, gcov.T)
        r = np.exp(X1); th = np.pi * X2 + 0.5 * (1 - h) * np.sin(2 * np.pi * X2)
        Sig = r * r + a * a * np.cos(th) ** 2
        detL = r * np.pi * (1 + (1 - h) * np.cos(2 * np.pi * X2))
        assert abs(sg - Sig * np.sin(th) * detL) < 1e-12 * sg
        assert abs(sg - np.sqrt(-np.linalg.det(gcov))) < 1e-10 * sg
        assert abs(alpha - 1 / np.sqrt(-gcon[0, 0])) < 1e-15
        # connection: symmetric, metric compatible  d_l g_mn = Gamma_mnl + Gamma_nml (central FD check)
        conn = og.kerr_mks_conn(a, h, X1, X2)
        assert np.max(abs(conn - conn.transpose(0, 2, 1))) < 1e-13 * abs(conn).max()
        low = np.einsum("kl,lmn->kmn", gcov, conn)      # Gamma_{k m n}
        d = 1e-5
        for l, (d1, d2) in ((1, (d, 0)), (2, (0, d))):
            gp = og.geom_arrays(og.kerr_mks(a, h, X1 + d1, X2 + d2))[0]
            gm = og.geom_arrays(og.kerr_mks(a, h, X1 - d1, X2 - d2))[0]
            dg = (gp - gm) / (2 * d)
            assert np.max(abs(dg - (low[:, :, l] + low[:, :, l].T))) < 1e-6 * max(1, abs(dg).max())
        for l in (0, 3):                                  # stationary, axisymmetric
            assert np.max(abs(low[:, :, l] + low[:, :, l].T)) < 1e-12 * max(1, abs(low).max())


def test_kerr_a0_is_schwarzschild_ingoing():
    g = og.kerr_mks(0.0, 1.0, np.log(6.0), 0.5)    # h=1: theta = pi X2
    gcov = og.geom_arrays(g)[0]
    r = 6.0
    assert abs(gcov[0, 0] + (1 - 2 / r)) < 1e-14
    assert abs(gcov[0, 1] - (2 / r) * r) < 1e-13
    assert abs(gcov[1, 1] - (1 + 2 / r) * r * r) < 1e-12
    assert abs(gcov[2, 2] - r * r * np.pi ** 2) < 1e-11
    assert abs(gcov[3, 3] - r * r) < 1e-12 and gcov[0, 3] == 0


def test_minkowski_geometry():
    gcov, gcon, sg, alpha = og.geom_arrays(og.minkowski())
    assert np.array_equal(gcov, np.diag([-1.0, 1, 1, 1])) and np.array_equal(gcon, gcov) and sg == 1 and alpha == 1


def test_kerr_polar_axis_face_is_finite():
    """C-21: on a face lying on the polar axis (X2 = 0 or 1) sin(theta) = 0 and the metric is singular; the floor
    |sin theta| >= 1e-20 keeps g^{mu nu} finite (g g^-1 = 1 still holds) while sqrt(-g) ~ 1e-20 shuts the flux
    through the axis off.  Away from the axis the floor is inactive (bit-identical metric)."""
    for X2 in (0.0, 1.0):
        g = og.kerr_mks(0.9375, 0.3, np.log(5.0), X2)
        gcov, gcon, sg, al = og.geom_arrays(g)
        assert np.isfinite(gcov).all() and np.isfinite(gcon).all() and np.isfinite(al)
        assert 0.0 < sg < 1e-12      # X2 = 1: sin(pi) = 1.2e-16 in fp64, already non-zero; X2 = 0: the floor
        I = gcov @ gcon
        assert abs(I - np.eye(4)).max() < 1e-12
    g1 = og.geom_arrays(og.kerr_mks(0.9375, 0.3, np.log(5.0), 1e-3))
    assert g1[2] > 1e-3      # floor inactive: sqrt(-g) = Sigma sin(theta) |det L| is of order r^3 * 2 pi X2
