"""Pins of og_choose_dt and of the speeds[] reduction of og_stage_prepare (reading C-15 of PAPER.md L651 "courant
factor" with the LLF speed bound of L164 and eqs 43-48):

    speeds[d] = max_z  max(c^d_face(z), c^d_face(z+1)) / dX^d         d = 1..3
    speeds[3] = max_z  sum_d max(c^d_face(z), c^d_face(z+1)) / dX^d
    dt        = cfl / speeds[3]

Nothing here calls the oracle for an expected value.  The expected speeds are closed forms written out in numpy:
the ideal-MHD v_max^2 = c_s^2 + v_A^2 - c_s^2 v_A^2 (eq 43 without the extended-MHD terms), and, for a fluid that
moves, the two roots of the comoving dispersion relation omega'^2 = v_max^2 k'^2 for a wave vector along X^d
(which is what eqs 45-48 solve): with s = omega/k, gamma the Lorentz factor and v_d the velocity along X^d,

    [gamma^2 (1-vm^2) + vm^2] s^2 - 2 gamma^2 (1-vm^2) v_d s + gamma^2 (1-vm^2) v_d^2 - vm^2 = 0 .

A sum taken where a maximum belongs (or the reverse), a wrong 1/dX^d, a dropped direction, or a face speed that
looks at one side only each fail one of the cases below."""
import numpy as np
import pytest

import oracle as og

GAM = 4.0 / 3.0


def _comoving_b2(ut, B):
    """b^2 of a fluid with u~^i = ut in Minkowski space: b^0 = B.u, b^i = (B^i + b^0 u^i)/u^0."""
    u0 = np.sqrt(1.0 + ut @ ut)
    b0 = B @ ut
    bi = (B + b0 * ut) / u0
    return bi @ bi - b0 * b0


def _vmax_ideal(rho, u, ut, B):
    b2 = _comoving_b2(np.asarray(ut, float), np.asarray(B, float))
    w = rho + GAM * u
    cs2 = GAM * (GAM - 1.0) * u / w
    va2 = b2 / (w + b2)
    return np.sqrt(cs2 + va2 - cs2 * va2)


def _cmax_closed_form(rho, u, ut, B, d):
    """max |omega/k| over the two roots of the quadratic in the module docstring, direction d = 0, 1, 2."""
    ut = np.asarray(ut, float)
    vm = _vmax_ideal(rho, u, ut, B)
    g2 = 1.0 + ut @ ut
    vd = ut[d] / np.sqrt(g2)
    a = g2 * (1.0 - vm * vm)
    r = np.roots([a + vm * vm, -2.0 * a * vd, a * vd * vd - vm * vm])
    assert np.isreal(r).all()
    return np.abs(r.real).max()


def _grid(dim, n, xend, cfl=0.37, nvar=8):
    return og.Grid(n[0], n[1], n[2], dim=dim, xend=xend, nvar=nvar, recon=og.MINMOD, cfl=cfl, bc=og.BC_PERIODIC)


def _fill(g, prim):
    P = g.zeros()
    for v, x in enumerate(prim):
        P[v] = x
    return P


@pytest.mark.parametrize("dim,n,xend", [(1, (24, 1, 1), (1.7, 1, 1)), (2, (12, 10, 1), (1.0, 0.3, 1)),
                                        (3, (8, 6, 10), (1.0, 0.45, 3.1))])
def test_choose_dt_uniform_state_at_rest(dim, n, xend):
    """Every c^d is v_max (eq 43), so dt = cfl / (v_max sum_d 1/dX^d) with unequal dX^d; speeds[d] = v_max/dX^d."""
    g = _grid(dim, n, xend)
    rho, u, B = 1.3, 0.7, np.array([0.2, -0.35, 0.1])
    P = _fill(g, [rho, u, 0, 0, 0, *B])
    vm = _vmax_ideal(rho, u, np.zeros(3), B)
    inv = [n[a] / xend[a] for a in range(dim)]
    _, _, sp = g.stage_prepare(P, P, 1.0)
    for a in range(dim):
        assert abs(sp[a] - vm * inv[a]) < 1e-13 * vm * inv[a]
    for a in range(dim, 3):
        assert sp[a] == 0.0
    assert abs(sp[3] - vm * sum(inv)) < 1e-13 * sp[3]
    dt = g.choose_dt(P)
    assert abs(dt - 0.37 / (vm * sum(inv))) < 1e-13 * dt
    if dim > 1:         # a maximum over directions instead of the sum would give this
        assert abs(dt - 0.37 / (vm * max(inv))) > 0.1 * dt


def test_choose_dt_rest_state_extended_mhd_uses_eq43():
    """nvar = 10: v_max of eq 43 with the conduction and viscosity terms (pinned by psi_max of L325 in
    test_oracle_pins.py) exceeds the ideal one, and dt follows it."""
    g = _grid(2, (10, 8, 1), (1.0, 0.6, 1), nvar=10)
    prim = [1.0, 0.5, 0, 0, 0, 0.1, 0.2, 0.0, 0.0, 0.0]
    P = _fill(g, prim)
    m = og.model(nvar=10)
    vm = np.sqrt(og.vmax2(m, og.minkowski(), 1.0, np.array(prim)))
    assert vm > _vmax_ideal(1.0, 0.5, np.zeros(3), np.array([0.1, 0.2, 0.0])) + 1e-3
    dt = g.choose_dt(P)
    assert abs(dt - 0.37 / (vm * (10 / 1.0 + 8 / 0.6))) < 1e-13 * dt


def test_choose_dt_uniform_boosted_state():
    """A fluid moving obliquely: each direction has its own c^d from the dispersion relation (relativistic velocity
    addition along the motion, time dilation across it); a reduction that mixed the directions up, or used dX^1
    for every direction, fails."""
    n, xend = (10, 12, 8), (1.0, 2.9, 0.55)
    g = _grid(3, n, xend)
    rho, u, ut, B = 0.9, 1.1, np.array([0.8, -0.25, 0.1]), np.array([0.3, 0.1, -0.2])
    P = _fill(g, [rho, u, *ut, *B])
    c = [_cmax_closed_form(rho, u, ut, B, d) for d in range(3)]
    assert c[0] > c[1] + 0.1 and c[0] > c[2] + 0.1        # the case separates the directions
    inv = [n[a] / xend[a] for a in range(3)]
    _, _, sp = g.stage_prepare(P, P, 1.0)
    for a in range(3):
        assert abs(sp[a] - c[a] * inv[a]) < 1e-12 * sp[a], (a, sp[a], c[a] * inv[a])
    want = sum(c[a] * inv[a] for a in range(3))
    assert abs(sp[3] - want) < 1e-12 * want
    assert abs(g.choose_dt(P) - 0.37 / want) < 1e-12 * 0.37 / want


def test_cmax_along_the_motion_is_velocity_addition():
    """The quadratic above, for motion along X^1 only, is the textbook velocity addition: checks the closed form
    this file uses against a second, independent one."""
    rho, u, B = 1.0, 2.0, np.array([0.1, 0.3, 0.0])
    ut = np.array([0.6, 0.0, 0.0])
    vm = _vmax_ideal(rho, u, ut, B)
    v = ut[0] / np.sqrt(1 + ut[0] ** 2)
    want = max(abs((v + vm) / (1 + v * vm)), abs((v - vm) / (1 - v * vm)))
    assert abs(_cmax_closed_form(rho, u, ut, B, 0) - want) < 1e-14
    gl = np.sqrt(1 + ut[0] ** 2)
    assert abs(_cmax_closed_form(rho, u, ut, B, 1) - vm / np.sqrt(gl ** 2 * (1 - vm ** 2) + vm ** 2)) < 1e-14


def test_choose_dt_is_max_over_zones_of_the_sum_over_directions():
    """Plateaus A | N | B | N along X^1 (each wider than the stencil, so minmod slopes vanish and every face sees
    the two plateau states): A is fast along X^1, B along X^2, N is at rest.  The zone speed in direction d is the
    larger of its two face speeds, a face speed the larger of its two sides (L164), so
    speed_d(z) = max(c^d(z-1), c^d(z), c^d(z+1)); the sum of the per-direction maxima over the grid is larger than
    the maximum of the sums, and dt must come from the latter."""
    n1, n2 = 32, 6
    xend = (1.0, 0.21, 1)
    g = _grid(2, (n1, n2, 1), xend)
    rho, u, B = 1.0, 0.4, np.array([0.1, 0.1, 0.05])
    states = {"A": np.array([1.6, 0.0, 0.0]), "N": np.zeros(3), "B": np.array([0.0, 0.9, 0.0])}
    layout = ["A"] * 8 + ["N"] * 8 + ["B"] * 8 + ["N"] * 8
    P = g.zeros()
    ng = 3
    c = np.zeros((2, n1))
    for i, s in enumerate(layout):
        P[0, :, :, ng + i], P[1, :, :, ng + i] = rho, u
        for k in range(3):
            P[2 + k, :, :, ng + i] = states[s][k]
            P[5 + k, :, :, ng + i] = B[k]
        for d in range(2):
            c[d, i] = _cmax_closed_form(rho, u, states[s], B, d)
    inv = [n1 / xend[0], n2 / xend[1]]
    zone = np.zeros((2, n1))
    zone[0] = np.maximum(c[0], np.maximum(np.roll(c[0], 1), np.roll(c[0], -1)))       # neighbours along X^1
    zone[1] = c[1]                                                                    # uniform along X^2
    want = [zone[0].max() * inv[0], zone[1].max() * inv[1]]
    want_sum = (zone[0] * inv[0] + zone[1] * inv[1]).max()
    assert want[0] + want[1] > 1.05 * want_sum            # the two reductions differ on this state
    _, _, sp = g.stage_prepare(P, P, 1.0)
    assert abs(sp[0] - want[0]) < 1e-12 * want[0]
    assert abs(sp[1] - want[1]) < 1e-12 * want[1]
    assert abs(sp[3] - want_sum) < 1e-12 * want_sum
    dt = g.choose_dt(P)
    assert abs(dt - 0.37 / want_sum) < 1e-12 * dt
