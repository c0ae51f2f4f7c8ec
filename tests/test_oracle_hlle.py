"""Pins of the oracle's HLLE flux (NEXT-4; eq 18).  The paper states the formula and three
properties, which are the pins: "the two [LLF and HLLE] are identical when the maximum left-going and right-going
speeds are equal"; HLLE "switches to upwind reconstruction when all characteristic speeds have the same sign";
and, as for any numerical flux, F(P, P) = F(P)."""
import numpy as np
import pytest

import oracle as og
from common import oracle_grid, random_smooth_state


def states(rng, n=10):
    Fm, Fp, Um, Up = (rng.standard_normal(n) for _ in range(4))
    return Fm, Fp, Um, Up


def test_hlle_equals_llf_for_equal_speeds():
    rng = np.random.default_rng(0)
    for _ in range(20):
        Fm, Fp, Um, Up = states(rng)
        c = rng.uniform(0.1, 1.0)
        assert np.allclose(og.hlle(Fm, Fp, Um, Up, c, c), og.llf(Fm, Fp, Um, Up, c), rtol=1e-14, atol=1e-15)


def test_hlle_is_upwind_when_all_speeds_have_one_sign():
    rng = np.random.default_rng(1)
    Fm, Fp, Um, Up = states(rng)
    # everything moves right: the left state's flux (to the rounding of c F / c); everything moves left: the right's
    assert np.allclose(og.hlle(Fm, Fp, Um, Up, 0.7, 0.0), Fm, rtol=4e-16, atol=0)
    assert np.allclose(og.hlle(Fm, Fp, Um, Up, 0.0, 0.4), Fp, rtol=4e-16, atol=0)


def test_hlle_formula_eq18():
    rng = np.random.default_rng(2)
    Fm, Fp, Um, Up = states(rng)
    cR, cL = 0.8, 0.3
    ref = (cR * Fm + cL * Fp - cR * cL * (Up - Um)) / (cL + cR)
    assert np.allclose(og.hlle(Fm, Fp, Um, Up, cR, cL), ref, rtol=1e-15, atol=0)
    assert np.allclose(og.hlle(Fm, Fm, Um, Um, cR, cL), Fm, rtol=1e-15, atol=1e-16)   # consistency


@pytest.mark.parametrize("dim,nvar", [(2, 8), (3, 10)])
def test_hlle_scheme_conserves_and_stays_close_to_llf(dim, nvar):
    """On smooth subsonic data both solvers are consistent discretisations of the same equations: one step with HLLE
    conserves, and differs from the LLF step only at the level of the (different) numerical dissipation."""
    n = (14, 11, 9 if dim == 3 else 1)
    out = {}
    for rs in (og.LLF, og.HLLE):
        g = oracle_grid(dict(n1=n[0], n2=n[1], n3=n[2], dim=dim, nvar=nvar, recon=og.MP5, riemann=rs))
        P = random_smooth_state(g, nvar, np.random.default_rng(4), amp=0.05)
        g.fill_ghosts(P)
        m, geo = og.model(nvar=nvar), og.minkowski()
        Pi = g.interior(P).reshape(nvar, -1)
        U0 = sum(og.prim_to_U(m, geo, 1.0, Pi[:, z]) for z in range(Pi.shape[1]))
        dt = g.choose_dt(P) if rs == og.LLF else out["dt"]
        out["dt"] = dt
        st = g.timestep(P, dt)
        assert st.unconverged[1] == 0
        Pi = g.interior(P).reshape(nvar, -1)
        U1 = sum(og.prim_to_U(m, geo, 1.0, Pi[:, z]) for z in range(Pi.shape[1]))
        assert np.max(abs(U1[:8] - U0[:8])) < 1e-11 * abs(U0).max()
        out[rs] = g.interior(P).copy()
    d = abs(out[og.HLLE] - out[og.LLF]).max()
    assert 0 < d < 1e-3
