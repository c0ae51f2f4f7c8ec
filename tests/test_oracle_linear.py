"""Oracle pins from linear theory: Table 1 (P-1), ideal-MHD closed forms (P-3, P-13), psi_max (P-6),
shock-table flux equality (P-4).  CPU only."""
import numpy as np
import pytest

import linear_modes as lm
import oracle as og
from conftest import read_golden_table


@pytest.fixture(scope="module")
def emhd_pencil(table1):
    P0, dP, w, k = table1
    m = og.model(nvar=10, gam=4.0 / 3.0, phi=1.0, psi=1.0)
    A, GP = lm.pencil(m, P0, tau=1.0)
    return m, A, GP


def test_table1_null_vector(table1, emhd_pencil):
    """the printed (dP, omega) solves the oracle's linearised equations."""
    P0, dP, w, k = table1
    m, A, GP = emhd_pencil
    M = lm.char_matrix(A, GP, w, k)
    r = np.linalg.norm(M @ dP) / (np.linalg.norm(dP) * np.linalg.norm(M, 2))
    assert r < 1e-9, r


def test_table1_eigenvalue_and_vector(table1, emhd_pencil):
    P0, dP, w, k = table1
    m, A, GP = emhd_pencil
    ev, vec = lm.eigenmodes(A, GP, k)
    i = np.argmin(abs(ev - w))
    assert abs(ev[i] - w) < 1e-9
    v = vec[:, i] / vec[1, i] * dP[1]
    assert np.max(abs(v - dP)) < 1e-8
    # the spectrum also holds the Alfven pair  w = +- i k.B / sqrt(rho + gamma u + b^2)  (P-13)
    wA = (k[0] * 0.1 + k[1] * 0.3) / np.sqrt(1 + 4.0 / 3.0 * 2 + 0.1)
    assert min(abs(ev - 1j * wA)) < 1e-8 and min(abs(ev + 1j * wA)) < 1e-8


@pytest.mark.parametrize("variant", ["eq32_printed_sign", "gamma_5_3", "phi_2", "psi_half"])
def test_table1_rejects_wrong_readings(table1, emhd_pencil, variant):
    """The pin has teeth: eq 32's printed sign (G-3), another adiabatic index or other closure
    coefficients all miss the printed mode grossly."""
    P0, dP, w, k = table1
    m, A, GP = emhd_pencil
    if variant == "eq32_printed_sign":
        A = [a.copy() for a in A]
        for j in (1, 2, 3):
            A[j][5:8, :] *= -1.0
    else:
        kw = {"gamma_5_3": dict(gam=5.0 / 3.0), "phi_2": dict(phi=2.0), "psi_half": dict(psi=0.5)}[variant]
        A, GP = lm.pencil(og.model(nvar=10, **{**dict(gam=4.0 / 3.0, phi=1.0, psi=1.0), **kw}), P0, tau=1.0)
    M = lm.char_matrix(A, GP, w, k)
    r = np.linalg.norm(M @ dP) / (np.linalg.norm(dP) * np.linalg.norm(M, 2))
    assert r > 1e-3


def test_ideal_mhd_dispersion_closed_form():
    """P-3/P-13: relativistic magnetosonic quartic and Alfven frequency in the fluid rest frame."""
    gam = 4.0 / 3.0
    m = og.model(nvar=8, gam=gam)
    P0 = np.array([1.0, 2.0, 0, 0, 0, 0.1, 0.3, 0.0])
    A, GP = lm.pencil(m, P0)
    k = np.array([2 * np.pi, 2 * np.pi, 0.0])
    ev, vec = lm.eigenmodes(A, GP, k)
    rho, u, B = 1.0, 2.0, np.array([0.1, 0.3, 0.0])
    bsq = B @ B
    cs2 = gam * (gam - 1) * u / (rho + gam * u)
    E = rho + gam * u + bsq
    va2 = bsq / E
    kva = (k @ B) / np.sqrt(E)
    k2 = k @ k
    b_ = k2 * (va2 + cs2 * (1 - va2)) + cs2 * kva ** 2
    c_ = k2 * cs2 * kva ** 2
    w2f = 0.5 * (b_ + np.sqrt(b_ * b_ - 4 * c_))
    w2s = 0.5 * (b_ - np.sqrt(b_ * b_ - 4 * c_))
    for wref in (np.sqrt(w2f), np.sqrt(w2s), abs(kva)):
        assert min(abs(ev - 1j * wref)) < 1e-8 * wref + 1e-9, (wref, ev)
        assert min(abs(ev + 1j * wref)) < 1e-8 * wref + 1e-9
    assert abs(np.sqrt(w2f) - 4.4145848550) < 1e-9      # value quoted in SURVEY P-3 (closed form)
    # fast eigenvector: adiabatic  du/drho = gamma u/rho, and k.dB = 0
    i = np.argmin(abs(ev - 1j * np.sqrt(w2f)))
    v = lm.normalise_phase(vec[:, i], 0)
    assert abs(v[1] / v[0] - gam * u / rho) < 1e-7
    assert abs(k[0] * v[5] + k[1] * v[6]) < 1e-7
    assert np.max(abs(v.imag)) < 1e-7


def test_psi_max_causal_bound():
    """P-6, L325: with psi = phi and cs^2 = gamma - 1 the corrected sound speed reaches 1 at psi ~ 1.3
    (gamma = 4/3) and ~ 0.29 (gamma = 5/3).  B = 0 so vmax^2 = c~s^2; cs^2 -> gamma-1 as u/rho -> inf."""
    g = og.minkowski()
    for gam, psi_max in ((4.0 / 3.0, 1.3), (5.0 / 3.0, 0.29)):
        P = np.array([1e-12, 1.0, 0, 0, 0, 1e-30, 0, 0, 0, 0])
        def v2(psi):
            return og.vmax2(og.model(nvar=10, gam=gam, phi=psi, psi=psi), g, 1.0, P)
        assert abs(v2(psi_max) - 1.0) < 0.01
        lo, hi = 0.0, 3.0
        for _ in range(60):
            mid = 0.5 * (lo + hi)
            lo, hi = (mid, hi) if v2(mid) < 1 else (lo, mid)
        assert abs(lo - psi_max) < 0.02 * max(1, psi_max) + 0.005


def test_shock_table_flux_equality():
    """P-4, L517-528: F^1(P_left) = F^1(P_right) to the table's 9 digits; gamma = 5/3 fails."""
    t = read_golden_table("shock_table_ideal_mhd.txt")
    names = ["rho", "u", "u1", "u2", "u3", "B1", "B2", "B3"]
    PL = np.array([t[n][0] for n in names])
    PR = np.array([t[n][1] for n in names])
    g = og.minkowski()
    m = og.model(nvar=8, gam=4.0 / 3.0)
    FL, FR = og.prim_to_F(m, g, 1.0, 1, PL), og.prim_to_F(m, g, 1.0, 1, PR)
    # left state: rho u^1 = 1, T^1_0 = -(rho+u+P) u^1 u^t = -(7/3) sqrt 2, T^1_1 = (7/3) + 1/3 (B ~ 1e-5 negligible)
    assert abs(FL[0] - 1.0) < 1e-12
    assert abs(FL[1] + 7.0 / 3.0 * np.sqrt(2.0)) < 1e-9
    assert abs(FL[2] - 8.0 / 3.0) < 1e-9
    assert np.max(abs(FL[:3] - FR[:3]) / abs(FL[:3])) < 5e-8
    m53 = og.model(nvar=8, gam=5.0 / 3.0)
    FL, FR = og.prim_to_F(m53, g, 1.0, 1, PL), og.prim_to_F(m53, g, 1.0, 1, PR)
    assert np.max(abs(FL[:3] - FR[:3]) / abs(FL[:3])) > 0.1
