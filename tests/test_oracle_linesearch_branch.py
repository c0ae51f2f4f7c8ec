"""Pin of the backtracking branch of the oracle's newton_zone (section 3.2: the acceptance test
of L223, eq 25 at L230) and of what the paper leaves open around it (reading C-14: a non-finite trial halves
lambda; after lsmax rejected trials the last trial is taken and the zone is flagged).

One Newton iteration of the standalone inversion (og.invert with kmax = 1) is replayed here in plain numpy from
og.prim_to_U alone (pinned by Table 1 / the shock table elsewhere): the residual R(P) = (U(P) - U*) / ||U*||, the
finite-difference Jacobian of eqs 22-23 (L198-214), delta P from numpy.linalg.solve (LAPACK), and the line search
typed from the paper's three bullets.  The oracle's iterate, residual norm, back-track count and status word must
be the replay's.  Zones are config 2's with guesses far enough (50 % scatter) that the full step is rejected in
a fair share of them."""
import numpy as np
import pytest

import oracle as og
from paper_1702_01106_b200 import workloads

FD_EPS, EPS_BT = 4e-8, 1e-4


def _residual(m, geo, Ustar, P):
    """R(P) = (U(P) - U*) / ||U*||.  The norm is summed left to right and applied as a reciprocal, the rounding order
    of the oracle: config 2's Jacobians have condition numbers up to ~1e8, and a last-bit difference in R, divided
    by the 4e-8 P of eq 23, would otherwise show up in delta P at 1e-4."""
    s2 = 0.0
    for x in Ustar:
        s2 += x * x
    with np.errstate(all="ignore"):
        return (og.prim_to_U(m, geo, 1.0, P) - Ustar) * (1.0 / np.sqrt(s2))


def _replay_one_iteration(m, geo, Ustar, P, lsmax):
    """Section 3.1-3.2 written out.  Returns (P_new, ||R(P_new)||, lambdas tried, accepted, f0)."""
    n = len(P)
    R0 = _residual(m, geo, Ustar, P)
    f0 = R0 @ R0
    J = np.zeros((n, n))
    for j in range(n):
        Pe = P.copy()
        Pe[j] = FD_EPS if abs(P[j]) < 5 * FD_EPS else (1 + FD_EPS) * P[j]          # eq 23 with small()
        J[:, j] = (_residual(m, geo, Ustar, Pe) - R0) * (1.0 / (Pe[j] - P[j]))      # eq 22
    dP = np.linalg.solve(J, -R0)                                                    # eq 21
    lam, lams, accepted = 1.0, [], False
    for ls in range(lsmax + 1):
        lams.append(lam)
        Pt = P + lam * dP
        Rt = _residual(m, geo, Ustar, Pt)
        ft = Rt @ Rt
        if np.sqrt(ft) < np.sqrt(f0) * (1 - EPS_BT * lam):                          # L223
            accepted = True
            break
        if ls == lsmax:
            break
        lam = f0 / (ft + (2 * lam - 1) * f0) * lam ** 2 if np.isfinite(ft) else lam / 2   # eq 25 | C-14
    return Pt, np.sqrt(ft), lams, accepted, f0, dP


def _zones(nvar, nz, seed, scatter):
    Pt, _ = workloads.config2(nz, seed=seed, nvar=nvar)
    rng = np.random.Generator(np.random.PCG64(seed + 1))
    guess = Pt * (1 + scatter * rng.uniform(-1, 1, Pt.shape))
    return Pt, guess


@pytest.mark.parametrize("nvar,scatter", [(8, 0.5), (10, 0.5)])
def test_one_iteration_with_backtracking_equals_the_papers_procedure(nvar, scatter):
    nz, lsmax = 400, 8
    m, geo = og.model(nvar=nvar), og.minkowski()
    Pt, guess = _zones(nvar, nz, 77, scatter)
    U = np.stack([og.prim_to_U(m, geo, 1.0, Pt[:, z]) for z in range(nz)], axis=1)
    sv = og.solver(fd_eps=FD_EPS, eps_bt=EPS_BT, rtol=1e-12, kmax=1, lsmax=lsmax)
    n_bt = n_second = n_nonfinite = n_checked = 0
    for z in range(nz):
        Pn, rn, lams, acc, f0, dP = _replay_one_iteration(m, geo, U[:, z], guess[:, z].copy(), lsmax)
        Po, it, st, ro, bt = og.invert(m, sv, U[:, z:z + 1], guess[:, z:z + 1])
        if not np.isfinite(rn):
            continue
        # near-ties of the acceptance test could go either way between two roundings of delta P: skip them
        margin = abs(rn - np.sqrt(f0) * (1 - EPS_BT * lams[-1])) / np.sqrt(f0)
        if margin < 1e-6:
            continue
        n_checked += 1
        assert it[0] == 1
        assert bt == len(lams) - 1, (z, bt, lams)
        scale = np.abs(guess[:, z]) + np.abs(dP)
        assert (np.abs(Po[:, 0] - Pn) <= 1e-7 * scale).all(), (z, lams, Po[:, 0], Pn)
        assert abs(ro[0] - rn) <= 1e-6 * max(rn, 1e-12), (z, ro[0], rn)
        assert bool(st[0] & og.ST_LS_EXHAUSTED) == (not acc)
        if acc:
            # what the oracle returns is an improvement by the margin of L223
            assert ro[0] < np.sqrt(f0) * (1 - EPS_BT * lams[-1]) * (1 + 1e-9)
        if len(lams) > 1:
            n_bt += 1
            R1 = _residual(m, geo, U[:, z], guess[:, z] + dP)
            f1 = R1 @ R1
            if np.isfinite(f1):
                lam2 = f0 / (f1 + f0)                     # eq 25 at lambda_old = 1
                assert abs(lams[1] - lam2) < 1e-15
                assert 0 < lam2 < 0.5 + 1e-4              # a rejected full step has f1 > ~f0
                if len(lams) == 2 and acc:
                    n_second += 1
                    assert (np.abs(Po[:, 0] - (guess[:, z] + lam2 * dP)) <= 1e-7 * scale).all()
            else:
                n_nonfinite += 1
                assert lams[1] == 0.5
    assert n_checked > 0.9 * nz
    assert n_bt >= 20 and n_second >= 5, (n_bt, n_second)
    if nvar == 10:
        assert n_nonfinite >= 3, n_nonfinite             # full steps into u < 0: Theta^{1/2} is not a number


def test_exhausted_line_search_takes_the_last_trial_and_sets_the_bit():
    """lsmax = 0: the full Newton step is taken whether or not it passes L223; lsmax = 1: a zone whose second trial
    fails too ends at P + lambda_2 delta P (lambda_2 from eq 25, or 1/2 after a non-finite full step).  Both carry
    ST_LS_EXHAUSTED, neither back-tracks more than lsmax times; a last trial that is not a number is still the
    one taken, and the zone is flagged non-finite as well."""
    nz = 400
    geo = og.minkowski()
    seen = {0: 0, 1: 0, "nonfinite": 0}
    for lsmax, nvar, scatter in ((0, 8, 0.7), (1, 10, 0.9)):
        m = og.model(nvar=nvar)
        Pt, guess = _zones(nvar, nz, 91, scatter)
        U = np.stack([og.prim_to_U(m, geo, 1.0, Pt[:, z]) for z in range(nz)], axis=1)
        sv = og.solver(fd_eps=FD_EPS, eps_bt=EPS_BT, rtol=1e-12, kmax=1, lsmax=lsmax)
        Po, it, st, ro, bt = og.invert(m, sv, U, guess)
        assert bt <= lsmax * nz
        for z in range(nz):
            Pn, rn, lams, acc, f0, dP = _replay_one_iteration(m, geo, U[:, z], guess[:, z].copy(), lsmax)
            if acc:
                continue
            if np.isfinite(rn) and abs(rn - np.sqrt(f0) * (1 - EPS_BT * lams[-1])) < 1e-6 * np.sqrt(f0):
                continue
            assert len(lams) == lsmax + 1
            assert st[z] & og.ST_LS_EXHAUSTED and not st[z] & og.ST_CONVERGED
            scale = np.abs(guess[:, z]) + np.abs(dP)
            assert (np.abs(Po[:, z] - (guess[:, z] + lams[-1] * dP)) <= 1e-7 * scale).all()
            if np.isfinite(rn):
                seen[lsmax] += 1
                assert not st[z] & og.ST_NONFINITE
                assert abs(ro[z] - rn) <= 1e-6 * rn
                assert ro[z] >= np.sqrt(f0) * (1 - EPS_BT * lams[-1]) * (1 - 1e-9)  # it really was a rejected trial
            else:
                seen["nonfinite"] += 1
                assert st[z] & og.ST_NONFINITE and not np.isfinite(ro[z])
    assert seen[0] >= 20 and seen[1] >= 2 and seen["nonfinite"] >= 3, seen


def test_whole_solve_with_backtracking_descends():
    """Whole solves (kmax = 30) of far guesses: a zone the oracle calls converged has ||R|| < rtol by an independent
    evaluation; a zone whose line search never ran out ends no higher than it started (every accepted step
    descends, L223); the back-track total is at least what the first iterations alone need."""
    nvar, nz = 8, 300
    m, geo = og.model(nvar=nvar), og.minkowski()
    Pt, guess = _zones(nvar, nz, 123, 0.5)
    U = np.stack([og.prim_to_U(m, geo, 1.0, Pt[:, z]) for z in range(nz)], axis=1)
    sv = og.solver(fd_eps=FD_EPS, eps_bt=EPS_BT, rtol=1e-12, kmax=30, lsmax=8)
    Po, it, st, ro, bt = og.invert(m, sv, U, guess)
    conv = (st & og.ST_CONVERGED) != 0
    assert conv.mean() > 0.5
    first = 0
    for z in range(nz):
        R = _residual(m, geo, U[:, z], Po[:, z])
        rn = np.sqrt(R @ R)
        if conv[z]:
            assert rn < 1e-12 and not st[z] & (og.ST_LS_EXHAUSTED | og.ST_NONFINITE | og.ST_SINGULAR)
        if not st[z] & (og.ST_LS_EXHAUSTED | og.ST_NONFINITE | og.ST_SINGULAR):
            R0 = _residual(m, geo, U[:, z], guess[:, z])
            assert rn <= np.sqrt(R0 @ R0)
            assert abs(ro[z] - rn) <= 1e-9 * rn + 1e-300
        first += len(_replay_one_iteration(m, geo, U[:, z], guess[:, z].copy(), 8)[2]) - 1
    assert bt >= first > 0
