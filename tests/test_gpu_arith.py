"""The library's speculative fp64 division / reciprocal / square root (csrc/fp64ops.cuh) against the IEEE operators
on the device, bit for bit.  This is what lets the kernels run straight-line Newton-Raphson sequences and still be
bit-identical to the oracle's `/` and `sqrt`."""
import pytest

from common import cuda_grid

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def grid():
    return cuda_grid(dict(n1=8, n2=8, n3=1, dim=2, nvar=8))


@pytest.mark.parametrize("seed", [0, 1702, 987654321])
def test_speculative_arithmetic_is_correctly_rounded_in_range(grid, seed):
    n = 1 << 28
    bad, accepted = grid.arith_selftest(n, seed=seed, wide=False)
    assert bad == [0, 0, 0, 0, 0]
    assert accepted == n          # every in-range sample takes the straight-line path


@pytest.mark.parametrize("seed", [3, 1106])
def test_guard_rejects_what_the_straight_line_code_gets_wrong(grid, seed):
    """Whole fp64 range: zeros, subnormals, infinities, NaNs, negative radicands, quotients that overflow or turn
    subnormal.  Whatever the guard lets through must still equal the IEEE result."""
    n = 1 << 28
    bad, accepted = grid.arith_selftest(n, seed=seed, wide=True)
    assert bad == [0, 0, 0, 0, 0]
    assert 0 < accepted < n


@pytest.mark.parametrize("scale,nvar", [(1e150, 8), (1e150, 10), (1e-140, 8)])
def test_replay_path_on_extreme_magnitudes(scale, nvar):
    """States scaled far outside the speculative arithmetic's safe range [2^-480, 2^480) (the equations are
    homogeneous in rho, u, B^2, q, dP): every face, zone and Newton solve trips a guard and is replayed with the exact
    operators, in every kernel.  The result -- converged at 1e150, non-finite at 1e-140 where the finite-difference
    step of eq 23 swamps the state -- must still be the oracle's, bit for bit, statistics included."""
    import numpy as np

    import oracle as og
    from common import oracle_grid, random_smooth_state, to_dev
    gk = dict(n1=37, n2=21, n3=1, dim=2, nvar=nvar, recon=og.MP5, rtol=1e-14, kmax=8, lsmax=5)
    go, gc = oracle_grid(gk), cuda_grid(gk)
    P = random_smooth_state(go, nvar, np.random.default_rng(3), amp=0.05)
    P[0] *= scale
    P[1] *= scale
    P[5:8] *= np.sqrt(scale)
    if nvar == 10:
        P[8] *= scale
        P[9] *= scale
    go.fill_ghosts(P)
    dt = go.choose_dt(P)
    Po, dP = P.copy(), to_dev(P)
    so = go.timestep(Po, dt)
    _, sc = gc.timestep(dP, dt, want_stats=True)
    for s in range(2):
        assert list(so.iters_hist[s]) == list(sc.iters_hist[s])
        assert so.unconverged[s] == sc.unconverged[s]
    assert np.array_equal(go.interior(dP.cpu().numpy()), go.interior(Po), equal_nan=True)
    if scale > 1:
        assert so.unconverged[1] == 0 and np.isfinite(go.interior(Po)).all()
