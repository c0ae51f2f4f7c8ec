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
