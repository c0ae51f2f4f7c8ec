"""grim_invert_primitives_static: the inversion for callers that cannot allocate device memory.

Who needs it: code that runs inside an application whose own memory pool has taken the GPU's memory at start-up (the
library's cudaMalloc would fail there, or eat memory the pool has promised to someone else), and code inside a
time-critical loop (cudaMalloc / cudaFree wait for the whole device).  Every other entry point needs a `Grid`, whose
creation allocates; this one takes the caller's input and output buffers and nothing else, and keeps its zone lists
and counters in a fixed 8 MiB array inside the library (hence the 2^20-zone limit per call).

The checks: its results equal those of `Grid.invert_primitives` -- the path the other GPU tests hold against the oracle
-- bit for bit (the tolerance those tests use: `array_equal` on primitives, residual norms, statuses and iteration
counts), on two calls in a row with different inputs and sizes, the second smaller than the first so that it runs over
whatever the first left in the shared array; and a batch beyond the limit is refused with a message that names it.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests.  It does not depend on them: it passes alone in a fresh process too (the first call then does the per-device
set-up)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SOLVER = dict(rtol=1e-12, kmax=30, lsmax=8)


def _workload(nz, nvar, seed):
    """config-2 targets (BASELINE config 2 recipe) built on the device by the library's own U(P)."""
    import torch
    import paper_1702_01106_b200 as gb
    from paper_1702_01106_b200 import workloads
    Ptrue, guess = workloads.config2(nz, seed=seed, nvar=nvar)
    g = gb.Grid(8, 8, 1, dim=2, model=nvar, **SOLVER)
    dPt = torch.from_numpy(Ptrue).cuda()
    dU = torch.empty_like(dPt)
    g.prim_to_conserved(dPt, dU)
    torch.cuda.synchronize()
    return g, dU, guess


def _outputs(nz):
    import torch
    # start from garbage so that a zone the kernel failed to write shows up
    return (torch.full((nz,), -7, dtype=torch.int32, device="cuda"),
            torch.full((nz,), -7, dtype=torch.int32, device="cuda"),
            torch.full((nz,), float("nan"), dtype=torch.float64, device="cuda"))


@pytest.mark.parametrize("nvar", [8, 10])
def test_static_inversion_equals_allocating_path_twice_in_a_row(nvar):
    import torch
    import paper_1702_01106_b200 as gb
    # first call: several thousand blocks and a ragged tail; second: smaller, other inputs, same shared scratch
    for call, (nz, seed) in enumerate([(50021, 1702), (7013, 99)]):
        g, dU, guess = _workload(nz, nvar, seed)
        P_ref = torch.from_numpy(guess.copy()).cuda()
        it_ref, st_ref, rn_ref = _outputs(nz)
        g.invert_primitives(dU, P_ref, it_ref, st_ref, rn_ref)
        P_new = torch.from_numpy(guess.copy()).cuda()
        it_new, st_new, rn_new = _outputs(nz)
        gb.invert_primitives_static(dU, P_new, it_new, st_new, rn_new, model=nvar, **SOLVER)
        torch.cuda.synchronize()
        assert torch.equal(it_new, it_ref), "iteration counts differ on call %d" % call
        assert torch.equal(st_new, st_ref), "status words differ on call %d" % call
        assert np.array_equal(rn_new.cpu().numpy(), rn_ref.cpu().numpy(), equal_nan=True)
        assert np.array_equal(P_new.cpu().numpy(), P_ref.cpu().numpy(), equal_nan=True)
        # the comparison saw real work: every zone ended, iteration counts spread over several sweeps
        assert int((st_ref & gb.ST_TERMINAL).ne(0).sum()) == nz
        assert int(it_ref.max()) > 8 and int(it_ref.min()) >= 1
        g.close()


def test_static_inversion_with_per_zone_geometry_equals_allocating_path():
    """geom != NULL (the general-metric kernel variant): a boosted, sheared but valid metric per zone."""
    import torch
    import paper_1702_01106_b200 as gb
    nz, nvar = 9001, 8
    g, dU, guess = _workload(nz, nvar, 5)
    rng = np.random.default_rng(12)
    geom = np.zeros((15, nz))
    # a diagonal metric with lapse != 1 and unequal spatial scale factors: g = diag(-al^2, a1, a2, a3)
    al = rng.uniform(0.5, 1.5, nz)
    a = rng.uniform(0.5, 2.0, (3, nz))
    geom[0] = -al * al
    geom[4], geom[7], geom[9] = a[0], a[1], a[2]
    geom[13] = al * np.sqrt(a[0] * a[1] * a[2])
    geom[14] = al
    dgeom = torch.from_numpy(geom).cuda()
    P_ref = torch.from_numpy(guess.copy()).cuda()
    it_ref, st_ref, rn_ref = _outputs(nz)
    g.invert_primitives(dU, P_ref, it_ref, st_ref, rn_ref, geom=dgeom)
    P_new = torch.from_numpy(guess.copy()).cuda()
    it_new, st_new, rn_new = _outputs(nz)
    gb.invert_primitives_static(dU, P_new, it_new, st_new, rn_new, geom=dgeom, model=nvar, **SOLVER)
    torch.cuda.synchronize()
    assert torch.equal(it_new, it_ref) and torch.equal(st_new, st_ref)
    assert np.array_equal(rn_new.cpu().numpy(), rn_ref.cpu().numpy(), equal_nan=True)
    assert np.array_equal(P_new.cpu().numpy(), P_ref.cpu().numpy(), equal_nan=True)
    g.close()


def test_static_inversion_refuses_a_batch_beyond_its_fixed_scratch():
    import torch
    import paper_1702_01106_b200 as gb
    nz = gb.STATIC_MAX_ZONES + 1
    U = torch.ones((8, nz), dtype=torch.float64, device="cuda")
    P = torch.ones((8, nz), dtype=torch.float64, device="cuda")
    it, st, rn = _outputs(nz)
    with pytest.raises(gb.GrimError, match="GRIM_STATIC_MAX_ZONES = %d" % gb.STATIC_MAX_ZONES):
        gb.invert_primitives_static(U, P, it, st, rn, model=8, **SOLVER)
    torch.cuda.synchronize()
    assert bool((P == 1.0).all()) and bool((it == -7).all())     # refused before any work was enqueued
    # an empty batch is a no-op
    e = torch.zeros((8, 0), dtype=torch.float64, device="cuda")
    ei = torch.zeros(0, dtype=torch.int32, device="cuda")
    gb.invert_primitives_static(e, e.clone(), ei, ei.clone(), torch.zeros(0, dtype=torch.float64, device="cuda"))
