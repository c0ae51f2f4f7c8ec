"""The multi-GPU path end to end on ONE device: two ranks (processes) of distributed.py::SlabGrid over the gloo backend
(ghost planes staged through the host; on a multi-GPU node the same code runs over NCCL, device to device), each
holding a slab of a periodic n x n x 2n grid.  dt from the all-reduced wave speeds and two time steps must be
bit-identical to the single-grid run -- every zone sees the same stencil values.  The two
processes only exchange host buffers between kernel launches; no kernel waits on another process."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from common import cuda_grid

pytestmark = pytest.mark.gpu

N, NG, STEPS = 12, 3, 2


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, dim, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    from paper_1702_01106_b200 import distributed as gdist
    from paper_1702_01106_b200 import workloads
    gk, P0 = workloads.config3(n=N, dim=dim, ranks=world, rank=rank)
    slab = gdist.SlabGrid(gk, world, rank, device=0)
    dP = torch.from_numpy(P0).cuda()
    dt = slab.choose_dt(dP)
    for _ in range(STEPS):
        slab.timestep(dP, dt)
    out[rank] = (dt, dP.cpu().numpy())
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("dim", [3, 2])
def test_two_ranks_equal_single_grid(dim):
    """dim = 3: slabs along X^3; dim = 2: slabs along X^2."""
    from paper_1702_01106_b200 import workloads
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), dim, out), nprocs=world, join=True)
    parts = [workloads.config3(n=N, dim=dim, ranks=world, rank=r) for r in range(world)]
    ax = 4 - dim                      # tensor dimension of the slab direction in P[nvar, s3, s2, s1]
    if dim == 3:
        gk = dict(parts[0][0], n3=world * N, xend=(1.0, 1.0, float(world)))
    else:
        gk = dict(parts[0][0], n2=world * N, xend=(1.0, float(world), 1.0))
    lo = np.take(parts[0][1], range(NG + N), axis=ax)
    hi = np.take(parts[1][1], range(NG, N + 2 * NG), axis=ax)
    P = np.concatenate([lo, hi], axis=ax)
    g = cuda_grid(gk)
    dP = torch.from_numpy(np.ascontiguousarray(P)).cuda()
    dt, _ = g.timestep(dP.clone(), 0.0, want_dt=True)
    for _ in range(STEPS):
        g.timestep(dP, dt)
    ref = dP.cpu().numpy()
    assert dt == out[0][0] == out[1][0]
    for r in range(world):
        got = np.take(out[r][1], range(NG, NG + N), axis=ax)
        exp = np.take(ref, range(NG + N * r, NG + N * (r + 1)), axis=ax)
        for a in range(4 - dim, 4):           # interior zones of the other active directions
            if a != ax:
                got, exp = np.take(got, range(NG, NG + N), axis=a), np.take(exp, range(NG, NG + N), axis=a)
        assert got.shape == exp.shape and np.array_equal(got, exp)


def _worker_torus(rank, world, port, n1, n2, out):
    """X^2 slabs of the 2-D Kerr torus grid: the end ranks keep the polar-reflection boundary, the inner sides are
    fed by the neighbours; each rank's geometry is that of its own X^2 range."""
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    from paper_1702_01106_b200 import distributed as gdist
    from paper_1702_01106_b200 import workloads
    gk, P0 = workloads.fm_torus(n1, n2, 1)
    m = n2 // world
    lo, hi = gk["xstart"][1] + rank * m / n2, gk["xstart"][1] + (rank + 1) * m / n2
    gl = dict(gk, n2=m, xstart=(gk["xstart"][0], lo, 0.0), xend=(gk["xend"][0], hi, gk["xend"][2]))
    Pl = np.ascontiguousarray(P0[:, :, rank * m:rank * m + m + 2 * NG])
    slab = gdist.SlabGrid(gl, world, rank, device=0)
    dP = torch.from_numpy(Pl).cuda()
    dt = slab.choose_dt(dP)
    for _ in range(STEPS):
        slab.timestep(dP, dt)
    out[rank] = (dt, dP.cpu().numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_torus_x2_slabs_match_single_grid_to_roundoff():
    """The library computes each rank's Kerr geometry from the rank's own coordinate range, so zone centres are
    x_start' + (j + 1/2) dx with another x_start' than in the single grid: the geometry tables agree to round-off, not to
    the bit, and so do the results (1e-10 on zones whose solves converge; a sharded MINKOWSKI run is bit-identical,
    above).  What this test pins is the slab logic with physical boundaries on the end ranks."""
    from paper_1702_01106_b200 import workloads
    world, n1, n2 = 2, 40, 48
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker_torus, args=(world, _free_port(), n1, n2, out), nprocs=world, join=True)
    gk, P0 = workloads.fm_torus(n1, n2, 1)
    g = cuda_grid(gk)
    dP = torch.from_numpy(P0).cuda()
    g.fill_ghosts(dP)
    dt, _ = g.timestep(dP.clone(), 0.0, want_dt=True)
    for _ in range(STEPS):
        _, st = g.timestep(dP, dt, want_stats=True)
    ref = dP.cpu().numpy()
    assert abs(out[0][0] - dt) < 1e-12 * dt and out[0][0] == out[1][0]
    m = n2 // world
    worst = 0.0
    for r in range(world):
        got = out[r][1][:, 0, NG:NG + m, NG:NG + n1]
        exp = ref[:, 0, NG + m * r:NG + m * (r + 1), NG:NG + n1]
        scale = np.maximum(abs(exp), 1e-6 * abs(exp).max(axis=(1, 2), keepdims=True))
        rel = abs(got - exp) / scale
        # zones at kmax / with an exhausted line search are sensitive to the last bit (test_gpu_torus.py): compare the bulk
        worst = max(worst, float(np.quantile(rel[:8], 0.9)))
        assert np.isfinite(got).all()
    assert worst < 1e-9, worst
