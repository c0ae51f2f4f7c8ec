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


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    from paper_1702_01106_b200 import distributed as gdist
    from paper_1702_01106_b200 import workloads
    gk, P0 = workloads.config3(n=N, ranks=world, rank=rank)
    slab = gdist.SlabGrid(gk, world, rank, device=0)
    dP = torch.from_numpy(P0).cuda()
    dt = slab.choose_dt(dP)
    for _ in range(STEPS):
        slab.timestep(dP, dt)
    out[rank] = (dt, dP.cpu().numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_equal_single_grid():
    from paper_1702_01106_b200 import workloads
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    parts = [workloads.config3(n=N, ranks=world, rank=r) for r in range(world)]
    gk = dict(parts[0][0], n3=world * N, xend=(1.0, 1.0, float(world)))
    P = np.concatenate([parts[0][1][:, :NG + N], parts[1][1][:, NG:]], axis=1)
    g = cuda_grid(gk)
    dP = torch.from_numpy(np.ascontiguousarray(P)).cuda()
    dt, _ = g.timestep(dP.clone(), 0.0, want_dt=True)
    for _ in range(STEPS):
        g.timestep(dP, dt)
    ref = dP.cpu().numpy()
    assert dt == out[0][0] == out[1][0]
    for r in range(world):
        got = out[r][1][:, NG:NG + N, NG:-NG, NG:-NG]
        exp = ref[:, NG + N * r:NG + N * (r + 1), NG:-NG, NG:-NG]
        assert np.array_equal(got, exp)
