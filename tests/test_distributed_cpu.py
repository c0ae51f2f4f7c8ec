"""Multi-rank host logic on CPU (gloo, world_size 2 and 3): the X^3 ghost-plane exchange of
paper_1702_01106_b200/distributed.py reproduces the single-domain ghost fill of the stacked grid, so that every
rank's zones see the same stencil values as in a single-GPU run."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle as og


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, periodic, n, ng, nvar, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1702_01106_b200.distributed import exchange_x3
    rng = np.random.default_rng(123)
    # the stacked global grid, ghosts filled the single-domain way by the oracle's fill (periodic or outflow in X^3)
    bc3 = og.BC_PERIODIC if periodic else og.BC_OUTFLOW
    gg = og.Grid(n[0], n[1], n[2] * world, ng=ng, dim=3, nvar=nvar,
                 bc=[[og.BC_PERIODIC] * 2, [og.BC_PERIODIC] * 2, [bc3] * 2])
    Pg = rng.standard_normal(gg.shape)
    gg.fill_ghosts(Pg)
    # this rank's slab: interior planes from the global array, X^1/X^2 ghosts already consistent, X^3 ghosts poisoned
    k0 = ng + rank * n[2]
    loc = np.full((nvar, n[2] + 2 * ng, Pg.shape[2], Pg.shape[3]), np.nan)
    loc[:, ng:ng + n[2]] = Pg[:, k0:k0 + n[2]]
    if not periodic:      # physical boundaries keep their own (outflow) ghosts on the end ranks
        if rank == 0:
            loc[:, :ng] = Pg[:, :ng]
        if rank == world - 1:
            loc[:, ng + n[2]:] = Pg[:, ng + n[2] * world:]
    t = torch.from_numpy(loc)
    exchange_x3(t, ng, world, rank, periodic)
    expect = Pg[:, k0 - ng:k0 + n[2] + ng]
    out[rank] = bool(np.array_equal(t.numpy(), expect))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,periodic", [(2, True), (3, True), (2, False), (3, False)])
def test_slab_exchange_matches_single_domain_fill(world, periodic):
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), periodic, (6, 5, 4), 3, 10, out), nprocs=world, join=True)
    assert all(out[r] for r in range(world)), dict(out)


def test_exchange_single_rank_is_periodic_copy():
    from paper_1702_01106_b200.distributed import exchange_x3
    g = og.Grid(5, 4, 6, ng=2, dim=3, nvar=8)
    P = np.random.default_rng(0).standard_normal(g.shape)
    Q = P.copy()
    g.fill_ghosts(Q)
    # only the X^3 ghosts of interior X^1/X^2 columns are comparable (the oracle also filled X^1, X^2 ghosts)
    t = torch.from_numpy(P.copy())
    exchange_x3(t, 2, 1, 0, True)
    assert np.array_equal(t.numpy()[:, :2, 2:6, 2:7], Q[:, :2, 2:6, 2:7])
    assert np.array_equal(t.numpy()[:, -2:, 2:6, 2:7], Q[:, -2:, 2:6, 2:7])


def _worker2d(rank, world, port, bc2, n, ng, nvar, out):
    """X^2 slabs of a 2-D grid: the stacked n1 x (world n2) grid with periodic X^1 and periodic /
    outflow / polar-reflection X^2, ghosts filled the single-domain way by the oracle; each rank fills its own X^1
    ghosts (as grim_fill_ghosts does, X^2 being BC_NONE towards a neighbour) and then exchanges."""
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1702_01106_b200.distributed import exchange_slab
    rng = np.random.default_rng(321)
    gg = og.Grid(n[0], n[1] * world, 1, ng=ng, dim=2, nvar=nvar, bc=[[og.BC_PERIODIC] * 2, [bc2] * 2, [0, 0]])
    Pg = rng.standard_normal(gg.shape)
    gg.fill_ghosts(Pg)
    j0 = ng + rank * n[1]
    loc = np.full((nvar, 1, n[1] + 2 * ng, Pg.shape[3]), np.nan)
    loc[:, :, ng:ng + n[1], ng:-ng] = Pg[:, :, j0:j0 + n[1], ng:-ng]          # interior only
    periodic = bc2 == og.BC_PERIODIC
    if not periodic:      # the physical boundary rows of the end ranks (the library fills them after X^1)
        if rank == 0:
            loc[:, :, :ng] = Pg[:, :, :ng]
        if rank == world - 1:
            loc[:, :, ng + n[1]:] = Pg[:, :, ng + n[1] * world:]
    # X^1 ghosts of the interior rows: periodic copy (what fill_ghosts_kernel<0> does)
    loc[:, :, ng:ng + n[1], :ng] = loc[:, :, ng:ng + n[1], n[0]:n[0] + ng]
    loc[:, :, ng:ng + n[1], ng + n[0]:] = loc[:, :, ng:ng + n[1], ng:2 * ng]
    t = torch.from_numpy(loc)
    exchange_slab(t, ng, world, rank, periodic, axis=2)
    expect = Pg[:, :, j0 - ng:j0 + n[1] + ng]
    out[rank] = bool(np.array_equal(t.numpy(), expect))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,bc2", [(2, og.BC_PERIODIC), (3, og.BC_PERIODIC), (2, og.BC_OUTFLOW), (3, og.BC_REFLECT_POLAR)])
def test_x2_slab_exchange_of_2d_grid_matches_single_domain_fill(world, bc2):
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker2d, args=(world, _free_port(), bc2, (6, 5), 3, 10, out), nprocs=world, join=True)
    assert all(out[r] for r in range(world)), dict(out)
