"""Slab decomposition of the grid along its slowest active direction -- X^3 of a 3-D grid, X^2 of a 2-D grid (SURVEY
8(e)) -- over torch.distributed ranks (one process per GPU).

The Newton solve, Jacobian, LU and line search are independent per zone; the only coupling between
ranks is the stencil of the flux / explicit-gradient step, ng zones deep, so each stage needs ONE exchange of the
ng ghost planes of P_E with the two neighbouring ranks (the paper's `communicate()`, L406-410, there staged through
the host; here device-to-device over NCCL/NVLink), plus one scalar max-reduction when dt is chosen from the CFL
number.  Every rank's zones see the same stencil values as in a single-domain run, so a sharded run is
bit-identical to the single-GPU run.

This module only sequences C-ABI calls and moves ghost planes; all arithmetic runs in the library's kernels.
The exchange itself is written on torch tensors of any device so that its index logic is tested on CPU with the
gloo backend (tests/test_distributed_cpu.py).
"""
import torch
import torch.distributed as dist


def exchange_slab(P, ng, world, rank, periodic=True, group=None, axis=1):
    """Fills the ghost planes along tensor dimension `axis` (1: X^3, 2: X^2) of the local padded array
    P[nvar, s3, s2, s1] from the neighbouring ranks' interior planes (full padded planes of the other directions, so
    edge and corner ghosts come along).  Rank r's lower neighbour is r-1, upper r+1, wrapping if periodic; a missing
    neighbour leaves those ghosts untouched."""
    n = P.shape[axis] - 2 * ng
    pl = lambda a, b: P.narrow(axis, a, b - a)       # planes [a, b) along the slab direction (a view)  # noqa: E731
    if world == 1:
        if periodic:
            pl(0, ng).copy_(pl(n, n + ng))
            pl(ng + n, n + 2 * ng).copy_(pl(ng, 2 * ng))
        return
    lo = rank - 1 if rank > 0 else (world - 1 if periodic else None)
    hi = rank + 1 if rank < world - 1 else (0 if periodic else None)
    send_lo = pl(ng, 2 * ng).contiguous()            # my lowest interior planes -> lower neighbour's upper ghosts
    send_hi = pl(n, n + ng).contiguous()             # my highest interior planes -> upper neighbour's lower ghosts
    if P.is_cuda and dist.get_backend(group) == "gloo":
        # gloo moves host memory only: stage the planes through the host (the NCCL path is device to device)
        send_lo, send_hi = send_lo.cpu(), send_hi.cpu()
    recv_lo, recv_hi = torch.empty_like(send_lo), torch.empty_like(send_hi)
    # Message kinds: "up" (tag 0) = my highest interior planes -> upper neighbour's lower ghosts; "down" (tag 1) =
    # my lowest interior planes -> lower neighbour's upper ghosts.  Sends are posted (up, down) and receives
    # (up-from-lower, down-from-upper), so that with two periodic ranks, where both neighbours are the same peer
    # and NCCL matches by issue order, the first message from the peer (its "up") lands in my lower ghosts.
    ops = []
    if hi is not None:
        ops.append(dist.P2POp(dist.isend, send_hi, hi, group=group, tag=0))
    if lo is not None:
        ops.append(dist.P2POp(dist.isend, send_lo, lo, group=group, tag=1))
    if lo is not None:
        ops.append(dist.P2POp(dist.irecv, recv_lo, lo, group=group, tag=0))
    if hi is not None:
        ops.append(dist.P2POp(dist.irecv, recv_hi, hi, group=group, tag=1))
    for w in dist.batch_isend_irecv(ops):
        w.wait()
    if hi is not None:
        pl(ng + n, n + 2 * ng).copy_(recv_hi)
    if lo is not None:
        pl(0, ng).copy_(recv_lo)


def exchange_x3(P, ng, world, rank, periodic=True, group=None):
    """exchange_slab along X^3."""
    exchange_slab(P, ng, world, rank, periodic, group, axis=1)


class SlabGrid:
    """One rank's slab of an n1 x n2 x (world n3) grid (3-D) or an n1 x (world n2) grid (2-D).  world == 1 is the plain
    single-GPU grid."""

    def __init__(self, gk, world=1, rank=0, device=0):
        from . import binding as gb
        self.world, self.rank = world, rank
        k = dict(gk)
        dim = k.get("dim", 3)
        self.sdir = dim - 1                      # slab direction: the slowest active one (X^3, or X^2 of a 2-D grid)
        self.axis = 3 - self.sdir                # its tensor dimension in P[nvar, s3, s2, s1]
        bc = k.get("bc", gb.BC_PERIODIC)
        if isinstance(bc, int):
            bc = [[bc, bc], [bc, bc], [bc, bc]]
        bc = [list(b) for b in bc]
        self.periodic3 = bc[self.sdir][0] == gb.BC_PERIODIC
        if world > 1:
            if dim < 2:
                raise gb.GrimError("slab decomposition needs a 2-D or 3-D grid")
            phys = bc[self.sdir]
            bc[self.sdir] = [gb.BC_NONE, gb.BC_NONE]                       # these ghosts come from the neighbours
            if not self.periodic3:
                if rank == 0:
                    bc[self.sdir][0] = phys[0]
                if rank == world - 1:
                    bc[self.sdir][1] = phys[1]
        self.ng = k.get("ng", 3)
        self.grid = gb.Grid(k["n1"], k.get("n2", 1), k.get("n3", 1), ng=self.ng, dim=k.get("dim", 3),
                            xstart=k.get("xstart", (0, 0, 0)), xend=k.get("xend", (1, 1, 1)), bc=bc,
                            model=k.get("nvar", 10), recon=k.get("recon", 0),
                            limiter_theta=k.get("limiter_theta", 1.0), gamma=k.get("gam", 4.0 / 3.0),
                            phi=k.get("phi", 1.0), psi=k.get("psi", 1.0), tau_mode=k.get("tau_mode", 0),
                            tau=k.get("tau", 1.0), fd_eps=k.get("fd_eps", 4e-8), eps_bt=k.get("eps_bt", 1e-4),
                            atol=k.get("atol", 0.0), rtol=k.get("rtol", 1e-14), kmax=k.get("kmax", 8),
                            lsmax=k.get("lsmax", 5), cfl=k.get("cfl", 0.5), metric=k.get("metric", 0),
                            metric_params=k.get("metric_params", ()), device=device,
                            flux_ct=k.get("flux_ct", False), reduced=k.get("reduced", False),
                            riemann=k.get("riemann", 0), closure=k.get("closure", 0))
        self.cfl = k.get("cfl", 0.5)
        g = self.grid
        if world > 1:
            t = torch
            self.Ph = g.zeros(g.nvar)
            self.rn = g.zeros()
            self.st, self.it = g.zeros(dtype=t.int32), g.zeros(dtype=t.int32)
            self.sp = t.zeros(4, dtype=t.float64, device=g.device)

    def _ghosts(self, P):
        self.grid.fill_ghosts(P)
        if self.world > 1:
            exchange_slab(P, self.ng, self.world, self.rank, self.periodic3, axis=self.axis)

    def choose_dt(self, P):
        """dt = cfl / max over all ranks' zones of sum_d c^d/dX^d (C-15)."""
        g = self.grid
        if self.world == 1:
            dtu, _ = g.timestep(P.clone(), 0.0, want_dt=True)
            return dtu
        self._ghosts(P)
        g.compute_fluxes(P, P, 1.0, speeds_out=self.sp)
        dist.all_reduce(self.sp, op=dist.ReduceOp.MAX)
        return self.cfl / float(self.sp[3])

    def timestep(self, P, dt):
        """One time step in place (same stage sequence as grim_timestep, with the ghost exchange in between)."""
        g = self.grid
        if self.world == 1:
            g.timestep(P, dt)
            return
        # no stage-buffer copies: each solve reads its guess from P_E and writes the interior of its output; the
        # X^3 ghost planes of P_{n+1/2} come from the neighbours, the others from the boundary conditions; the
        # second solve writes P_{n+1} over P_n zone by zone (grim_newton_solve)
        self._ghosts(P)
        g.compute_fluxes(P, P, 0.5 * dt)
        g.newton_solve(P, P, None, None, 0.5 * dt, P, self.Ph, self.rn, self.st, self.it)
        self._ghosts(self.Ph)
        g.compute_fluxes(self.Ph, P, dt)
        g.newton_solve(P, self.Ph, None, None, dt, self.Ph, P, self.rn, self.st, self.it)

    def timestep_host(self, hP, dt):
        """End to end with a HOST (pinned) buffer: H2D, one step, D2H."""
        g = self.grid
        if self.world == 1:
            g.timestep_host(hP, 1, dt)
            return
        if not hasattr(self, "_stage"):
            self._stage = g.zeros(g.nvar)
        self._stage.copy_(hP, non_blocking=True)
        self.timestep(self._stage, dt)
        hP.copy_(self._stage, non_blocking=True)
        torch.cuda.current_stream(g.device).synchronize()
