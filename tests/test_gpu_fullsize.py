"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times, on sampled outputs the oracle
can compute one by one.

* config 3 headline (EMHD, MP5, 3-D Minkowski, 256^3; also 128^3): one grim_timestep on the GPU; for each sampled
  zone the oracle advances the 13^3 sub-box centred on it (ghosts = the true neighbouring data, periodic wrap).
  A zone's domain of dependence over the two stages is +-6 zones (stage 2 reads P_{n+1/2} at +-3, each of which
  read P_n at +-3 more, MP5 + the 3-point EMHD slopes), so the centre of the sub-box is exact.
* config 2 (2^24 zones): zones are independent, the oracle inverts a seeded sample of them.
"""
import numpy as np
import pytest

import oracle as og
from common import cuda_grid, to_dev

pytestmark = pytest.mark.gpu

R = 6           # domain-of-dependence radius of one time step
NG = 3


def subbox(P, c, ngd):
    """[nvar, 2(R+NG)+1]^3 block of the padded array P centred on interior zone c=(k,j,i) (interior indices),
    periodic wrap."""
    n = [P.shape[1] - 2 * ngd, P.shape[2] - 2 * ngd, P.shape[3] - 2 * ngd]
    w = R + NG
    idx = [(np.arange(c[a] - w, c[a] + w + 1) % n[a]) + ngd for a in range(3)]
    return np.ascontiguousarray(P[:, idx[0]][:, :, idx[1]][:, :, :, idx[2]])


@pytest.mark.parametrize("n", [128, 256])
def test_config3_fullsize_sampled(n):
    from paper_1702_01106_b200 import workloads
    gk, P0 = workloads.config3(n=n)
    gc = cuda_grid(gk)
    import torch
    dP = to_dev(P0)
    dtu, st = gc.timestep(dP, 0.0, want_dt=True, want_stats=True)      # dt from the CFL number; statistics branch
    # the branch bench.py times: fixed dt, no statistics, P_{n+1} written in place of P_n by the stage-2 Newton kernel
    dQ = to_dev(P0)
    gc.timestep(dQ, dtu)
    assert torch.equal(gc.interior(dQ), gc.interior(dP))
    P1 = gc.interior(dQ).cpu().numpy()
    del dP, dQ
    assert st.unconverged[0] == 0 and st.unconverged[1] == 0
    # every zone takes 1, 2 or 3 iterations per stage (C-13: two, except on either side of the threshold); the
    # histogram of the sampled sub-boxes is compared with the oracle's below, bin by bin
    for s in range(2):
        h = st.iters_hist[s]
        assert h[1] + h[2] + h[3] == n ** 3 and h[2] > 0.999 * n ** 3
    rng = np.random.default_rng(n)
    cs = [tuple(rng.integers(0, n, 3)) for _ in range(40)]
    cs += [(0, 0, 0), (n - 1, n - 1, n - 1), (0, n - 1, 5), (n // 2, 0, n - 1)]          # wrap-around corners
    m = 2 * R + 1
    sub = dict(gk, n1=m, n2=m, n3=m, bc=og.BC_NONE, xstart=(0.0, 0.0, 0.0), xend=(m / n, m / n, m / n))
    go = og.Grid(sub["n1"], sub["n2"], sub["n3"], ng=NG, dim=3, xstart=sub["xstart"], xend=sub["xend"],
                 bc=og.BC_NONE, nvar=10, recon=gk["recon"], limiter_theta=gk["limiter_theta"], gam=gk["gam"],
                 phi=gk["phi"], psi=gk["psi"], tau=gk["tau"], rtol=gk["rtol"], kmax=gk["kmax"], lsmax=gk["lsmax"])
    assert go.dx[0] == 1.0 / n
    # per-zone iteration counts, statuses and residual norms of the first stage at full size (north star: "identical
    # Newton iteration counts per zone"): grim_compute_fluxes + grim_newton_step on the whole grid, against the oracle's
    # stage on each sampled sub-box -- every interior zone of a sub-box has its true stencil in stage 1
    dP0 = to_dev(P0)
    gc.fill_ghosts(dP0)
    gc.compute_fluxes(dP0, dP0, 0.5 * dtu)
    dPh = dP0.clone()
    drn, dst, dit = gc.zeros(), gc.zeros(dtype=torch.int32), gc.zeros(dtype=torch.int32)
    assert gc.newton_step(dP0, dP0, None, None, 0.5 * dtu, 0, dPh, drn, dst, dit) == 0
    it_full = gc.interior(dit).cpu().numpy()
    st_full = gc.interior(dst).cpu().numpy()
    rn_full = gc.interior(drn).cpu().numpy()
    del dP0, dPh, drn, dst, dit
    hist_gpu, hist_ora = np.zeros(16, dtype=np.int64), np.zeros(16, dtype=np.int64)
    worst = 0.0
    for c in cs:
        Ps = subbox(P0, c, NG)
        Cs, Gs, _ = go.stage_prepare(Ps, Ps, 0.5 * dtu)
        Pq = Ps.copy()
        _, (rno, sto, ito), _ = go.newton(Ps, Ps, Cs, Gs, 0.5 * dtu, Pq)
        ii = [np.arange(c[a] - R, c[a] + R + 1) % n for a in range(3)]
        sel = np.ix_(ii[0], ii[1], ii[2])
        assert np.array_equal(it_full[sel], go.interior(ito)), c
        assert np.array_equal(st_full[sel], go.interior(sto)), c
        assert np.array_equal(rn_full[sel], go.interior(rno)), c
        hist_gpu += np.bincount(it_full[sel].ravel(), minlength=16)[:16]
        hist_ora += np.bincount(go.interior(ito).ravel(), minlength=16)[:16]
        so = go.timestep(Ps, dtu)
        got = P1[:, c[0], c[1], c[2]]
        exp = Ps[:, NG + R, NG + R, NG + R]
        assert np.array_equal(got, exp), (c, got, exp)
        # and the +-3 neighbourhood, which is exact too
        blk = Ps[:, NG + R - 3:NG + R + 4, NG + R - 3:NG + R + 4, NG + R - 3:NG + R + 4]
        ii = [np.arange(c[a] - 3, c[a] + 4) % n for a in range(3)]
        gpu = P1[:, ii[0]][:, :, ii[1]][:, :, :, ii[2]]
        worst = max(worst, abs(gpu - blk).max())
    assert worst == 0.0
    assert np.array_equal(hist_gpu, hist_ora) and hist_ora.sum() == len(cs) * (2 * R + 1) ** 3


def test_config2_fullsize_sampled():
    import torch
    from paper_1702_01106_b200 import workloads
    nz, nvar = 1 << 24, 8
    Ptrue, guess = workloads.config2(nz, seed=1702, nvar=nvar)
    gc = cuda_grid(dict(n1=8, n2=8, n3=1, dim=2, nvar=nvar, rtol=1e-12, kmax=30, lsmax=8))
    dU = torch.empty((nvar, nz), dtype=torch.float64, device="cuda")
    gc.prim_to_conserved(to_dev(Ptrue), dU)
    dP = to_dev(guess)
    dit = torch.zeros(nz, dtype=torch.int32, device="cuda")
    dst = torch.zeros_like(dit)
    drn = torch.zeros(nz, dtype=torch.float64, device="cuda")
    gc.invert_primitives(dU, dP, dit, dst, drn)
    sel = np.sort(np.random.default_rng(24).choice(nz, 30000, replace=False))
    sel[:3] = [0, 1, 2]; sel[-1] = nz - 1
    sel = np.unique(sel)
    U = dU.cpu().numpy()[:, sel]
    m = og.model(nvar=nvar)
    Po, ito, sto, rno, _ = og.invert(m, og.solver(rtol=1e-12, kmax=30, lsmax=8), U, guess[:, sel])
    tsel = torch.from_numpy(sel).cuda()
    assert np.array_equal(dit[tsel].cpu().numpy(), ito)
    assert np.array_equal(dst[tsel].cpu().numpy(), sto)
    assert np.array_equal(dP[:, tsel].cpu().numpy(), Po, equal_nan=True)
    assert np.array_equal(drn[tsel].cpu().numpy(), rno, equal_nan=True)
    # every zone reached a terminal status; the unconverged tail is the algorithm's own (~3 %)
    st = dst.cpu().numpy()
    assert ((st & (og.ST_CONVERGED | og.ST_KMAX | og.ST_SINGULAR | og.ST_NONFINITE)) != 0).all()
    frac_conv = ((st & og.ST_CONVERGED) != 0).mean()
    assert 0.9 < frac_conv < 1.0
