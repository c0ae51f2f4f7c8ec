"""grim_timestep_host with one step and a fixed dt runs pipelined over slabs of X^3 planes (host -> device copy, the two
stages' kernels and the device -> host copy of different slabs at the same time; api.cu).  Its results must be those of
grim_timestep on a device-resident array bit for bit -- on a periodic Minkowski grid (wrap between the first and the
last slab) and on a Kerr grid (outflow / polar reflection / periodic), with a ragged last slab."""
import numpy as np
import pytest

from common import cuda_grid, to_dev

pytestmark = pytest.mark.gpu


def _check(gk, P0, steps=2):
    import os
    import torch
    os.environ["GRIM_HOST_PIPELINE"] = "1"       # small grids here: the library pipelines from 1.5 M zones on its own
    try:
        gc = cuda_grid(gk)
    finally:
        del os.environ["GRIM_HOST_PIPELINE"]
    dP = to_dev(P0)
    gc.fill_ghosts(dP)
    dt, _ = gc.timestep(dP.clone(), 0.0, want_dt=True)
    hP = torch.from_numpy(P0.copy()).pin_memory()
    assert gc.last_host_mode() == "none"
    l0 = gc.launch_count()
    for _ in range(steps):
        gc.timestep(dP, dt)
    per_step = (gc.launch_count() - l0) // steps
    l0 = gc.launch_count()
    for _ in range(steps):
        gc.timestep_host(hP, 1, dt)
    assert (gc.launch_count() - l0) // steps > 4 * per_step          # the slab-wise launches did run
    assert gc.last_host_mode() == "pipelined"
    assert torch.equal(gc.interior(hP), gc.interior(dP).cpu())
    # pageable host memory takes the same path
    hQ = torch.from_numpy(P0.copy())
    for _ in range(steps):
        gc.timestep_host(hQ, 1, dt)
    assert torch.equal(gc.interior(hQ), gc.interior(dP).cpu())
    # several steps per call: copy in, step, copy out (not pipelined), same result
    hR = torch.from_numpy(P0.copy())
    gc.timestep_host(hR, steps, dt)
    assert gc.last_host_mode() == "whole"
    assert torch.equal(gc.interior(hR), gc.interior(dP).cpu())


def test_pipelined_host_step_periodic_minkowski():
    from paper_1702_01106_b200 import workloads
    gk, P0 = workloads.config3(n=64)
    _check(gk, P0)
    gk, P0 = workloads.config3(n=64)
    gk = dict(gk, n3=76, xend=(1.0, 1.0, 76.0 / 64.0))         # ragged slabs; the state is not periodic over 76: irrelevant
    X = workloads.padded_centres((64, 64, 76), (3, 3, 3), gk["xstart"], gk["xend"])
    t = workloads.mode_tables()["config3"]
    _check(gk, workloads.linear_mode_state(t["P0"], t["modes"], 1e-4, *X))


def test_pipelined_host_step_kerr_torus():
    from paper_1702_01106_b200 import workloads
    gk, P0 = workloads.fm_torus(48, 40, 64)
    _check(gk, P0)


def test_timestep_is_capturable_in_a_cuda_graph():
    """grim_timestep with a fixed dt and no statistics enqueues kernels only (no synchronisation, no allocation once the
    context is warm), so a caller can capture it into a CUDA graph on the context's stream and replay it -- worth 5-15 %
    on grids of 32^3-64^3, where the 22 launches of a step are a visible share of its 0.2-0.7 ms.  Replays give the
    bits of direct calls."""
    import torch
    import paper_1702_01106_b200 as gb
    from paper_1702_01106_b200 import workloads
    gk, P0 = workloads.config3(n=32)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        gc = gb.Grid(gk["n1"], gk["n2"], gk["n3"], dim=3, model=10, recon=1, rtol=gk["rtol"], kmax=gk["kmax"],
                     lsmax=gk["lsmax"], stream=s.cuda_stream)
        dP, dQ = to_dev(P0), to_dev(P0)
        dt, _ = gc.timestep(dP.clone(), 0.0, want_dt=True)
        warm = dP.clone()
        for _ in range(3):
            gc.timestep(warm, dt)               # scratch lists exist, tensor-map entry point resolved
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            gc.timestep(dQ, dt)                 # captured, not executed
        s.synchronize()
        assert torch.equal(dQ, to_dev(P0))
        for _ in range(4):
            g.replay()
            gc.timestep(dP, dt)
        s.synchronize()
    assert torch.equal(gc.interior(dQ), gc.interior(dP))
