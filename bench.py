#!/usr/bin/env python
"""bench.py -- throughput of the grim hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--n 256] [--impl ours|reference]

Workload: BASELINE.json config 3's generator at n^3 (headline n = 256): EMHD (10 primitives), 3-D Minkowski,
periodic, four seeded linear modes of amplitude 1e-4 on the background rho=1, u=2, B=(0.1,0.3,0); MP5 + LLF,
CFL 0.5.  A "step" is one grim_timestep: 2 stages x (ghost fill, reconstruction + LLF fluxes + stage constants,
fused per-zone Newton solve).  value = zones advanced one time step per second, whole job.

N > 1 (torchrun): the grid is cut into N slabs along X^3 (weak scaling: every rank holds n^3 zones of an
n x n x (N n) grid); each stage's ghost planes in X^3 are exchanged between neighbouring ranks with
torch.distributed (NCCL) device-to-device, everything else is rank-local.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "fp64 zone-updates/sec per Newton step (EMHD 10-var) and % of HBM roofline"
UNIT = "zone-updates/s"

# per zone and stage of the Newton kernel, Minkowski EMHD, 2 Newton iterations.
# Algorithmic fp64 work: DADD + DMUL + DFMA thread instructions that the method's definition requires under the strict
# arithmetic contract (every + - * separately rounded, / and sqrt as correctly rounded Newton-Raphson sequences), counted
# with ncu on the round's first kernel (profiles/r1a_ncu_full_stage_kernels_baseline.md) and then FROZEN, so that later
# kernels cannot raise the fraction by executing more instructions.  (What the current kernel executes: EXECUTED_FP64_INSTR_PER_ZONE_STAGE_NEWTON below.)
ALG_FP64_INSTR_PER_ZONE_STAGE_NEWTON = 6114.0
ALG_BYTES_PER_ZONE_STAGE_NEWTON = 8.0 * (10 + 10 + 10 + 10 + 3 + 10 + 1) + 4 * 4   # P^k,P_n,P_E,C,G in; P,|R| out; status,iters in/out
# dram__bytes_read.sum + dram__bytes_write.sum of the Newton kernel per zone, mean of the stage-1 and stage-2 launches
# (profiles/r2c_final_kernels.md: 288 B and 367 B per zone, ncu --set full captures of this round's final kernel)
NCU_DRAM_BYTES_PER_ZONE_STAGE_NEWTON = 327.0
# What the current kernel executes (DADD + DMUL + DFMA per zone and stage at 2 iterations, profiles/r2c_final_kernels.md):
# fewer than the frozen algorithmic count, because structural zeros of the Jacobian and of the LU are skipped.
# roofline.frac credits the frozen count (work the method defines); roofline.frac_executed is the fp64-pipe utilisation.
EXECUTED_FP64_INSTR_PER_ZONE_STAGE_NEWTON = 5274.0
NEWTON_KERNEL = "newton_stage_kernel<10,flat>"
NCU_TRAFFIC_SOURCE = "profiles/r2c_final_kernels.md"
# Flux class (3 face-flux launches + boundary-face boxes + stage constant) per zone and stage.  Algorithmic bytes: SURVEY
# 8(d) "Flux + stage constant, EMHD": P_E 10 (x 1.3-1.5 halo re-read) + P_n 10 in, C 10 + G 3 out -> 320-400 B; the
# upper figure.  Algorithmic fp64 work: DADD + DMUL + DFMA thread instructions of the same four kernels in the round's
# capture of the round-1 kernels (3997 per zone-stage: 3 x 1084 face + 744 stage constant; profiles/r2c_final_kernels.md
# and DESIGN.md 15.3), frozen like the Newton count.
ALG_BYTES_PER_ZONE_STAGE_FLUX = 400.0
ALG_FP64_INSTR_PER_ZONE_STAGE_FLUX = 3997.0
NCU_DRAM_BYTES_PER_ZONE_STAGE_FLUX = 1075.0
FP64_INSTR_PER_CLK_PER_SM = 64.0                 # B200: 64 fp64 lanes per SM (guide: unit counts), 148 SMs
N_SM = 148


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d.get("hbm_gbs", 6650.0), d.get("sm_max_mhz", 1965.0), "measured"
    return 6650.0, 1965.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks line of the profiling recipe, sampled every 50 ms during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, device):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(device), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "50"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            t = [x.strip() for x in line.split(",")]
            if len(t) < 9:
                continue
            try:
                sm.append(float(t[1])); mx.append(float(t[2]))
            except ValueError:
                continue
            for nm, v in zip(names, t[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


def oracle_sample(n, steps, warmup):
    """The oracle, as it stands, on the config-3 generator at n^3; returns (zone-updates/s, s per step, cores)."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import oracle as og
    from paper_1702_01106_b200 import workloads
    gk, P = workloads.config3(n=n)
    go = og.Grid(gk["n1"], gk["n2"], gk["n3"], ng=gk.get("ng", 3), dim=gk["dim"], xstart=gk.get("xstart", (0, 0, 0)),
                 xend=gk.get("xend", (1, 1, 1)), bc=gk.get("bc", og.BC_PERIODIC), nvar=gk["nvar"], recon=gk["recon"],
                 gam=gk.get("gam", 4.0 / 3.0), phi=gk.get("phi", 1.0), psi=gk.get("psi", 1.0), tau=gk.get("tau", 1.0),
                 fd_eps=gk.get("fd_eps", 4e-8), eps_bt=gk.get("eps_bt", 1e-4), atol=gk.get("atol", 0.0),
                 rtol=gk.get("rtol", 1e-14), kmax=gk.get("kmax", 8), lsmax=gk.get("lsmax", 5), cfl=gk.get("cfl", 0.5))
    dt = go.choose_dt(P)
    for _ in range(warmup):
        go.timestep(P, dt)
    t0 = time.perf_counter()
    for _ in range(steps):
        go.timestep(P, dt)
    el = time.perf_counter() - t0
    return n ** 3 * steps / el, el / steps, og.num_threads()


def other_workloads(local):
    """Secondary measurements, N = 1 only, after the headline timing (reported beside it, not bench lines):
    BASELINE config 2 (2^24 standalone inversions, ideal MHD) and one EMHD time step on config 5's grid
    (Kerr a = 0.9375, 256 x 256 x 128, synthetic state -- workloads.kerr_synthetic)."""
    import torch
    import paper_1702_01106_b200 as gb
    from paper_1702_01106_b200 import workloads
    out = {}

    def ev():
        return torch.cuda.Event(enable_timing=True)

    nz, nvar = 1 << 24, 8
    Ptrue, guess = workloads.config2(nz, seed=1702, nvar=nvar)
    g = gb.Grid(8, 8, 1, dim=2, model=nvar, rtol=1e-12, kmax=30, lsmax=8, device=local)
    dU = torch.empty((nvar, nz), dtype=torch.float64, device="cuda")
    g.prim_to_conserved(torch.from_numpy(Ptrue).cuda(), dU)
    dG = torch.from_numpy(guess).cuda()
    it = torch.zeros(nz, dtype=torch.int32, device="cuda")
    st = torch.zeros_like(it)
    rn = torch.zeros(nz, dtype=torch.float64, device="cuda")
    best = None
    for _ in range(4):
        dP = dG.clone()
        torch.cuda.synchronize()
        e0, e1 = ev(), ev()
        e0.record()
        g.invert_primitives(dU, dP, it, st, rn)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        best = ms if best is None else min(best, ms)
    out["config2_inversion_2^24"] = {"ms": best, "solves_per_s": nz / best * 1e3,
                                     "zone_iterations_per_s": float(it.double().sum()) / best * 1e3,
                                     "mean_iterations": float(it.double().mean()),
                                     "converged_fraction": float(((st & 1) != 0).double().mean())}
    del g, dU, dG, dP, it, st, rn
    torch.cuda.empty_cache()

    gk, P = workloads.kerr_synthetic(256, 256, 128)
    g = gb.Grid(gk["n1"], gk["n2"], gk["n3"], dim=3, xstart=gk["xstart"], xend=gk["xend"], bc=gk["bc"], model=10,
                recon=1, tau_mode=gk["tau_mode"], rtol=gk["rtol"], kmax=gk["kmax"], lsmax=gk["lsmax"],
                metric=gk["metric"], metric_params=gk["metric_params"], device=local)
    dP = torch.from_numpy(P).cuda()
    dt, _ = g.timestep(dP.clone(), 0.0, want_dt=True)
    for _ in range(3):
        g.timestep(dP, dt)
    torch.cuda.synchronize()
    e0, e1 = ev(), ev()
    K = 5
    e0.record()
    for _ in range(K):
        g.timestep(dP, dt)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / K
    _, sst = g.timestep(dP, dt, want_stats=True)
    out["kerr_emhd_256x256x128_synthetic"] = {"ms_per_step": ms, "zone_updates_per_s": g.zones / ms * 1e3,
                                              "unconverged": [int(x) for x in sst.unconverged]}
    del g, dP
    torch.cuda.empty_cache()

    # BASELINE config 5 as stated: Fishbone-Moncrief torus, field loop at beta = 100, seeded noise (workloads.fm_torus)
    gk, P = workloads.fm_torus(256, 256, 128)
    g = gb.Grid(gk["n1"], gk["n2"], gk["n3"], dim=3, xstart=gk["xstart"], xend=gk["xend"], bc=gk["bc"], model=10,
                recon=gk["recon"], tau_mode=gk["tau_mode"], rtol=gk["rtol"], kmax=gk["kmax"], lsmax=gk["lsmax"],
                metric=gk["metric"], metric_params=gk["metric_params"], device=local)
    dP = torch.from_numpy(P).cuda()
    dt, _ = g.timestep(dP.clone(), 0.0, want_dt=True)
    for _ in range(3):
        g.timestep(dP, dt)
    torch.cuda.synchronize()
    e0, e1 = ev(), ev()
    e0.record()
    for _ in range(K):
        g.timestep(dP, dt)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / K
    _, sst = g.timestep(dP, dt, want_stats=True)
    its = [sum(i * sst.iters_hist[s][i] for i in range(16)) / g.zones for s in range(2)]
    out["config5_fm_torus_256x256x128_minmod"] = {"ms_per_step": ms, "zone_updates_per_s": g.zones / ms * 1e3,
                                                  "mean_newton_iterations": its,
                                                  "backtracks": [int(x) for x in sst.backtracks],
                                                  "unconverged": [int(x) for x in sst.unconverged]}
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n = args.ref_n
    v, sps, cores = oracle_sample(n, args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "config3-emhd-mp5-llf-minkowski-%d^3" % args.n,
                   "sample": "each step = one oracle time step of the same generator at %d^3" % n},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": "config-3 generator at %d^3, %d steps" % (n, args.steps)},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    import paper_1702_01106_b200 as gb
    from paper_1702_01106_b200 import distributed as gdist
    from paper_1702_01106_b200 import workloads

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    if args.backend == "gloo":
        local = local % torch.cuda.device_count()      # ranks may share a device (host-staged exchange; 1-GPU boxes)
    torch.cuda.set_device(local)
    if world > 1:
        if args.backend == "nccl":
            # the communicator log (rank count, transports, NVLS) goes to stderr, where the driver reads it; stdout
            # carries the one JSON line
            os.environ.setdefault("NCCL_DEBUG", "INFO")
            os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("gloo")
    n = args.n
    gk, P0 = workloads.config3(n=n, dim=args.dim, ranks=world, rank=rank)
    gk["flux_ct"] = bool(args.flux_ct)
    gk["reduced"] = bool(args.reduced)
    slab = gdist.SlabGrid(gk, world, rank, device=local)
    g = slab.grid
    dP = torch.from_numpy(P0).cuda()
    dt = slab.choose_dt(dP)                      # CFL 0.5 on the initial data, min over ranks; then held fixed
    zones = g.zones
    pbytes = dP.numel() * 8

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        slab.timestep(dP, dt)
    barrier()
    l0 = g.launch_count()
    g.set_timing(True)
    sampler = ClockSampler(local) if rank == 0 else None
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    ev[0].record()
    for k in range(args.steps):
        slab.timestep(dP, dt)
        ev[k + 1].record()                       # one event between steps: value stays the mean over the whole region
    barrier()
    ms = ev[0].elapsed_time(ev[args.steps])
    per_step = sorted(ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps))
    clocks = sampler.stop() if sampler else None
    timing = g.get_timing()
    g.set_timing(False)
    launches = g.launch_count() - l0
    _, st = g.timestep(dP.clone(), dt, want_stats=True) if world == 1 else (None, None)

    # end to end through the C ABI with HOST buffers (pinned): H2D of P, one step, D2H of P, every step
    hP = torch.from_numpy(P0.copy()).pin_memory()
    e2e_steps = max(1, min(args.steps, 5))
    e2e_s = float("nan")
    if not args.no_e2e:
        slab.timestep_host(hP, dt)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            slab.timestep_host(hP, dt)
        barrier()
        e2e_s = (time.perf_counter() - t0) / e2e_steps
    # the pipelined host path moves the interior X^3 planes only (the ghost planes are filled on the device); which form
    # the call took is the library's decision (grid, arguments, GRIM_HOST_PIPELINE), so ask it
    pipelined = world == 1 and g.last_host_mode() == "pipelined"
    e2e_bytes = pbytes * g.n[2] // g.sz[2] if pipelined else pbytes

    med = per_step[len(per_step) // 2] if per_step else float("nan")
    tmax = torch.tensor([ms, e2e_s, med, per_step[0] if per_step else float("nan")], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    ms, e2e_s, ms_median, ms_min = (float(x) for x in tmax)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    hbm_gbs, sm_max, which = peaks()
    stages = 2 * args.steps
    nk_ms, nk_n = timing["newton"]
    newton_ms = nk_ms / max(nk_n, 1)
    flux_ms = timing["flux"][0] / stages                                       # all flux-class launches of one stage
    alu_peak = N_SM * FP64_INSTR_PER_CLK_PER_SM * sm_max * 1e6 / 1e12          # T fp64 thread-instr/s
    # measured on this device, now: 8 independent DFMA chains per thread, 8 x 256 threads per SM (grim_fp64_probe)
    probe = max(g.fp64_probe(True, 1 << 15) for _ in range(3)) / 1e12
    headline = (not args.reduced) and (not args.flux_ct) and args.dim == 3
    mean_it = None if st is None else [sum(i * st.iters_hist[s][i] for i in range(16)) / max(zones, 1) for s in range(2)]
    # the frozen count is for 2 Newton iterations per zone and stage; other iteration counts scale it (set-up included:
    # a slight overstatement of the work for > 2 iterations, an understatement for < 2)
    it_scale = 1.0 if mean_it is None else 0.5 * (mean_it[0] + mean_it[1]) / 2.0
    alu_ach = ALG_FP64_INSTR_PER_ZONE_STAGE_NEWTON * it_scale * zones / (newton_ms * 1e-3) / 1e12
    hbm_ach = ALG_BYTES_PER_ZONE_STAGE_NEWTON * zones / (newton_ms * 1e-3) / 1e9
    flux_alu = ALG_FP64_INSTR_PER_ZONE_STAGE_FLUX * zones / (flux_ms * 1e-3) / 1e12
    flux_hbm = ALG_BYTES_PER_ZONE_STAGE_FLUX * zones / (flux_ms * 1e-3) / 1e9
    line = {
        "metric": METRIC, "value": zones * world * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
        "ms_per_step_median": ms_median, "ms_per_step_min": ms_min, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "config3-emhd-mp5-llf-minkowski-%d^%d%s" % (n, args.dim, ("-fluxct" if args.flux_ct else "") + ("-reduced7" if args.reduced else "")),
                   "zones_per_gpu": zones,
                   "update": "one zone advanced one grim_timestep = 2 stages x (ghosts, MP5+LLF fluxes, stage "
                             "constants, fused Newton solve)", "dt": "fixed: CFL 0.5 on the initial data",
                   "l2": "inputs (%.2f GB per field) larger than L2" % (pbytes / 1e9),
                   "parallelism": "slab%d" % world, "backend": args.backend if world > 1 else None,
                   "nccl_log": "stderr (NCCL_DEBUG=INFO, INIT)" if (world > 1 and args.backend == "nccl") else None},
        "clocks": clocks,
        "e2e": {"value": zones * world / e2e_s, "unit": UNIT, "h2d_bytes_per_step": e2e_bytes,
                "d2h_bytes_per_step": e2e_bytes,
                "how": "grim_timestep_host, pinned host buffer, one step per call: %s" % (
                    "interior X^3 planes copied slab by slab on two copy streams while the kernels of other slabs run"
                    if pipelined else "copy in, step, copy out")},
        "gpu_launches": int(launches),
        "roofline": None if not headline else {
            "bound": "alu", "kernel": NEWTON_KERNEL, "achieved": alu_ach, "peak": alu_peak,
            "unit": "T fp64 instr/s", "frac": alu_ach / alu_peak,
            "traffic": NCU_DRAM_BYTES_PER_ZONE_STAGE_NEWTON * zones, "traffic_source": NCU_TRAFFIC_SOURCE,
            "peak_source": "148 SM x 64 fp64 lanes x %s sm_max_mhz %.0f" % (which, sm_max),
            "peak_measured": probe, "peak_measured_source": "grim_fp64_probe (DFMA, 8 chains/thread), this run",
            "frac_of_measured": alu_ach / probe,
            "alg_fp64_instr_per_zone_stage": ALG_FP64_INSTR_PER_ZONE_STAGE_NEWTON * it_scale,
            "executed_fp64_instr_per_zone_stage": EXECUTED_FP64_INSTR_PER_ZONE_STAGE_NEWTON * it_scale,
            "frac_executed": alu_ach / alu_peak * EXECUTED_FP64_INSTR_PER_ZONE_STAGE_NEWTON / ALG_FP64_INSTR_PER_ZONE_STAGE_NEWTON,
            "mean_newton_iterations": mean_it, "launch_ms": newton_ms, "launches": int(nk_n)},
        "roofline_hbm": None if not headline else {
            "bound": "hbm", "kernel": NEWTON_KERNEL, "achieved": hbm_ach,
            "peak": hbm_gbs, "unit": "GB/s", "frac": hbm_ach / hbm_gbs, "peak_source": which},
        "roofline_flux": None if not headline else {
            "bound": "alu", "kernel": "face_flux_tma_kernel x3 + face_box x3 + stage_const_tma_kernel (all flux-class launches of one stage)",
            "achieved": flux_alu, "peak": alu_peak, "unit": "T fp64 instr/s", "frac": flux_alu / alu_peak,
            "hbm_achieved_gbs": flux_hbm, "hbm_frac": flux_hbm / hbm_gbs,
            "traffic": NCU_DRAM_BYTES_PER_ZONE_STAGE_FLUX * zones, "traffic_source": NCU_TRAFFIC_SOURCE,
            "alg_fp64_instr_per_zone_stage": ALG_FP64_INSTR_PER_ZONE_STAGE_FLUX,
            "alg_bytes_per_zone_stage": ALG_BYTES_PER_ZONE_STAGE_FLUX, "stage_ms": flux_ms},
        "kernel_ms_per_step": {k: v[0] / args.steps for k, v in timing.items()},
        "newton_zone_iterations_per_s": (None if st is None else
                                         sum(i * (st.iters_hist[0][i] + st.iters_hist[1][i]) for i in range(16))
                                         / (2 * newton_ms * 1e-3)),
        "paper_context": "138,000 zones/s per K20 GPU, 48,000 zones/s per 16-core node (PAPER.md L414; 64^3/device)",
    }
    if world == 1 and not args.no_cpu_baseline:
        v, sps, cores = oracle_sample(args.ref_n, args.ref_steps, 0)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": "config-3 generator at %d^3, %d time steps (%.1f s)"
                                          % (args.ref_n, args.ref_steps, args.ref_steps * sps)}
    if world == 1 and not args.no_extras:
        del dP, hP, slab, g
        torch.cuda.empty_cache()
        try:
            line["other_workloads"] = other_workloads(local)
        except Exception as e:          # secondary numbers never cost the headline line
            line["other_workloads"] = {"error": repr(e)}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--n", type=int, default=256, help="zones per direction per GPU (headline 256)")
    ap.add_argument("--ref-n", type=int, default=96, help="grid size of the oracle's bounded sample")
    ap.add_argument("--ref-steps", type=int, default=12,
                    help="time steps of the oracle's sample in the cpu_baseline leg (96^3 x 12 ~ 15 s on 16 cores)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--flux-ct", action="store_true", help="flux-CT averaging of the B-field fluxes (not the headline)")
    ap.add_argument("--reduced", action="store_true",
                    help="the paper's reduced solve (B explicit, 7 x 7 Jacobian) instead of BASELINE's 10 unknowns")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs: keeps the launch list "
                                                            "to the device-resident steps)")
    ap.add_argument("--no-extras", action="store_true", help="skip the secondary workloads (config 2, Kerr step)")
    ap.add_argument("--dim", type=int, default=3, choices=[2, 3], help="2: the same generator on an n x n grid (X^2 slabs)")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"],
                    help="N > 1: nccl = one GPU per rank, device-to-device ghost planes; gloo = host-staged planes, ranks "
                         "may share a device (how a 1-GPU box exercises the N > 1 path)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # a plain `python bench.py --gpus N`: start one rank per GPU ourselves with the environment torchrun would set
        # (torchrun's own argument parser rejects script options it can read as abbreviations of its own, e.g. --n)
        import socket
        sk = socket.socket()
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
        sk.close()
        procs = []
        for r in range(args.gpus):
            env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(args.gpus), LOCAL_WORLD_SIZE=str(args.gpus),
                       MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
            procs.append(subprocess.Popen([sys.executable, os.path.abspath(__file__)] + sys.argv[1:], env=env))
        raise SystemExit(max(abs(p.wait()) for p in procs))
    if args.impl == "reference":
        run_reference(args)
    else:
        if args.warmup < 3:
            args.warmup = 3      # timing rule: at least 3 warm-up steps
        run_ours(args)


if __name__ == "__main__":
    main()
