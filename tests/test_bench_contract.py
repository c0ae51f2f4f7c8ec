"""bench.py's reference arm (the oracle timed on the host cores) prints ONE JSON line with the contract's keys; rank != 0
of a multi-rank launch prints nothing.  Runs on CPU with a tiny sample."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run(env_extra=None):
    env = dict(os.environ)
    env.update(env_extra or {})
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                        "--warmup", "0", "--ref-n", "12"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr
    return [l for l in r.stdout.splitlines() if l.strip()]


def test_reference_arm_json_line():
    lines = run()
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["higher_is_better"] is True and d["unit"] == "zone-updates/s"
    assert d["value"] > 0 and d["steps"] == 1 and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["cpu_baseline"]["value"] == d["value"] == d["e2e"]["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["vs_baseline"] is None and "workload" in d["config"]


def test_reference_arm_other_ranks_are_silent():
    assert run({"RANK": "1", "WORLD_SIZE": "2"}) == []


import pytest


@pytest.mark.gpu
def test_our_arm_json_line_small():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--n", "32", "--steps", "3", "--warmup", "3",
                        "--no-extras", "--ref-n", "12", "--ref-steps", "1"], capture_output=True, text=True,
                       timeout=600)
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] == 3 and d["scaling"] == "weak"
    assert d["value"] > 0 and abs(d["value"] - 32 ** 3 * 3 / (d["ms_per_step"] * 3e-3)) < 1e-6 * d["value"]
    assert d["gpu_launches"] > 0
    rf = d["roofline"]
    assert rf["bound"] == "alu" and 0 < rf["frac"] < 1 and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-12
    assert rf["traffic"] > 0
    assert d["e2e"]["value"] > 0 and d["e2e"]["h2d_bytes_per_step"] == d["e2e"]["d2h_bytes_per_step"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] > 0
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    assert d["vs_baseline"] is None and d["dtype"] == "f64" and d["data"] == "synthetic"


def _run_two_ranks(backend):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--backend", backend, "--n", "16",
                        "--steps", "3", "--warmup", "3", "--no-extras", "--no-cpu-baseline"], capture_output=True,
                       text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                     # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "weak" and d["config"]["parallelism"] == "slab2"
    assert d["config"]["backend"] == backend and d["config"]["zones_per_gpu"] == 16 ** 3
    assert abs(d["value"] - 2 * 16 ** 3 * 3 / (d["ms_per_step"] * 3e-3)) < 1e-6 * d["value"]
    assert d["gpu_launches"] > 0 and d["e2e"]["value"] > 0


@pytest.mark.gpu
def test_bench_gpus2_plain_invocation_gloo_on_one_device():
    """`python bench.py --gpus 2` with no torchrun environment starts its own two ranks; with --backend gloo they may
    share the device (host-staged ghost planes), which is how a 1-GPU box runs the N > 1 code path end to end."""
    _run_two_ranks("gloo")


@pytest.mark.gpu
def test_bench_gpus2_nccl():
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs: the NCCL path has not been run on hardware (DESIGN.md section 9)")
    _run_two_ranks("nccl")
