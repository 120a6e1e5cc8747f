"""bench.py contract checks that need no GPU: the reference arm (the FP64 oracle on the host cores) prints one
JSON line with the keys the driver reads, and the native arm refuses to run without a CUDA device instead of
falling back to anything."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*args):
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                          cwd=ROOT, timeout=600)


def test_reference_arm_prints_the_contract_line():
    r = _run("--impl", "reference", "--steps", "1", "--warmup", "1", "--n", "4096")
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "Ginteractions/s" and line["higher_is_better"] is True
    assert line["value"] > 0 and line["steps"] == 1 and line["dtype"] == "f64" and line["data"] == "synthetic"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["cpu_baseline"]["value"] == line["value"]
    assert line["e2e"] == {"value": line["value"], "unit": line["unit"], "h2d_bytes_per_step": 0,
                           "d2h_bytes_per_step": 0}
    assert line["vs_baseline"] is None and "workload" in line["config"]


def test_native_arm_has_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        return                                   # on the GPU box the native arm is exercised by the driver
    r = _run("--steps", "1", "--warmup", "0", "--n", "4096", "--no-cpu-baseline", "--no-step-loops")
    assert r.returncode != 0
    assert "no CPU fallback" in (r.stderr + r.stdout)


def test_reference_arm_under_torchrun_env_only_rank0_prints():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--n", "4096"], capture_output=True, text=True, cwd=ROOT,
                       env=env, timeout=600)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_native_arm_with_more_gpus_than_the_box_has_fails_loudly():
    """`python bench.py --gpus N` (no torchrun) starts N ranks itself; with fewer than N devices it must refuse
    instead of timing one GPU and printing n_gpus: 1 (round-1 finding)."""
    import torch
    need = torch.cuda.device_count() + 2
    r = _run("--gpus", str(need), "--steps", "1", "--warmup", "0")
    assert r.returncode != 0
    assert "refusing to run fewer ranks" in (r.stderr + r.stdout)


def test_native_arm_rejects_a_world_size_that_contradicts_gpus():
    env = dict(os.environ, RANK="0", WORLD_SIZE="2", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "4", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, cwd=ROOT, env=env, timeout=600)
    assert r.returncode != 0 and "WORLD_SIZE=2" in (r.stderr + r.stdout)
