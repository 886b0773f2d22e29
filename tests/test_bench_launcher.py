"""bench.py's multi-rank launch path on CPU: `python bench.py --gpus 2` with no
torchrun environment starts two ranks by itself (torch.distributed.run, gloo here because the arm is the CPU oracle),
prints ONE JSON line whose n_gpus is the number of ranks that joined, and refuses to print an n_gpus that the launch
does not back."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BENCH = os.path.join(ROOT, "bench.py")
SMALL = ["--impl", "reference", "--config", "1", "--muons", "3000", "--draws", "20000", "--steps", "1", "--warmup", "1",
         "--ref-seconds", "0.3"]


def _env(**extra):
    env = {k: v for k, v in os.environ.items()
           if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT", "MT_BENCH_SELF_LAUNCHED")}
    env.update(extra)
    return env


def _json_lines(stdout):
    return [json.loads(l) for l in stdout.splitlines() if l.startswith("{")]


def test_gpus_2_starts_two_ranks_by_itself():
    r = subprocess.run([sys.executable, BENCH, "--gpus", "2"] + SMALL, env=_env(), capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    assert len(lines) == 1                                      # rank 0 alone prints
    line = lines[0]
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["gpu_launches"] == 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert "torch.distributed.run" in r.stderr and "--nproc-per-node 2" in r.stderr


def test_gpus_1_runs_in_process():
    r = subprocess.run([sys.executable, BENCH, "--gpus", "1"] + SMALL, env=_env(), capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    assert len(lines) == 1 and lines[0]["n_gpus"] == 1
    assert "torch.distributed.run" not in r.stderr


def test_mismatched_world_size_is_refused():
    """a torchrun environment with fewer ranks than --gpus must not print a line that claims --gpus"""
    r = subprocess.run([sys.executable, BENCH, "--gpus", "4"] + SMALL,
                       env=_env(WORLD_SIZE="1", RANK="0", LOCAL_RANK="0"), capture_output=True, text=True, timeout=600)
    assert r.returncode != 0 and not _json_lines(r.stdout)
    assert "--gpus 4 but WORLD_SIZE=1" in r.stderr


def test_gpu_arm_without_a_gpu_fails_loudly():
    """no CPU fallback: on a box without CUDA the product arm refuses to run (and prints no line), also when it starts
    its own ranks"""
    import torch
    if torch.cuda.is_available():
        import pytest
        pytest.skip("this check is for the CPU box")
    for gpus in ("1", "2"):
        r = subprocess.run([sys.executable, BENCH, "--gpus", gpus, "--config", "1", "--muons", "1000", "--draws", "20000"],
                           env=_env(), capture_output=True, text=True, timeout=600)
        assert r.returncode != 0 and not _json_lines(r.stdout)
        assert "no CPU fallback" in r.stderr
