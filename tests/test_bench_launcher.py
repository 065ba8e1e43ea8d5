"""bench.py --gpus N: the launcher sets up N worker environments itself and refuses to print an N-GPU number
from fewer devices (CPU-side checks; the GPU runs are the driver's)."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_launcher_envs_one_rank_per_gpu():
    import bench
    envs = bench.launcher_envs(4, 29517, {"PATH": "/x", "NCCL_DEBUG": "WARN"})
    assert len(envs) == 4
    for i, e in enumerate(envs):
        assert e["RANK"] == str(i) and e["LOCAL_RANK"] == str(i) and e["WORLD_SIZE"] == "4"
        assert e["MASTER_ADDR"] == "127.0.0.1" and e["MASTER_PORT"] == "29517"
        assert e["PATH"] == "/x" and e["NCCL_DEBUG"] == "WARN"      # the caller's settings win
    assert bench.launcher_envs(2, 1, {})[1]["NCCL_DEBUG"] == "INFO"  # communicator lines on by default


def test_gpus_flag_fails_loudly_without_enough_devices():
    """On a box with fewer than N CUDA devices `bench.py --gpus N` exits non-zero and prints no JSON line."""
    import torch
    have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    n = have + 2
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", str(n), "--steps", "1", "--warmup", "1"],
                       env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode != 0
    assert "refusing" in r.stderr and "{" not in r.stdout


def test_world_size_must_match_gpus_flag():
    env = dict(os.environ, WORLD_SIZE="2", RANK="0", LOCAL_RANK="0", MASTER_ADDR="127.0.0.1", MASTER_PORT="29518")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "4", "--steps", "1", "--warmup", "1"],
                       env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode != 0 and "{" not in r.stdout
