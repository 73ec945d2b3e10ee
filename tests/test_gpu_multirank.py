"""N > 1 on hardware: `python bench.py --gpus 2` re-executes itself under torch.distributed.run, one
rank per GPU over NCCL, each rank a handle with its own first_realization.
Skipped on a box with fewer than two GPUs (this pool hands out one per call)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_two_ranks_run_the_sharded_bench():
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "2", "--warmup", "3",
                        "--sweeps-per-step", "100", "--no-per-config"], capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["scaling"] == "weak" and line["gpu_launches"] >= 2
    assert line["digest_ok"] in (True, None)          # rank 0's shard is the config itself


def test_gpus_flag_must_match_the_launcher():
    env = dict(os.environ, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--no-per-config"],
                       capture_output=True, text=True, timeout=600, env=env)
    assert r.returncode != 0 and "--gpus 2 but WORLD_SIZE is 1" in r.stderr
