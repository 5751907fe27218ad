"""bench.py --gpus N cannot silently run fewer ranks than it was asked for (no GPU needed)."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(args, env_extra=None, drop=("WORLD_SIZE", "RANK", "LOCAL_RANK")):
    env = {k: v for k, v in os.environ.items() if k not in drop}
    env.update(env_extra or {})
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, env=env,
                          timeout=300)


def test_more_gpus_than_devices_fails_loudly():
    import torch
    if torch.cuda.is_available() and torch.cuda.device_count() >= 2:
        pytest.skip("two CUDA devices present: the launch would go ahead")
    r = _run(["--gpus", "2", "--steps", "1", "--warmup", "1", "--workload", "C0"])
    assert r.returncode != 0
    assert "--gpus 2" in r.stderr and "not running on fewer" in r.stderr
    assert r.stdout.strip() == ""            # no JSON line that could be read as a measurement


def test_world_size_that_contradicts_gpus_fails_loudly():
    r = _run(["--gpus", "2", "--steps", "1", "--warmup", "1", "--workload", "C0"],
             env_extra={"WORLD_SIZE": "3", "RANK": "0", "LOCAL_RANK": "0"})
    assert r.returncode != 0 and "WORLD_SIZE = 3" in r.stderr and r.stdout.strip() == ""
    r = _run(["--steps", "1", "--warmup", "1", "--workload", "C0"], env_extra={"WORLD_SIZE": "2", "RANK": "0", "LOCAL_RANK": "0"})
    assert r.returncode != 0 and "--gpus 1" in r.stderr
