"""bench.py's multi-rank launcher: `--gpus N` must start N ranks or
fail loudly -- never run fewer ranks than asked and never report a world size it did not run.  CPU only."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def test_launcher_command_is_the_drivers_form():
    cmd = bench.launcher_command(4, ["--gpus", "4", "--steps", "7", "--warmup", "3"], 29555)
    assert cmd[:3] == [sys.executable, "-m", "torch.distributed.run"]
    assert "--nnodes=1" in cmd and "--nproc-per-node=4" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"
    assert cmd[cmd.index("--master-port") + 1] == "29555"
    i = cmd.index(os.path.join(ROOT, "bench.py"))
    assert cmd[i + 1:] == ["--gpus", "4", "--steps", "7", "--warmup", "3"]      # the ranks see the same arguments


def test_resolve_world():
    assert bench.resolve_world(1, {}) == (1, 0, 0, False)
    assert bench.resolve_world(8, {}) == (8, 0, 0, True)                        # no torchrun yet: must spawn
    env = {"WORLD_SIZE": "8", "RANK": "5", "LOCAL_RANK": "5"}
    assert bench.resolve_world(8, env) == (8, 5, 5, False)
    with pytest.raises(SystemExit):                                             # launcher and --gpus disagree
        bench.resolve_world(4, env)
    with pytest.raises(SystemExit):
        bench.resolve_world(1, {"WORLD_SIZE": "2", "RANK": "0", "LOCAL_RANK": "0"})
    with pytest.raises(SystemExit):
        bench.resolve_world(0, {})


def test_gpus_2_without_two_gpus_fails_loudly():
    import torch
    if torch.cuda.is_available() and torch.cuda.device_count() >= 2:
        pytest.skip("box has two GPUs")
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--no-rows"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode != 0
    assert "needs 2 CUDA devices" in (r.stderr + r.stdout)
    assert '"n_gpus"' not in r.stdout                                           # no JSON line from a run that did not happen


def test_reference_arm_reports_the_real_world_size():
    """Under torchrun only rank 0 of the reference arm works; the other ranks exit 0 without output."""
    env = dict(os.environ, WORLD_SIZE="2", RANK="1", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
