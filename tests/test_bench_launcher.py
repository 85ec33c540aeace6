"""`python bench.py --gpus N` starts N ranks by itself (one process per GPU, rows sharded, no
collective on the data path) and never reports a smaller run under the label of a larger one."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402


def test_child_command_starts_one_rank_per_gpu_on_this_node():
    cmd = bench.launcher_command(8, ["--gpus", "8", "--steps", "5", "--warmup", "3"], master_port=29511)
    assert cmd[:3] == [sys.executable, "-m", "torch.distributed.run"]
    assert "--nnodes=1" in cmd and "--nproc-per-node=8" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"
    assert cmd[cmd.index("--master-port") + 1] == "29511"
    script = cmd.index(os.path.join(ROOT, "bench.py"))
    assert cmd[script + 1:] == ["--gpus", "8", "--steps", "5", "--warmup", "3"]  # the ranks see the same arguments


def test_more_gpus_than_visible_is_refused():
    with pytest.raises(SystemExit) as e:
        bench.check_gpus(8, 1)
    assert "8" in str(e.value) and "1 CUDA device" in str(e.value)
    with pytest.raises(SystemExit):
        bench.check_gpus(0, 1)
    bench.check_gpus(2, 2)
    bench.check_gpus(1, 8)


def test_the_documented_command_fails_loudly_without_enough_devices():
    import torch

    if torch.cuda.is_available() and torch.cuda.device_count() >= 2:
        pytest.skip("two GPUs visible: the command would really run")
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "1"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode != 0
    assert "--gpus 2 requested" in r.stderr and '"n_gpus"' not in r.stdout
