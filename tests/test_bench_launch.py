"""CPU-only: `python bench.py --gpus N` starts its own N ranks (one process per GPU, replicas / shards with no
data-path collective).  The re-exec plumbing is pure host logic and is checked here without a GPU; on a box with fewer than
N GPUs the launcher must refuse loudly instead of printing an n_gpus it did not run on."""
import argparse
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402


def _args(gpus, impl="arachne", sp="none"):
    return argparse.Namespace(gpus=gpus, impl=impl, sp=sp)


def test_self_launch_is_needed_only_outside_torchrun_for_more_than_one_gpu():
    assert not bench.needs_self_launch(_args(1), {})
    assert bench.needs_self_launch(_args(8), {})
    assert not bench.needs_self_launch(_args(8), {"WORLD_SIZE": "8"})          # the driver's torchrun launch: ranks exist already
    assert not bench.needs_self_launch(_args(8, "reference"), {})              # the oracle arm runs on rank 0's host cores only


def test_self_launch_command_is_the_driver_contract_with_the_callers_flags():
    argv = ["--gpus", "4", "--steps", "7", "--warmup", "3", "--workload", "heavytail"]
    cmd = bench.self_launch_argv(argv, 4, 29555, python="python3")
    assert cmd[:3] == ["python3", "-m", "torch.distributed.run"]
    assert "--nnodes=1" in cmd and "--nproc-per-node=4" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29555"
    i = cmd.index(os.path.join(ROOT, "bench.py"))
    assert cmd[i + 1:] == argv                                                 # every flag reaches the ranks unchanged
    p = bench.free_port()
    assert 1024 <= p < 65536


def test_more_gpus_than_the_node_has_is_refused_loudly():
    """Here (no GPU) and on a 1-GPU box alike: --gpus 2 must not silently run as one rank."""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1"], capture_output=True, text=True,
                       env={k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}, timeout=300)
    assert r.returncode != 0
    assert "refusing to emulate ranks" in r.stderr and '"n_gpus"' not in r.stdout
