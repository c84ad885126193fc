"""bench.py's multi-GPU launch logic without a GPU: which process becomes which
rank, when bench.py re-executes itself under torch.distributed.run, and that it refuses -- with a
non-zero exit instead of a line whose n_gpus differs from --gpus -- what it cannot honour."""
import os
import subprocess
import sys

import bench
from paper_2606_21784_b200.workloads import shard_markets

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_single_gpu_runs_in_process():
    assert bench.launch_plan(1, {}, 1, []) == ("run", 0, 0, 1)
    assert bench.launch_plan(1, {}, 8, ["--steps", "2"]) == ("run", 0, 0, 1)


def test_torchrun_environment_is_honoured():
    env = {"WORLD_SIZE": "4", "RANK": "2", "LOCAL_RANK": "2"}
    assert bench.launch_plan(4, env, 8, []) == ("run", 2, 2, 4)
    assert bench.launch_plan(4, {"WORLD_SIZE": "4", "RANK": "3"}, 8, []) == ("run", 3, 3, 4)


def test_mismatches_are_errors_not_silent_single_gpu_runs():
    # torchrun with another rank count than --gpus
    assert bench.launch_plan(8, {"WORLD_SIZE": "2", "RANK": "0", "LOCAL_RANK": "0"}, 8, [])[0] == "error"
    assert bench.launch_plan(1, {"WORLD_SIZE": "2", "RANK": "0", "LOCAL_RANK": "0"}, 8, [])[0] == "error"
    # more ranks than visible devices
    assert bench.launch_plan(2, {"WORLD_SIZE": "2", "RANK": "1", "LOCAL_RANK": "1"}, 1, [])[0] == "error"
    assert bench.launch_plan(2, {}, 1, [])[0] == "error"
    assert bench.launch_plan(0, {}, 1, [])[0] == "error"
    assert bench.launch_plan(2, {"WORLD_SIZE": "2", "RANK": "5", "LOCAL_RANK": "0"}, 8, [])[0] == "error"


def test_plain_python_with_gpus_n_spawns_torchrun():
    kind, cmd = bench.launch_plan(2, {}, 2, ["--gpus", "2", "--steps", "3"])
    assert kind == "spawn"
    assert cmd[0] == sys.executable and cmd[1:3] == ["-m", "torch.distributed.run"]
    assert "--nproc-per-node" in cmd and cmd[cmd.index("--nproc-per-node") + 1] == "2"
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"
    assert 1024 <= int(cmd[cmd.index("--master-port") + 1]) < 65536
    assert cmd[-5:] == [os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "3"]


def test_reference_arm_needs_no_spawn():
    # CPU oracle: rank 0 alone works, whatever --gpus says; under torchrun the other ranks exit
    assert bench.launch_plan(4, {}, None, [], impl="reference") == ("run", 0, 0, 4)
    assert bench.launch_plan(4, {"WORLD_SIZE": "4", "RANK": "3", "LOCAL_RANK": "3"}, None, [], impl="reference") == ("run", 3, 3, 4)


def test_rank_markets_weak_and_strong():
    M = 65536
    for world in (1, 2, 4, 8):
        weak = [bench.rank_markets(M, r, world, "weak") for r in range(world)]
        assert [b for b, _, _ in weak] == [r * M for r in range(world)]
        assert all(n == M and tot == world * M for _, n, tot in weak)
        strong = [bench.rank_markets(M, r, world, "strong") for r in range(world)]
        assert [(b, n) for b, n, _ in strong] == [shard_markets(M, r, world) for r in range(world)]
        assert sum(n for _, n, _ in strong) == M and all(tot == M for _, _, tot in strong)
    b, n, tot = bench.rank_markets(7, 1, 2, "strong")
    assert (b, n, tot) == (4, 3, 7)


def test_bench_exits_nonzero_when_it_cannot_run_n_gpus():
    """On a box with fewer than 2 GPUs `python bench.py --gpus 2` must fail loudly (here: no GPU at all)."""
    import torch
    if torch.cuda.is_available() and torch.cuda.device_count() >= 2:
        import pytest
        pytest.skip("two GPUs are present")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=300)
    assert p.returncode != 0
    assert p.stdout.strip() == ""              # no JSON line
    assert "CUDA device" in p.stderr


def test_sass_counted_constants_cover_every_model():
    assert set(bench.EXEC_MULTS_PER_EVENT) == set(bench.ALG_MULTS_PER_EVENT)
    for k in bench.EXEC_MULTS_PER_EVENT:
        assert bench.EXEC_MULTS_PER_EVENT[k] <= bench.ALG_MULTS_PER_EVENT[k]
