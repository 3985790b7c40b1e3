"""`python bench.py --gpus N` must start N ranks (one process per GPU) when it is not already under torchrun
(work items are independent, so the path shards by index range)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_launcher_command_starts_one_rank_per_gpu():
    sys.path.insert(0, ROOT)
    import bench
    cmd = bench.launcher_command(["--gpus", "4", "--steps", "2"], 4, port=29511)
    assert cmd[:3] == [sys.executable, "-m", "torch.distributed.run"]
    assert "--nproc-per-node=4" in cmd and "--nnodes=1" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29511"
    k = cmd.index(os.path.join(ROOT, "bench.py"))
    assert cmd[k + 1:] == ["--gpus", "4", "--steps", "2"]
    free = bench.launcher_command([], 2)                     # picks a free port itself
    assert 1024 < int(free[free.index("--master-port") + 1]) < 65536


@pytest.mark.gpu
def test_bare_gpus_flag_runs_two_ranks_gloo_rehearsal():
    """The bare command, not under torchrun: two ranks are started, each integrates its shard of the doubled
    ensemble (disjoint global trajectory indices) and the moment sums are exchanged.  One GPU here, so the
    ranks share it and the collective is gloo (NCCL refuses two ranks on one device); the device-side path of
    sharding.MomentExchange is the same code with the reduce on the host tensor."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--backend", "gloo",
                        "--config", "3", "--sim-steps", "2000", "--steps", "2", "--warmup", "1"],
                       capture_output=True, text=True, env=env, timeout=900)
    assert r.returncode == 0, r.stderr[-3000:]
    assert "--nproc-per-node=2" in r.stderr
    assert r.stderr.count("[bench rank 0/2]") == 1 and r.stderr.count("[bench rank 1/2]") == 1
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                   # rank 0 alone prints
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["scaling"] == "weak" and out["value"] > 0
    assert out["result"]["step"] == 2000
    # the job's moments are those of 2 x 1,048,576 trajectories: checked against the single-rank run's sums
    # in tests/test_sharding.py (gloo, CPU); here the count of exchanged records is what matters
    assert out["config"]["moments_every"] == 1000 and out["gpu_launches"] > 0


@pytest.mark.gpu
@pytest.mark.parametrize("config,shard", [("3", "particles"), ("2", "sets")])
def test_strong_scaling_arm_two_ranks_gloo_rehearsal(config, shard):
    """--scaling strong divides the ONE ensemble: realisations of the single set (config[3]) or whole parameter
    sets (config[2]) per rank; the job's particle-steps are those of the undivided workload, and the exchanged
    moments count all of its trajectories."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--backend", "gloo",
                        "--scaling", "strong", "--config", config, "--sim-steps", "1000", "--steps", "2",
                        "--warmup", "1"], capture_output=True, text=True, env=env, timeout=900)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["scaling"] == "strong" and out["config"]["shard"] == shard
    total = {"3": 1_048_576, "2": 4_194_304}[config]
    assert out["config"]["trajectories_per_gpu"] == total // 2
    assert abs(out["value"] * out["ms_per_step"] * 1e-3 - total * 1000) < 1e-6 * total * 1000
    assert out["result"]["step"] == 1000


@pytest.mark.gpu
def test_gpus_flag_must_match_world_size():
    env = dict(os.environ, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--config", "0"],
                       capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode != 0 and "WORLD_SIZE is 1" in r.stderr
