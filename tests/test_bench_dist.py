"""Host logic of bench.py's multi-process path, on CPU with gloo (world size 2).

The path does not shard (replicas only), so the only multi-rank logic is: every rank
times its own replica, the MAX over ranks is taken, rank 0 alone prints, and in the reference arm the other
ranks exit 0 without work.  No GPU is needed for either check.
"""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, torch.distributed as dist
sys.path.insert(0, os.environ["BENCH_ROOT"])
import bench                                    # bench.py's own reduction code, not a copy of it
dist.init_process_group("gloo")
rank = dist.get_rank()
dist.barrier()
value, sec = bench.whole_job_value(5, 1.0 + rank, dist, "cpu")     # per-rank seconds of the timed region: 1.0, 2.0
if rank == 0:
    print("VALUE", value, sec)
dist.barrier()
dist.destroy_process_group()
"""


def _torchrun(args, env_extra=None, timeout=300):
    env = dict(os.environ)
    env.update(env_extra or {})
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", "29611"] + args
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_max_over_ranks_and_whole_job_value(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    res = _torchrun([str(script)], env_extra={"BENCH_ROOT": ROOT})
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("VALUE")]
    assert len(lines) == 1                                   # rank 0 alone prints
    assert abs(float(lines[0].split()[1]) - 2 * 5 / 2.0) < 1e-12   # N*K / max(1.0, 2.0)
    assert abs(float(lines[0].split()[2]) - 2.0) < 1e-12           # the slowest rank's seconds


def test_single_process_reduction_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(1.25) == 1.25
    assert bench.whole_job_value(4, 2.0) == (2.0, 2.0)


def test_gpus_flag_must_match_world_size():
    """`--gpus 2` inside a 1-process environment that claims WORLD_SIZE=1 is refused, not silently run on one GPU."""
    import torch
    env = dict(os.environ, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0")
    res = subprocess.run([sys.executable, "bench.py", "--gpus", "2", "--steps", "1", "--warmup", "0"], cwd=ROOT, env=env,
                         capture_output=True, text=True, timeout=300)
    assert res.returncode != 0
    msg = res.stderr + res.stdout
    assert ("no CUDA device" in msg) if not torch.cuda.is_available() else ("WORLD_SIZE=1" in msg)


def test_reference_arm_rank0_only():
    """bench.py --impl reference under torchrun: rank 0 runs the oracle on a small bounded sample and prints
    one JSON line; rank 1 exits 0 without output."""
    res = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--workload",
                     "cfg1"], timeout=600)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "steps/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


def test_ours_arm_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    res = subprocess.run([sys.executable, "bench.py", "--steps", "1", "--warmup", "0"], cwd=ROOT, capture_output=True,
                         text=True, timeout=300)
    assert res.returncode != 0 and "no CUDA device" in (res.stderr + res.stdout)
