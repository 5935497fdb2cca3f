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
import os, sys, torch, torch.distributed as dist
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
# what bench.py does with the per-rank seconds of the timed region
t = torch.tensor([1.0 + rank], dtype=torch.float64)
dist.barrier()
dist.all_reduce(t, op=dist.ReduceOp.MAX)
steps = 5
if rank == 0:
    print("VALUE", world * steps / float(t.item()))
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
    res = _torchrun([str(script)])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("VALUE")]
    assert len(lines) == 1                                   # rank 0 alone prints
    assert abs(float(lines[0].split()[1]) - 2 * 5 / 2.0) < 1e-12   # N*K / max(1.0, 2.0)


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
