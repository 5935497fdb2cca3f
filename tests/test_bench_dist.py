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


@pytest.mark.parametrize("name,scheme", [("cfg5", "cf4"), ("cfg4", "m4"), ("cfg3", "m4"), ("cfg2", "cf4")])
def test_headline_line_stays_below_4_kb(name, scheme):
    """The driver keeps only the tail of stdout: a 21 KB line (round 2) lost `value`, `roofline` and `e2e`.  The line
    is built here from stub results with worst-case widths (17-digit floats, every optional part present, a long
    clocks record) by bench.py's own build_line and must stay below bench.MAX_LINE_BYTES = 4096."""
    sys.path.insert(0, ROOT)
    import bench
    import workloads as W
    cfg = W.CONFIGS[name]
    x = 1234.5678901234567
    st = {"total_matvecs": 123456789, "n_exp": 123456, "seconds_leja": x, "seconds_commutator": x,
          "seconds_device": x, "kernel_launches": 1234567890}
    peaks = {"hbm_gbs": 6543.2109876543, "source": "measured (MEASURED_PEAKS.json)"}
    path = {"leja_kernel": "csr_leja_iter_sliceoff_kernel", "bytes_per_iteration": 11250000000,
            "csr_bytes_per_iteration": bench.algorithmic_bytes_per_iteration(cfg, scheme) if cfg.kind == "xxz" else 0,
            "slices": 524288, "slots": 20000000, "entries": 620756992}
    roof = bench.roofline_for(cfg, scheme, st, peaks, 37.123456789012, path)
    clocks = {"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "power_w_max": 987.654321, "samples": 12345,
              "reasons": ["hw_slowdown", "hw_thermal_slowdown", "sw_power_cap", "sw_thermal_slowdown"]}
    e2e = {"value": x, "unit": "steps/s", "h2d_bytes_per_step": x * 1e6, "d2h_bytes_per_step": x * 1e5, "steps": 5,
           "seconds": x, "seconds_integrate": x, "seconds_h2d_create_d2h": x, "seconds_all_trials": [x, x, x],
           "reported": "median of 3 calls"}
    cpu = {"value": x, "unit": "steps/s", "cores": 128, "kind": "oracle",
           "sample": "1 Magnus step(s) (CF4, tau=0.05) of the cfg5 recipe at N=24 (reduced from 16384), 42.47 s per step"}
    line = bench.build_line(cfg, scheme, 8, 12345, 123, x, x, st, 0.99999999999999989, clocks, roof, e2e, (x, x), cpu)
    text = json.dumps(line)
    assert len(text) < bench.MAX_LINE_BYTES == 4096, len(text)
    back = json.loads(text)
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "dtype", "data", "config", "clocks", "gpu_launches", "roofline", "e2e", "cpu_baseline"):
        assert key in back, key
    assert "extra" not in back
    for key in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert key in back["roofline"], key
    assert back["value"] > 0 and "workload" in back["config"]
