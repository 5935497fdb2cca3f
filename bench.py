#!/usr/bin/env python
"""bench.py -- Magnus steps/s of the CUDA hot path on B200, with its roofline and the oracle beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5] [--scheme cf4]
    python bench.py --impl reference ...        # the CPU oracle on the same metric/config (rank 0 only)

A "step" is one Magnus time step t -> t + tau (rows S1..S8 of SURVEY.md section 8(a); D3/D4 too
for M4 on dense H) through the C-ABI call magnus_integrate on a synthetic workload of
BASELINE.json (workloads/configs.py).  Default workload: cfg5, the largest single-GPU config
(XXZ chain N=24, 620,756,992 stored entries, 12.4 GB of CSR: far larger than the 126 MB L2, so no
flush is needed between timed steps).  Rank 0 prints ONE JSON line.

  value      steps/s, inputs resident in HBM, CUDA events on the launching stream, max over ranks
  e2e        steps/s of magnus_integrate_host: HOST (pinned) H0, H1, psi -> H2D -> create -> K steps
             -> D2H psi, all inside the timed region (wall clock around the blocking call)
  roofline   fused Leja iteration kernel (dense: the GEMV variant; with --scheme m4 on dense H the
             DMMA commutator): algorithmic bytes (flops) per launch / mean launch time measured
             live with CUDA events inside the timed region, against MEASURED_PEAKS.json
  cpu_baseline  the oracle (oracle/, test infrastructure) timed on this box's host cores on a bounded sample:
             ONE Magnus step of the SAME workload at full size (N = 24 for cfg5; about 45 s)
  --extra FILE.json   (opt-in) secondary measurements (cfg1-cfg4 in both schemes, the beyond-paper shortcuts) written
             to FILE.json; they never enter the headline line, which stays below MAX_LINE_BYTES so that the driver's
             stored tail always holds it whole

Multi-GPU: the path does not shard ("replicas only"); --gpus N runs N
independent replicas, one process per GPU, no data-path collective, scaling "weak".
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "magnus_steps_per_s"
UNIT = "steps/s"

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed
# `ncu --set full` captures (profiles/r1_csr_rowblock_ncu.md, profiles/r1_dense_gemv_ncu.md); None = not captured.
# Keyed by (config, scheme, kernel): a capture only describes the kernel it was taken on.
NCU_TRAFFIC_BYTES = {("cfg5", "cf4", "csr_leja_iter_sliceoff_kernel"): 12.737e9,
                     ("cfg5", "cf4", "csr_leja_iter_rowblock_kernel"): 15.093e9,
                     ("cfg4", "cf4", "dense_leja_iter_kernel"): 4.299e9}
NCU_TRAFFIC_SOURCE = {("cfg5", "cf4", "csr_leja_iter_sliceoff_kernel"): "profiles/r2_csr_sliceoff_ncu.md",
                      ("cfg5", "cf4", "csr_leja_iter_rowblock_kernel"): "profiles/r1_csr_rowblock_ncu.md",
                      ("cfg4", "cf4", "dense_leja_iter_kernel"): "profiles/r1_dense_gemv_ncu.md"}
MAX_LINE_BYTES = 4096     # the headline JSON line must stay below this (a 21 KB line was cut off in the driver's record)


# ----------------------------------------------------------------------------- helpers
def load_peaks():
    """MEASURED_PEAKS.json (driver-written) or the fallback of B200_PROFILING.md."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            p = json.load(fh)
        return {"hbm_gbs": float(p["hbm_gbs"]), "source": "measured (MEASURED_PEAKS.json)"}
    except Exception:
        return {"hbm_gbs": 6650.0, "source": "fallback (B200_PROFILING.md)"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)     # at least one sample even for a very short region
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [x.strip() for x in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
                pw.append(float(parts[2]))
            except ValueError:
                continue
            for nm, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def workload_description(cfg, scheme):
    if cfg.kind == "xxz":
        N = cfg.size
        return (f"{cfg.name}: periodic XXZ chain N={N} (dim 2^{N}) + cos(2t) transverse field, CSR complex128/int32, "
                f"nnz {(1 << N) * (3 * N + 2) // 2}, {scheme.upper()}, tau={cfg.tau:g}, tol={cfg.tol:g}")
    return (f"{cfg.name}: dense random Hermitian H0 + sin(3t) H1, n={cfg.size} complex128 row-major, "
            f"{scheme.upper()}, tau={cfg.tau:g}, tol={cfg.tol:g}")


def algorithmic_bytes_per_iteration(cfg, scheme):
    """SURVEY.md section 8(d) / DESIGN.md section 5: what one fused Leja iteration must move."""
    n = cfg.n
    if cfg.kind == "xxz":
        N = cfg.size
        nnz = (1 << N) * (3 * N + 2) // 2            # H0 + H1 (disjoint patterns)
        terms = 2
        if scheme == "m4":
            nnz += N * (1 << (N - 1))                # cached C = [H0, H1]
            terms = 3
        return 20 * nnz + 4 * (n + 1) * terms + 64 * n
    return 16 * n * n + 64 * n


# ----------------------------------------------------------------------------- reference arm (CPU oracle)
def oracle_sample(cfg, scheme, max_size=None):
    """The bounded sample the oracle is timed on: ONE Magnus step of the workload's recipe at FULL size (same
    config as the GPU arm).  Only dense M4 by the plain definition (two n^3 products per step: hours at
    n = 16384) is reduced, to n = 4096, and the sample says so."""
    import workloads as W
    size = cfg.size
    if max_size is not None:
        size = min(size, max_size)
    elif cfg.kind == "dense" and scheme in ("m4", "m6"):
        size = min(size, 4096 if scheme == "m4" else 2048)
    elif cfg.kind == "xxz" and scheme == "m6":
        size = min(size, 12)
    return W.scaled(cfg, size, 1)


def time_oracle(cfg, scheme, steps, warmup, max_size=None):
    """Times `steps` single Magnus steps of the oracle as it stands (OpenMP over rows, plain loops)."""
    import numpy as np
    import torch
    import workloads as W
    from oracle import oracle as O
    sample = oracle_sample(cfg, scheme, max_size)
    dev = "cuda" if torch.cuda.is_available() else "cpu"     # generators only; the oracle gets host arrays
    H0, H1, psi0, f = W.build(sample, device=dev)
    if sample.kind == "xxz":
        o0, o1 = O.CsrHost.of(H0), O.CsrHost.of(H1)
    else:
        o0, o1 = H0.cpu().numpy(), H1.cpu().numpy()
    psi = psi0.cpu().numpy()
    del H0, H1
    cores = O.num_threads()
    times = []
    for i in range(warmup + steps):
        t = sample.t0 + i * sample.tau
        t0 = time.perf_counter()
        psi, _ = O.magnus_step(o0, o1, f, scheme, t, sample.tau, psi, sample.tol)
        dt = time.perf_counter() - t0
        if i >= warmup:
            times.append(dt)
    sec = sum(times) / len(times)
    desc = (f"{len(times)} Magnus step(s) ({scheme.upper()}, tau={sample.tau:g}) of the {cfg.name} recipe at "
            f"{'N' if sample.kind == 'xxz' else 'n'}={sample.size}"
            f"{'' if sample.size == cfg.size else f' (reduced from {cfg.size})'}, {sec:.2f} s per step")
    return {"value": 1.0 / sec, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
            "sample_size": sample.size, "full_size": cfg.size}


def run_reference(args):
    """The reference arm is the CPU oracle (the tier has no reference code).  It times ONE Magnus step of the same
    workload at full size, without warm-up (a step is tens of seconds of host time; `--steps K` would not end
    within minutes), and reports the steps it actually timed."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    import workloads as W
    cfg = W.CONFIGS[args.workload]
    scheme = args.scheme or cfg.schemes[0]
    timed = 1 if args.oracle_steps is None else max(1, args.oracle_steps)
    base = time_oracle(cfg, scheme, timed, 0, args.oracle_max_size)
    line = {"impl": "reference", "metric": METRIC, "value": base["value"], "unit": UNIT, "n_gpus": max(1, world),
            "steps": timed, "warmup": 0, "ms_per_step": 1e3 / base["value"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "complex128 (f64)", "data": "synthetic",
            "config": {"workload": workload_description(cfg, scheme), "scheme": scheme,
                       "note": "CPU oracle (oracle/), rank 0 only; timed steps = 'steps' (requested: "
                               f"--steps {args.steps} --warmup {args.warmup}); each step is one Magnus step of the sample",
                       "same_size_as_gpu_arm": base["sample_size"] == base["full_size"]},
            "cpu_baseline": {k: base[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": base["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------- our arm
XXZ_MATRIX_FREE = "xxz-matrix-free"      # shortcut key of measure_workload: magnus_create_xxz instead of matrices


def measure_workload(M, W, torch, cfg, scheme, steps, warmup, dev, barrier, sampler=None, shortcuts=0):
    """Warm up, then time exactly `steps` Magnus steps with inputs resident in HBM."""
    stream = torch.cuda.current_stream()
    out = {}
    if shortcuts == XXZ_MATRIX_FREE:       # BASELINE's chain: sx sx + sy sy + 0.5 sz sz, field sx, f = cos 2t
        from workloads import rng, xxz
        H0 = H1 = None
        psi0 = xxz.neel_state(cfg.size, device=dev) if cfg.psi0 == "neel" else rng.random_unit_vector(cfg.n, device=dev)
        f = cfg.f
        handle = M.magnus_create_xxz(cfg.size, 1.0, 0.5, 1.0, f, scheme, tol=cfg.tol, stream=stream)
    else:
        H0, H1, psi0, f = W.build(cfg, device=dev)
        handle = M.magnus_create(H0, H1, f, scheme, tol=cfg.tol, stream=stream, shortcuts=shortcuts)
    with handle as h:
        psi = psi0.clone()
        if warmup > 0:
            h.integrate(cfg.t0, cfg.t0 + warmup * cfg.tau, warmup, psi)
        psi.copy_(psi0)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        torch.cuda.synchronize()
        if sampler:
            sampler.start()
        e0.record(stream)
        st = h.integrate(cfg.t0, cfg.t0 + steps * cfg.tau, steps, psi)
        e1.record(stream)
        torch.cuda.synchronize()
        barrier()
        out["clocks"] = sampler.stop() if sampler else None
        out["seconds"] = e0.elapsed_time(e1) * 1e-3
        out["stats"] = st
        out["path"] = h.describe()
        out["norm"] = float(torch.linalg.vector_norm(psi))
    out["inputs"] = (H0, H1, psi0, f)
    return out


def matrix_bytes(H):
    if hasattr(H, "row_ptr"):
        return H.values.numel() * 16 + H.col_idx.numel() * 4 + H.row_ptr.numel() * 4
    return H.numel() * 16


def measure_e2e(M, torch, cfg, scheme, steps, inputs):
    """magnus_integrate_host with pinned HOST buffers: H2D + create + K steps + D2H inside the timed region."""
    from workloads import xxz
    H0, H1, psi0, f = inputs

    def pinned(t):
        return torch.empty(t.shape, dtype=t.dtype, pin_memory=True).copy_(t)

    if hasattr(H0, "row_ptr"):
        P0 = xxz.CSR(H0.n, pinned(H0.row_ptr), pinned(H0.col_idx), pinned(H0.values))
        P1 = xxz.CSR(H1.n, pinned(H1.row_ptr), pinned(H1.col_idx), pinned(H1.values))
    else:
        P0, P1 = pinned(H0), pinned(H1)
    psi = pinned(psi0)
    h2d = matrix_bytes(H0) + matrix_bytes(H1) + psi0.numel() * 16
    d2h = psi0.numel() * 16
    # the whole call three times, the MEDIAN reported (all three listed): its large device allocations take between
    # 0.02 s and 1 s depending on the state of the driver's memory pools, so a single call is noisy either way
    trials = []
    for _ in range(3):
        psi.copy_(psi0)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        st_i = M.magnus_integrate_host(P0, P1, f, scheme, cfg.t0, cfg.t0 + steps * cfg.tau, steps, psi, tol=cfg.tol,
                                       stream=torch.cuda.current_stream())
        torch.cuda.synchronize()
        trials.append((time.perf_counter() - t0, st_i))
    sec, st = sorted(trials, key=lambda x: x[0])[1]
    return {"seconds_all_trials": [round(t, 4) for t, _ in trials], "reported": "median of 3 calls",
            "value": steps / sec, "unit": UNIT, "h2d_bytes_per_step": h2d / steps, "d2h_bytes_per_step": d2h / steps,
            "seconds": sec, "seconds_integrate": st["seconds_device"], "seconds_h2d_create_d2h": sec - st["seconds_device"],
            "steps": steps, "matvecs": st["total_matvecs"]}


def roofline_for(cfg, scheme, st, peaks, fp64_peak_tflops, path=None):
    r = _roofline_for(cfg, scheme, st, peaks, fp64_peak_tflops, path)
    if r["bound"] == "hbm":
        key = (cfg.name, scheme, r["kernel"].split(" ")[0])
        r["traffic"] = NCU_TRAFFIC_BYTES.get(key)
        r["traffic_source"] = NCU_TRAFFIC_SOURCE.get(key)
    return r


def _roofline_for(cfg, scheme, st, peaks, fp64_peak_tflops, path=None):
    """Dominant kernel of the step: the fused Leja iteration (HBM) or, for M4 on dense H, the DMMA commutator."""
    leja_s, comm_s, mv = st["seconds_leja"], st["seconds_commutator"], max(1, st["total_matvecs"])
    nsteps_exp = max(1, st["n_exp"])
    if cfg.kind == "dense" and scheme in ("m4", "m6") and comm_s > leja_s:
        # M4: one complex product P = A2 A1 per step (K = P - P^H); M6: three (magnus.h at magnus_step)
        flops = 8.0 * cfg.n ** 3 * (3 if scheme == "m6" else 1)
        achieved = flops * nsteps_exp / comm_s / 1e12
        return {"kernel": "zgemm_dmma_kernel", "bound": "tensor", "achieved": achieved, "peak": fp64_peak_tflops,
                "unit": "TFLOP/s", "frac": achieved / fp64_peak_tflops if fp64_peak_tflops else None, "traffic": None,
                "peak_source": "magnus_fp64_peaks: DMMA m8n8k4 micro-benchmark run in this process",
                "flops_per_launch": flops}
    # bytes of the variant the library actually runs (magnus_describe): "never count bytes a variant does not
    # move"; the plain-CSR figure of SURVEY 8(d) is reported beside it as csr_equivalent
    csr_bytes = algorithmic_bytes_per_iteration(cfg, scheme)
    nbytes = path["bytes_per_iteration"] if path and path.get("bytes_per_iteration") else csr_bytes
    kernel = path["leja_kernel"] if path else ("dense_leja_iter_kernel" if cfg.kind == "dense" else "csr")
    if path and path.get("csr_bytes_per_iteration"):
        assert path["csr_bytes_per_iteration"] == csr_bytes, (path, csr_bytes)
    ms = leja_s / mv * 1e3
    achieved = nbytes / (ms * 1e-3) / 1e9
    if kernel.startswith("csr_leja_sweep_small") or (cfg.kind == "dense" and cfg.n <= 4096):
        kernel += " (L2-resident, latency bound)"
    r = {"kernel": kernel, "bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
         "frac": achieved / peaks["hbm_gbs"], "traffic": None, "peak_source": peaks["source"],
         "bytes_per_launch": nbytes, "ms_per_launch": ms, "frac_of_nominal_8TBs": achieved / 8000.0}
    if cfg.kind != "dense":
        eq = csr_bytes / (ms * 1e-3) / 1e9
        # SURVEY 8(d) plain-CSR bytes over the same time: what a CSR-reading kernel would have to sustain to be as
        # fast -- not a bandwidth this kernel achieves
        r["csr_equivalent"] = {"bytes_per_launch": csr_bytes, "gbs": eq, "frac": eq / peaks["hbm_gbs"]}
        if path and path.get("slots"):
            r["layout"] = {k: path[k] for k in ("slices", "slots", "entries")}
    return r


def max_over_ranks(seconds: float, dist=None, device="cpu") -> float:
    """The timed region of the job is the slowest rank's: MAX over ranks of the per-rank seconds (every rank gets
    the result).  `dist` is torch.distributed when a process group is up, else None (single process)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(seconds)
    import torch
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(steps: int, seconds_per_rank: float, dist=None, device="cpu"):
    """(value, seconds): steps/s summed over all replicas = world * steps / max-over-ranks seconds."""
    world = dist.get_world_size() if dist is not None and dist.is_initialized() else 1
    sec = max_over_ranks(seconds_per_rank, dist, device)
    return world * steps / sec, sec


def respawn_under_torchrun(args) -> int:
    """`python bench.py --gpus N` without a launcher: start N replicas, one process per GPU, over NCCL."""
    port = 29500 + (os.getpid() % 2000)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def measure_extra(M, W, torch, dev, peaks, dmma_tf):
    """Short secondary measurements for the default line, so that the driver's record carries every part of the
    metric: cfg4 CF4 (dense GEMV GB/s), cfg4 M4 (DMMA commutator TFLOP/s), the latency-bound configs cfg1 / cfg2
    (whole-sweep kernels, planned batches) and cfg3 (the CSR kernel at N = 20) and, reported separately from the
    mandated path, cfg4 M4 with the cached-commutator shortcut."""
    out = {}
    runs = (("cfg4", "cf4", 2, 1, 0, "cfg4_cf4"), ("cfg4", "m4", 1, 1, 0, "cfg4_m4"),
            ("cfg1", "cf4", 100, 20, 0, "cfg1_cf4"), ("cfg1", "m4", 100, 20, 0, "cfg1_m4"),
            ("cfg2", "cf4", 50, 10, 0, "cfg2_cf4"), ("cfg2", "m4", 20, 3, 0, "cfg2_m4"),
            ("cfg3", "cf4", 10, 3, 0, "cfg3_cf4"), ("cfg3", "m4", 10, 3, 0, "cfg3_m4"),
            ("cfg4", "m4", 2, 1, M.SHORTCUT_CACHED_COMMUTATOR, "cfg4_m4_shortcut_cached_commutator"),
            ("cfg4", "cf4", 2, 1, M.SHORTCUT_TIGHT_INTERVAL, "cfg4_cf4_shortcut_tight_interval"),
            ("cfg5", "cf4", 5, 3, M.SHORTCUT_REAL_VALUES, "cfg5_cf4_shortcut_real_values"),
            ("cfg5", "cf4", 5, 3, XXZ_MATRIX_FREE, "cfg5_cf4_shortcut_matrix_free"),
            ("cfg3", "cf4", 10, 3, XXZ_MATRIX_FREE, "cfg3_cf4_shortcut_matrix_free"))
    for name, scheme, steps, warmup, shortcuts, key in runs:
        cfg = W.CONFIGS[name]
        sampler = ClockSampler(torch.cuda.current_device())
        res = measure_workload(M, W, torch, cfg, scheme, steps, warmup, dev, lambda: None, sampler, shortcuts)
        st = res["stats"]
        roof = roofline_for(cfg, scheme, st, peaks, dmma_tf, res.get("path"))
        out[key] = {"workload": workload_description(cfg, scheme), "steps": steps, "warmup": warmup,
                    "shortcut": {XXZ_MATRIX_FREE: "matrix-free XXZ (magnus_create_xxz)",
                                 M.SHORTCUT_REAL_VALUES: "real-part storage", M.SHORTCUT_TIGHT_INTERVAL: "Lanczos interval",
                                 M.SHORTCUT_CACHED_COMMUTATOR: "cached dense commutator"}.get(shortcuts),
                    "value": steps / res["seconds"], "unit": UNIT, "ms_per_step": res["seconds"] / steps * 1e3,
                    "matvecs": st["total_matvecs"], "lanczos_matvecs": st.get("lanczos_matvecs", 0),
                    "seconds_leja": st["seconds_leja"],
                    "seconds_commutator": st["seconds_commutator"], "gpu_launches": st["kernel_launches"],
                    "clocks": res["clocks"], "roofline": roof, "psi_norm_after": res["norm"]}
        res["inputs"] = None
        del res
        torch.cuda.empty_cache()
    return out


def _r(x, digits=6):
    """Shorten a float to `digits` significant digits for the printed line."""
    return float(f"{x:.{digits}g}") if isinstance(x, float) and math.isfinite(x) else x


def build_line(cfg, scheme, world, steps, warmup, value, sec, st, psi_norm, clocks, roof, e2e, fp64_peaks, cpu_baseline):
    """The ONE headline JSON line, kept below MAX_LINE_BYTES: only what the bench contract names.  Explanations of
    how each figure is measured are in DESIGN.md section 7, not in the line."""
    roof_keys = ("kernel", "bound", "achieved", "peak", "unit", "frac", "traffic", "traffic_source", "bytes_per_launch",
                 "flops_per_launch", "ms_per_launch", "peak_source", "frac_of_nominal_8TBs", "csr_equivalent")
    line = {"metric": METRIC, "value": _r(value), "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
            "ms_per_step": _r(sec / steps * 1e3), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "complex128 (f64)", "data": "synthetic",
            "config": {"workload": workload_description(cfg, scheme), "scheme": scheme,
                       "parallelism": "replicas only (no sharding, no collective)" if world > 1 else "1 GPU",
                       "l2": "inputs larger than L2 (no flush needed)" if matrix_bytes_cfg(cfg) > 256e6 else
                             "fits L2: latency bound",
                       "matvecs": st["total_matvecs"], "exponentials": st["n_exp"],
                       "seconds_leja": _r(st["seconds_leja"]), "seconds_commutator": _r(st["seconds_commutator"]),
                       "psi_norm_after": psi_norm},
            "clocks": clocks, "gpu_launches": st["kernel_launches"],
            "roofline": {k: ({kk: _r(vv) for kk, vv in roof[k].items()} if isinstance(roof[k], dict) else _r(roof[k]))
                         for k in roof_keys if k in roof},
            "fp64_peaks_measured_tflops": {"dmma": _r(fp64_peaks[0]), "dfma": _r(fp64_peaks[1])}}
    if e2e:
        line["e2e"] = {k: _r(e2e[k]) for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "steps",
                                                "seconds", "seconds_integrate", "seconds_h2d_create_d2h",
                                                "seconds_all_trials", "reported") if k in e2e}
    if cpu_baseline:
        line["cpu_baseline"] = {k: _r(v) for k, v in cpu_baseline.items()}
    n = len(json.dumps(line))
    if n >= MAX_LINE_BYTES:      # never print a line the driver cannot store whole: drop the optional parts first
        for k in ("fp64_peaks_measured_tflops",):
            line.pop(k, None)
        line["roofline"].pop("csr_equivalent", None)
        line["config"] = {"workload": line["config"]["workload"][:200], "scheme": scheme}
    assert len(json.dumps(line)) < MAX_LINE_BYTES, "headline line too long"
    return line


def run_ours(args):
    import torch
    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback "
                         "(use --impl reference for the oracle)")
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch with torchrun --nproc-per-node "
                         f"{args.gpus} (or without a launcher: bench.py starts the replicas itself)")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        if dist is not None:
            dist.barrier()

    import paper_1709_06483_b200 as M     # raises if the CUDA library is missing
    import workloads as W
    M.lib()
    cfg = W.CONFIGS[args.workload]
    scheme = args.scheme or cfg.schemes[0]
    peaks = load_peaks()
    dmma_tf, dfma_tf = M.magnus_fp64_peaks()

    sampler = ClockSampler(local_rank) if rank == 0 else None
    res = measure_workload(M, W, torch, cfg, scheme, args.steps, args.warmup, dev, barrier, sampler)
    value, sec = whole_job_value(args.steps, res["seconds"], dist, dev)
    st = res["stats"]

    e2e = None
    if not args.no_e2e:
        e2e = measure_e2e(M, torch, cfg, scheme, args.steps, res["inputs"])
        e2e["value"], e2e["seconds"] = whole_job_value(args.steps, e2e["seconds"], dist, dev)
    res["inputs"] = None
    torch.cuda.empty_cache()

    if rank == 0:
        roof = roofline_for(cfg, scheme, st, peaks, dmma_tf, res.get("path"))
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            base = time_oracle(cfg, scheme, 1, 0, args.oracle_max_size)
            cpu = {k: base[k] for k in ("value", "unit", "cores", "kind", "sample")}
        if args.extra:      # opt-in secondary runs: to a side file, never into the headline line
            with open(args.extra, "w") as fh:
                json.dump(measure_extra(M, W, torch, dev, peaks, dmma_tf), fh, indent=1)
        line = build_line(cfg, scheme, world, args.steps, args.warmup, value, sec, st, res["norm"], res["clocks"], roof,
                          e2e, (dmma_tf, dfma_tf), cpu)
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def run_sweep(args):
    """The paper's sweeps (bench_sweeps.py, beside this file: a measurement harness, not part of the package) with the oracle timed beside the sizes it affords."""
    import bench_sweeps as sweeps
    from oracle import oracle as O

    def cpu_timer(example, N, H0, H1, psi0, f, tau, tol):
        o0 = H0.cpu().numpy() if example == 1 else O.CsrHost.of(H0)
        o1 = H1.cpu().numpy() if example == 1 else O.CsrHost.of(H1)
        if N <= 10:   # untimed first call: the OpenMP team starts up
            O.magnus_step(o0, o1, f, "cf4", 0.0, tau, psi0.cpu().numpy(), tol)
        t0 = time.perf_counter()
        O.magnus_step(o0, o1, f, "cf4", 0.0, tau, psi0.cpu().numpy(), tol)
        return time.perf_counter() - t0

    cmd = f"python bench.py --sweep {args.sweep}{' --sweep-quick' if args.sweep_quick else ''}"
    lines = sweeps.run_all(args.sweep, cpu_timer, args.sweep_quick, cmd + f" (oracle: {O.num_threads()} host threads)")
    print("\n".join(lines))


def matrix_bytes_cfg(cfg):
    if cfg.kind == "xxz":
        return 20 * (1 << cfg.size) * (3 * cfg.size + 2) // 2
    return 2 * 16 * cfg.size * cfg.size


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", default="cfg5", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--scheme", default=None, choices=["cf4", "m4", "m2", "cf4:3", "m6"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="accepted for compatibility: extras are opt-in now (--extra)")
    ap.add_argument("--extra", default=None, metavar="FILE.json",
                    help="also run the secondary measurements (cfg1-cfg4, shortcuts) and write them to FILE.json")
    ap.add_argument("--sweep", default=None, metavar="FILE.md",
                    help="instead of the benchmark line: re-run the paper's cost-vs-size and accuracy-vs-cost sweeps "
                         "(PAPER.md section 4) and write the tables to FILE.md")
    ap.add_argument("--sweep-quick", action="store_true")
    ap.add_argument("--oracle-steps", type=int, default=None,
                    help="reference arm: Magnus steps of the oracle to time (default 1: a step is tens of seconds)")
    ap.add_argument("--oracle-max-size", type=int, default=None,
                    help="cap N (xxz) or n (dense) of the oracle's bounded sample")
    args = ap.parse_args()
    if args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
            raise SystemExit(respawn_under_torchrun(args))
        if args.warmup < 3:
            sys.stderr.write("bench.py: note: fewer than 3 warm-up steps\n")
        run_ours(args)


if __name__ == "__main__":
    main()
