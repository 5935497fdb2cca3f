"""Writes tests/golden/<cfg>_<scheme>_full.json: the oracle's WHOLE integration of a BASELINE config (all K steps).

Calls ONLY oracle/ and workloads/ -- no value comes from the CUDA path, and none from the paper (it prints no
iteration counts or state vectors).  A file is what the oracle (pinned in tests/test_oracle_*.py)
produced; the -m gpu tests in tests/test_gpu_fullsize.py run the same K steps through the C-ABI and compare
  * every per-exponential iteration count                      exactly,
  * every snapped interval (a, b) and theta                    bit for bit (stored as float.hex()),
  * psi_K at NSAMPLE seeded indices, element by element        to 1e-9 * ||psi_K||  (north_star's bar),
  * ||psi_K||.
The steps are taken one by one with t_n = t0 + n * tau, tau = (t_end - t0) / K -- the loop of
oracle_magnus_integrate_* written out here so that the per-exponential info can be recorded.

    python tests/golden/make_golden_full.py cfg3:cf4 cfg3:m4 cfg5:cf4 cfg2:m4 cfg4:cf4

Wall time on the 8-core build container is recorded in each file's header.
"""
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import workloads as W  # noqa: E402
from oracle import oracle as O  # noqa: E402

NSAMPLE = 1024
SAMPLE_SEED = 170906483


def sample_indices(n: int) -> np.ndarray:
    """NSAMPLE distinct seeded indices (all of them when n <= NSAMPLE), ascending."""
    if n <= NSAMPLE:
        return np.arange(n, dtype=np.int64)
    r = np.random.default_rng(SAMPLE_SEED)
    return np.sort(r.choice(n, size=NSAMPLE, replace=False)).astype(np.int64)


def run(name: str, scheme: str) -> dict:
    cfg = W.CONFIGS[name]
    H0, H1, psi0, f = W.build(cfg)
    if cfg.kind == "xxz":
        H0, H1 = O.CsrHost.of(H0), O.CsrHost.of(H1)
    else:
        H0, H1 = H0.numpy(), H1.numpy()
    psi = psi0.numpy()
    tau = (cfg.t_end - cfg.t0) / cfg.nsteps
    iters, a, b, theta, substeps = [], [], [], [], []
    t_start = time.perf_counter()
    for s in range(cfg.nsteps):
        psi, infos = O.magnus_step(H0, H1, f, scheme, cfg.t0 + s * tau, tau, psi, cfg.tol)
        for i in infos:
            iters.append(int(i["iters"]))
            substeps.append(int(i["substeps"]))
            a.append(float(i["a"]).hex())
            b.append(float(i["b"]).hex())
            theta.append(float(i["theta"]).hex())
        print(f"{name} {scheme}: step {s + 1}/{cfg.nsteps}  {time.perf_counter() - t_start:.1f} s", flush=True)
    wall = time.perf_counter() - t_start
    idx = sample_indices(cfg.n)
    return {
        "source": "oracle/magnus_oracle.cpp via tests/golden/make_golden_full.py (oracle + workloads only)",
        "command": f"python tests/golden/make_golden_full.py {name}:{scheme}",
        "wall_seconds": round(wall, 1), "host_threads": O.num_threads(),
        "config": name, "scheme": scheme, "n": cfg.n, "nsteps": cfg.nsteps, "t0": cfg.t0, "t_end": cfg.t_end,
        "tol": cfg.tol, "iters": iters, "substeps": substeps, "a_hex": a, "b_hex": b, "theta_hex": theta,
        "norm": float(np.linalg.norm(psi)),
        "sample_seed": SAMPLE_SEED, "sample_index": [int(i) for i in idx],
        "sample_re": [float(x) for x in psi[idx].real], "sample_im": [float(x) for x in psi[idx].imag],
    }


def main():
    for spec in sys.argv[1:]:
        name, scheme = spec.split(":")
        out = run(name, scheme)
        path = os.path.join(HERE, f"{name}_{scheme}_full.json")
        with open(path, "w") as fh:
            json.dump(out, fh)
        print("wrote", path, "total matvecs", sum(out["iters"]), "wall", out["wall_seconds"], "s", flush=True)


if __name__ == "__main__":
    main()
