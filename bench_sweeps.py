"""The paper's own sweeps re-run on B200: `python bench_sweeps.py --out FILE.md`.

  * cost against problem size at tau = 1e-3 for Example 1 (non-local Heisenberg, stored dense, Figs. 2-3)
    and Example 2 (local Heisenberg, CSR, Figs. 5-6), for M2, M4, M6, Cf4, Cf4:3;
  * accuracy against cost at N = 2^12 for both examples (Figs. 4 and 8): error of every scheme
    against M6 with a small step, as in the paper, and the time of the run.

Timings are CUDA-event seconds of `magnus_integrate` (inputs resident, one warm-up run); the paper's figure data is
not available, so this is a re-run, not a comparison.  `bench.py --sweep FILE.md` runs the same sweeps with the CPU
oracle (test infrastructure, which this file never imports) timed beside the sizes it affords, through the
`cpu_timer` callback.  Marshalling only: every number comes from the C-ABI library.
"""
from __future__ import annotations

import argparse
import math
import os
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

SCHEMES = ["m2", "m4", "m6", "cf4", "cf4:3"]


def _inputs(example: int, nspins: int, dev):
    from workloads import paper_examples as pe
    if example == 1:
        H0, H1 = pe.example1_dense(nspins, device=dev)
    else:
        H0, H1 = pe.example2_csr(nspins, device=dev)
    return H0, H1, pe.initial_value(nspins, device=dev), pe.f_sin_t


def _run(M, H0, H1, f, scheme, psi0, t_end, nsteps, tol):
    psi = psi0.clone()
    with M.magnus_create(H0, H1, f, scheme, tol=tol) as h:
        warm = psi0.clone()
        h.integrate(0.0, t_end * min(3, nsteps) / nsteps, min(3, nsteps), warm)
        st = h.integrate(0.0, t_end, nsteps, psi)
    return psi, st


def cost_vs_size(M, torch, example, sizes, nsteps, tau, tol, cpu_timer, lines):
    dev = "cuda"
    lines.append(f"\n### Example {example}: seconds per step at tau = {tau:g} ({nsteps} timed steps), {'dense' if example == 1 else 'CSR'}\n")
    lines.append("| n = 2^N | " + " | ".join(SCHEMES) + " | mat-vecs/step (Cf4) |" + (" CPU oracle Cf4 s/step |" if cpu_timer else ""))
    lines.append("|---|" + "---|" * (len(SCHEMES) + 1 + (1 if cpu_timer else 0)))
    for N in sizes:
        H0, H1, psi0, f = _inputs(example, N, dev)
        row, mv = [], None
        for scheme in SCHEMES:
            if scheme == "m6" and example == 2 and (1 << N) > 16384:
                row.append("n/a")
                continue
            try:
                _, st = _run(M, H0, H1, f, scheme, psi0, nsteps * tau, nsteps, tol)
                row.append(f"{st['seconds_device'] / nsteps:.3e}")
                if scheme == "cf4":
                    mv = st["total_matvecs"] / nsteps
            except M.MagnusError as e:
                row.append(f"error {e.code}")
        extra = ""
        if cpu_timer:
            sec = cpu_timer(example, N, H0, H1, psi0, f, tau, tol)
            extra = f" {sec:.3e} |" if sec is not None else " - |"
        lines.append(f"| {N} | " + " | ".join(row) + f" | {mv:.1f} |" + extra)
        del H0, H1
        torch.cuda.empty_cache()


def accuracy_vs_cost(M, torch, example, N, t_end, steps_list, ref_steps, tol, lines):
    dev = "cuda"
    H0, H1, psi0, f = _inputs(example, N, dev)
    ref, _ = _run(M, H0, H1, f, "m6", psi0, t_end, ref_steps, tol)
    lines.append(f"\n### Example {example}, n = 2^{N}: error at T = {t_end:g} against M6 with {ref_steps} steps, and seconds of the run\n")
    lines.append("| steps (tau) | " + " | ".join(f"{s}: error / s" for s in SCHEMES) + " |")
    lines.append("|---|" + "---|" * len(SCHEMES))
    for ns in steps_list:
        row = []
        for scheme in SCHEMES:
            psi, st = _run(M, H0, H1, f, scheme, psi0, t_end, ns, tol)
            err = float(torch.linalg.vector_norm(psi - ref))
            row.append(f"{err:.2e} / {st['seconds_device']:.3f}")
        lines.append(f"| {ns} ({t_end / ns:.4g}) | " + " | ".join(row) + " |")


def run_all(out_path, cpu_timer=None, quick=False, command=""):
    import torch
    import paper_1709_06483_b200 as M
    if not torch.cuda.is_available():
        raise SystemExit("sweeps: no CUDA device (the library has no CPU fallback)")
    M.lib()
    lines = ["# The paper's sweeps re-run on one B200", "",
             f"Command: `{command}`; device: {torch.cuda.get_device_name(0)}; Leja tolerance 1e-10 (P:229-231); every "
             "GPU entry is the CUDA-event time of `magnus_integrate` with inputs resident in HBM, after a warm-up run."]
    tol = 1e-10
    s1 = range(6, 9) if quick else range(6, 14)
    s2 = range(6, 9) if quick else range(6, 15)
    cost_vs_size(M, torch, 1, s1, 20, 1e-3, tol, cpu_timer, lines)
    cost_vs_size(M, torch, 2, s2, 20, 1e-3, tol, cpu_timer, lines)
    Nacc = 8 if quick else 12
    accuracy_vs_cost(M, torch, 1, Nacc, 1.0, [8, 16, 32, 64], 128 if quick else 512, tol / 10, lines)
    accuracy_vs_cost(M, torch, 2, Nacc, 1.0, [8, 16, 32, 64], 128 if quick else 512, tol / 10, lines)
    with open(out_path, "w") as fh:
        fh.write("\n".join(lines) + "\n")
    return lines


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--out", required=True)
    ap.add_argument("--quick", action="store_true", help="small sizes only (a few seconds)")
    args = ap.parse_args()
    cmd = f"python bench_sweeps.py --out {args.out}{' --quick' if args.quick else ''}"
    print("\n".join(run_all(args.out, None, args.quick, cmd)))


if __name__ == "__main__":
    main()
