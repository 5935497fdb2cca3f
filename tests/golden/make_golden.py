"""Writes tests/golden/cfg1_oracle.json.  Calls ONLY oracle/ and workloads/.

No value here comes from the paper (it prints no iteration counts or state
vectors: SURVEY.md section 4) and none from the CUDA path.  The file records
what the oracle produced for CFG1 so that a later edit of the oracle that
changes its behaviour is noticed; it is a regression record, not a pin.

    python tests/golden/make_golden.py
"""
import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import workloads as W  # noqa: E402
from oracle import oracle as O  # noqa: E402


def main():
    cfg = W.CONFIGS["cfg1"]
    H0, H1, psi0, f = W.build(cfg)
    H0, H1 = O.CsrHost.of(H0), O.CsrHost.of(H1)
    out = {"source": "oracle/magnus_oracle.cpp via tests/golden/make_golden.py", "config": "cfg1"}
    for scheme in cfg.schemes:
        psi, iters = O.magnus_integrate(H0, H1, f, scheme, cfg.t0, cfg.t_end, cfg.nsteps, psi0.numpy(), cfg.tol)
        out[scheme] = {
            "total_matvecs": int(iters.sum()),
            "iters_first8": [int(x) for x in iters[:8]],
            "norm": float(np.linalg.norm(psi)),
            "psi_neel_component": [float(psi[341].real), float(psi[341].imag)],
        }
    with open(os.path.join(HERE, "cfg1_oracle.json"), "w") as fh:
        json.dump(out, fh, indent=1)
    print(json.dumps(out, indent=1))


if __name__ == "__main__":
    main()
