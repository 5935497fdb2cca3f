"""The five BASELINE.json configs as data (sizes, schemes, time grid).

Workload description only; nothing of the method is computed here.
`magnus_integrate(t0, t_end, nsteps)` arguments follow SURVEY.md section 8(b):
"T=1, 100 steps" -> (0, 1, 100); "10 steps, h=0.1" -> (0, 1.0, 10);
"5 steps, h=0.05" -> (0, 0.25, 5).
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Callable, Tuple

from . import dense, rng, xxz


@dataclass(frozen=True)
class Config:
    name: str
    kind: str                 # "xxz" (CSR) or "dense"
    size: int                 # N spins (xxz) or n (dense)
    schemes: Tuple[str, ...]  # subset of ("cf4", "m4")
    t0: float
    t_end: float
    nsteps: int
    tol: float
    psi0: str                 # "neel" or "random"

    @property
    def n(self) -> int:
        return (1 << self.size) if self.kind == "xxz" else self.size

    @property
    def tau(self) -> float:
        return (self.t_end - self.t0) / self.nsteps

    @property
    def f(self) -> Callable[[float], float]:
        return xxz.f_cos2t if self.kind == "xxz" else dense.f_sin3t


CONFIGS = {
    "cfg1": Config("cfg1", "xxz", 10, ("cf4", "m4"), 0.0, 1.0, 100, 1e-12, "neel"),
    "cfg2": Config("cfg2", "dense", 2048, ("cf4", "m4"), 0.0, 1.0, 50, 1e-12, "random"),
    "cfg3": Config("cfg3", "xxz", 20, ("cf4", "m4"), 0.0, 1.0, 20, 1e-12, "random"),
    "cfg4": Config("cfg4", "dense", 16384, ("cf4", "m4"), 0.0, 1.0, 10, 1e-12, "random"),
    "cfg5": Config("cfg5", "xxz", 24, ("cf4",), 0.0, 0.25, 5, 1e-12, "random"),
}


def scaled(cfg: Config, size: int, nsteps: int | None = None) -> Config:
    """Same recipe at another size (and step count, keeping tau) for parity tests."""
    ns = cfg.nsteps if nsteps is None else nsteps
    return Config(f"{cfg.name}@{size}", cfg.kind, size, cfg.schemes, cfg.t0,
                  cfg.t0 + cfg.tau * ns, ns, cfg.tol, cfg.psi0)


def build(cfg: Config, device="cpu"):
    """Return (H0, H1, psi0, f).  H0/H1 are xxz.CSR or dense complex128 tensors."""
    if cfg.kind == "xxz":
        H0 = xxz.xxz_h0(cfg.size, device=device)
        H1 = xxz.xxz_h1(cfg.size, device=device)
    else:
        H0 = dense.dense_h0(cfg.size, device=device)
        H1 = dense.dense_h1(cfg.size, device=device)
    if cfg.psi0 == "neel":
        psi0 = xxz.neel_state(cfg.size, device=device)
    else:
        psi0 = rng.random_unit_vector(cfg.n, device=device)
    return H0, H1, psi0, cfg.f
