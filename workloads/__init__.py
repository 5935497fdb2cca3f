"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This package holds none of the method's arithmetic (no Leja points, no
divided differences, no mat-vec, no scheme coefficients): only the
formula-defined Hamiltonians, initial states and driving functions of
BASELINE.json's five configs.  It imports neither `oracle` nor
`paper_1709_06483_b200`.
"""
from . import configs, dense, paper_examples, rng, xxz  # noqa: F401
from .configs import CONFIGS, Config, build, scaled  # noqa: F401
from .rng import SEED  # noqa: F401
