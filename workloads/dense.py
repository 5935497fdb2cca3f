"""Random dense Hermitian Hamiltonians (BASELINE.json configs 2 and 4).

Workload generator only: no arithmetic of the Magnus/Leja method lives here.

Reading g10 of SURVEY.md section 8(c): G_ij = x + iy with x, y ~ N(0, 1/2)
(E|G_ij|^2 = 1), H = (G + G^H) / sqrt(2n), so E|H_ij|^2 = 1/n off the diagonal
and the spectrum fills the semicircle [-2, 2].  H(t) = H0 + sin(3t) H1 with
H0 and H1 drawn from two different streams of the same seed.  Storage is
row-major (C-contiguous) complex128.
"""
from __future__ import annotations

import math

import torch

from .rng import SEED, complex_normal


def random_hermitian(n: int, stream: int, seed: int = SEED, device="cpu", block_rows: int = 1024) -> torch.Tensor:
    G = torch.empty((n, n), dtype=torch.complex128, device=device)
    for r0 in range(0, n, block_rows):
        r1 = min(n, r0 + block_rows)
        idx = torch.arange(r0 * n, r1 * n, dtype=torch.int64, device=device)
        G[r0:r1] = complex_normal(seed, stream, idx).view(r1 - r0, n)
    scale = 1.0 / math.sqrt(2.0 * n)
    # H = (G + G^H) * scale, built block-wise in place of a full transposed temporary.
    H = torch.empty_like(G)
    for r0 in range(0, n, block_rows):
        r1 = min(n, r0 + block_rows)
        H[r0:r1] = (G[r0:r1] + G[:, r0:r1].conj().transpose(0, 1)) * scale
    return H


def dense_h0(n: int, device="cpu") -> torch.Tensor:
    return random_hermitian(n, stream=1, device=device)


def dense_h1(n: int, device="cpu") -> torch.Tensor:
    return random_hermitian(n, stream=2, device=device)


def f_sin3t(t: float) -> float:
    """The driving of configs 2 and 4: f(t) = sin(3t)."""
    return math.sin(3.0 * t)
