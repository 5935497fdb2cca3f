"""The paper's own two workloads (section 4), as generators only.

Workload description: no arithmetic of the Magnus/Leja method lives here.

Example 1 ("dense matrix case", non-local Heisenberg model):
    H(t) = - sum_{i != j} J_ij sz_i sz_j - h(t) sum_i sx_i,   J_ij = 1/|i-j|,  h(t) = sin(t)
    H0 = - sum_{i != j} J_ij sz_i sz_j   (diagonal),   H1 = - sum_i sx_i;   stored DENSE as in the paper.
Example 2 ("sparse matrix case", local Heisenberg model):
    H(t) = -1/2 sum_j (Jx sx_j sx_{j+1} + Jy sy_j sy_{j+1} + Jz sz_j sz_{j+1} + h(t) sz_j),
    Jx, Jy, Jz = 1, 2, 3,  h(t) = sin(t);   H0 = the three couplings, H1 = -1/2 sum_j sz_j (diagonal);  CSR.
    Reading (the paper leaves sigma_{n+1} undefined): periodic, sigma_{n+1} = sigma_1, n bonds.  Because
    Jx != Jy every bond contributes one off-diagonal entry to every row (amplitude -(Jx+Jy)/2 on an
    antiparallel pair, -(Jx-Jy)/2 on a parallel pair): exactly n + 1 stored entries per row.
Initial value, eq. (13) (garbled in the source): spin 1 up, spin 2 down, the remaining
spins in a seeded random state, normalised.  Conventions as in workloads/xxz.py: site 1 is the most
significant bit, bit 0 <-> sz = +1.
"""
from __future__ import annotations

import math

import torch

from . import rng
from .xxz import CSR, bond_masks


def f_sin_t(t: float) -> float:
    """h(t) = sin(omega t), omega = 1 (both examples)."""
    return math.sin(t)


def _sz(r: torch.Tensor, bit: int) -> torch.Tensor:
    """Eigenvalue of sz on the spin stored in `bit` for basis states r: +1 for bit 0, -1 for bit 1."""
    return 1.0 - 2.0 * ((r >> bit) & 1).to(torch.float64)


def example1_dense(n: int, device="cpu"):
    """(H0, H1) of Example 1 as dense complex128 2^n x 2^n tensors."""
    N = 1 << n
    r = torch.arange(N, dtype=torch.int64, device=device)
    diag = torch.zeros(N, dtype=torch.float64, device=device)
    for i in range(1, n + 1):
        for j in range(1, n + 1):
            if i != j:
                diag -= (1.0 / abs(i - j)) * _sz(r, n - i) * _sz(r, n - j)
    H0 = torch.zeros((N, N), dtype=torch.complex128, device=device)
    H0[r, r] = torch.complex(diag, torch.zeros_like(diag))
    H1 = torch.zeros((N, N), dtype=torch.complex128, device=device)
    for b in range(n):
        H1[r, r ^ (1 << b)] = -1.0
    return H0, H1


def example2_csr(n: int, jx: float = 1.0, jy: float = 2.0, jz: float = 3.0, device="cpu"):
    """(H0, H1) of Example 2 as CSR; n + 1 stored entries per row of H0, the diagonal alone in H1."""
    N = 1 << n
    r = torch.arange(N, dtype=torch.int64, device=device)
    masks = bond_masks(n)
    cols = [r]
    diag = torch.zeros(N, dtype=torch.float64, device=device)
    vals = []
    for m in masks:
        hi, lo = m.bit_length() - 1, (m & -m).bit_length() - 1
        szz = _sz(r, hi) * _sz(r, lo)                       # +1 parallel, -1 antiparallel
        diag -= 0.5 * jz * szz
        # sx sx flips both spins with +1; sy sy flips both with -1 (parallel) or +1 (antiparallel)
        vals.append(-0.5 * (jx - jy * szz))
        cols.append(r ^ m)
    cols = torch.stack(cols, dim=1)                          # [N, n+1]
    vals = torch.stack([diag] + vals, dim=1)
    cols, order = torch.sort(cols, dim=1)
    vals = torch.gather(vals, 1, order)
    row_ptr = (torch.arange(N + 1, dtype=torch.int64, device=device) * (n + 1)).to(torch.int32)
    H0 = CSR(N, row_ptr, cols.reshape(-1).to(torch.int32),
             torch.complex(vals.reshape(-1), torch.zeros(N * (n + 1), dtype=torch.float64, device=device)))
    d1 = torch.zeros(N, dtype=torch.float64, device=device)
    for b in range(n):
        d1 -= 0.5 * _sz(r, b)
    H1 = CSR(N, torch.arange(N + 1, dtype=torch.int32, device=device), r.to(torch.int32),
             torch.complex(d1, torch.zeros_like(d1)))
    return H0, H1


def initial_value(n: int, device="cpu") -> torch.Tensor:
    """Reading of eq. (13): spin 1 up (bit n-1 = 0), spin 2 down (bit n-2 = 1), the rest random; unit norm."""
    if n < 3:
        raise ValueError("needs n >= 3 spins")
    rest = rng.random_unit_vector(1 << (n - 2), stream=13, device=device)
    psi = torch.zeros(1 << n, dtype=torch.complex128, device=device)
    base = 1 << (n - 2)                                      # prefix bits (0, 1)
    psi[base:2 * base] = rest
    return psi
