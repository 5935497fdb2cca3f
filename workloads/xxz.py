"""Periodic XXZ Heisenberg chain in a transverse field, as CSR complex128.

Workload generator only: no arithmetic of the Magnus/Leja method lives here.

BASELINE.json configs 1, 3, 5:
    H(t) = sum_i (sx_i sx_{i+1} + sy_i sy_{i+1} + 0.5 sz_i sz_{i+1}) + cos(2t) sum_i sx_i
so  H0 = sum over the N periodic bonds, H1 = sum_i sx_i, f(t) = cos(2t).

Conventions (eq. (11)-(12), reading g2 of SURVEY.md section 8(c)):
site 1 is the MOST significant bit of the basis index, bit 0 <-> (1,0)^T <->
sz = +1.  Site j sits on bit N-j.  The bonds are (bit b, bit b-1) for
b = N-1..1 plus the periodic bond (bit 0, bit N-1).

Structure: on a bond, sx sx + sy sy flips an
antiparallel pair with amplitude 2 and kills a parallel pair; 0.5 sz sz is
+0.5 (parallel) or -0.5 (antiparallel).  Row r of H0 therefore holds the
diagonal 0.5*(N - 2k) (k = number of antiparallel bonds, ALWAYS stored, even
when it is 0) and k entries 2.0 at r ^ (pair mask).  Row r of H1 holds N
entries 1.0 at r ^ (1 << b); it has no diagonal.  Stored entries:
nnz(H0) = 2^N (N/2 + 1), nnz(H1) = 2^N N, together 2^N (1.5 N + 1).

All index work is integer torch ops, so the result is bit-identical on CPU
and CUDA devices.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import torch


@dataclass
class CSR:
    n: int
    row_ptr: torch.Tensor  # int32 [n+1]
    col_idx: torch.Tensor  # int32 [nnz], ascending within a row
    values: torch.Tensor   # complex128 [nnz]

    @property
    def nnz(self) -> int:
        return int(self.col_idx.numel())

    def to(self, device) -> "CSR":
        return CSR(self.n, self.row_ptr.to(device), self.col_idx.to(device), self.values.to(device))

    def to_scipy(self):
        import scipy.sparse as sp
        return sp.csr_matrix(
            (self.values.cpu().numpy(), self.col_idx.cpu().numpy(), self.row_ptr.cpu().numpy()),
            shape=(self.n, self.n))


def bond_masks(N: int):
    """XOR masks of the N periodic nearest-neighbour bonds."""
    if N < 3:
        raise ValueError("periodic chain needs N >= 3 (N = 2 would double count its bond)")
    return [(1 << b) | (1 << (b - 1)) for b in range(N - 1, 0, -1)] + [(1 << (N - 1)) | 1]


def _rows_h0(r: torch.Tensor, N: int):
    """Candidate columns/values of H0 for the row block r (int64 [R])."""
    n = 1 << N
    masks = torch.tensor(bond_masks(N), dtype=torch.int64, device=r.device)      # [N]
    hi = torch.tensor([m.bit_length() - 1 for m in bond_masks(N)], dtype=torch.int64, device=r.device)
    lo = torch.tensor([(m & -m).bit_length() - 1 for m in bond_masks(N)], dtype=torch.int64, device=r.device)
    bit_hi = (r[:, None] >> hi[None, :]) & 1
    bit_lo = (r[:, None] >> lo[None, :]) & 1
    anti = bit_hi != bit_lo                                                      # [R, N]
    k = anti.sum(dim=1)                                                          # antiparallel bonds
    cols = torch.where(anti, r[:, None] ^ masks[None, :], torch.full_like(anti, n, dtype=torch.int64))
    cols = torch.cat([r[:, None], cols], dim=1)                                  # diagonal first
    vals = torch.full(cols.shape, 2.0, dtype=torch.float64, device=r.device)
    vals[:, 0] = 0.5 * (N - 2 * k).to(torch.float64)
    return cols, vals


def _rows_h1(r: torch.Tensor, N: int):
    n = 1 << N
    bits = torch.arange(N, dtype=torch.int64, device=r.device)
    cols = r[:, None] ^ (torch.ones_like(bits) << bits)[None, :]
    vals = torch.ones(cols.shape, dtype=torch.float64, device=r.device)
    return cols, vals


def _assemble(N: int, rows_fn, device, block_rows: int) -> CSR:
    n = 1 << N
    col_parts, val_parts, cnt_parts = [], [], []
    for r0 in range(0, n, block_rows):
        r = torch.arange(r0, min(n, r0 + block_rows), dtype=torch.int64, device=device)
        cols, vals = rows_fn(r, N)
        cols, order = torch.sort(cols, dim=1)            # invalid entries carry column n -> go last
        vals = torch.gather(vals, 1, order)
        keep = cols < n
        cnt_parts.append(keep.sum(dim=1))
        col_parts.append(cols[keep].to(torch.int32))
        val_parts.append(vals[keep])
    counts = torch.cat(cnt_parts)
    row_ptr = torch.zeros(n + 1, dtype=torch.int64, device=device)
    row_ptr[1:] = torch.cumsum(counts, dim=0)
    if int(row_ptr[-1]) >= 2 ** 31:
        raise ValueError("nnz does not fit int32 row pointers")
    re = torch.cat(val_parts)
    values = torch.complex(re, torch.zeros_like(re))
    return CSR(n, row_ptr.to(torch.int32), torch.cat(col_parts), values)


def xxz_h0(N: int, device="cpu", block_rows: int = 1 << 18) -> CSR:
    return _assemble(N, _rows_h0, device, block_rows)


def xxz_h1(N: int, device="cpu", block_rows: int = 1 << 18) -> CSR:
    return _assemble(N, _rows_h1, device, block_rows)


def xxz_nnz(N: int):
    """Exact stored-entry counts (nnz(H0), nnz(H1)); sum = 2^N (1.5N + 1)."""
    n = 1 << N
    return n + (n * N) // 2, n * N


def neel_index(N: int) -> int:
    """Site 1 up (bit 0 at the MSB), alternating: 0b0101...01 (341 for N=10)."""
    idx = 0
    for j in range(1, N + 1):          # site j on bit N-j; even sites are down (bit = 1)
        if j % 2 == 0:
            idx |= 1 << (N - j)
    return idx


def neel_state(N: int, device="cpu") -> torch.Tensor:
    psi = torch.zeros(1 << N, dtype=torch.complex128, device=device)
    psi[neel_index(N)] = 1.0
    return psi


def f_cos2t(t: float) -> float:
    """The driving of configs 1, 3, 5: f(t) = cos(2t)."""
    return math.cos(2.0 * t)
