"""Counter-based random numbers for the synthetic workloads.

Holds NO arithmetic of the method (arXiv 1709.06483): it only turns
(seed, stream, index) into reproducible normal variates.  Both the oracle
tests and the CUDA path receive the arrays produced here; neither generates
its own inputs.

Recipe: splitmix64 hash of (seed, stream, index) ->
two uniforms in (0,1) -> Box-Muller.  Everything is written with torch ops on
int64 (two's-complement wrap-around == uint64 arithmetic) so the same code
runs on the CPU or on a CUDA device.  The integer hash is bit-identical on
every device; the float64 log/cos/sin of Box-Muller may differ in the last
ulp between devices, so a test generates its inputs ONCE and hands the same
bits to both sides.
"""
from __future__ import annotations

import math

import torch

SEED = 170906483  # the arXiv number of the paper, used for every config


def _s64(x: int) -> int:
    """Interpret an unsigned 64-bit constant as a signed int64."""
    x &= (1 << 64) - 1
    return x - (1 << 64) if x >= (1 << 63) else x


_GOLDEN = _s64(0x9E3779B97F4A7C15)
_M1 = _s64(0xBF58476D1CE4E5B9)
_M2 = _s64(0x94D049BB133111EB)


def _lsr(x: torch.Tensor, k: int) -> torch.Tensor:
    """Logical shift right on int64 (torch's >> is arithmetic)."""
    return (x >> k) & ((1 << (64 - k)) - 1)


def splitmix64(z: torch.Tensor) -> torch.Tensor:
    """The splitmix64 finaliser, elementwise on an int64 tensor."""
    z = z + _GOLDEN
    z = (z ^ _lsr(z, 30)) * _M1
    z = (z ^ _lsr(z, 27)) * _M2
    return z ^ _lsr(z, 31)


def _splitmix64_int(z: int) -> int:
    mask = (1 << 64) - 1
    z = (z + 0x9E3779B97F4A7C15) & mask
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & mask
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & mask
    return z ^ (z >> 31)


def stream_key(seed: int, stream: int) -> int:
    """Scalar key of a (seed, stream) pair, as a signed int64."""
    return _s64(_splitmix64_int((seed & ((1 << 64) - 1)) ^ _splitmix64_int(stream)))


def uniform_pair(seed: int, stream: int, index: torch.Tensor):
    """Two uniforms in (0,1) for every int64 counter in `index`."""
    key = stream_key(seed, stream)
    a = splitmix64(index * 2 + key)
    b = splitmix64(index * 2 + 1 + key)
    scale = 2.0 ** -53
    u1 = (_lsr(a, 11).to(torch.float64) + 0.5) * scale
    u2 = (_lsr(b, 11).to(torch.float64) + 0.5) * scale
    return u1, u2


def normal_pair(seed: int, stream: int, index: torch.Tensor):
    """Two independent N(0,1) variates per counter (Box-Muller)."""
    u1, u2 = uniform_pair(seed, stream, index)
    r = torch.sqrt(-2.0 * torch.log(u1))
    ang = (2.0 * math.pi) * u2
    return r * torch.cos(ang), r * torch.sin(ang)


def complex_normal(seed: int, stream: int, index: torch.Tensor, var: float = 1.0) -> torch.Tensor:
    """x + iy with x, y ~ N(0, var/2), so that E|z|^2 = var."""
    x, y = normal_pair(seed, stream, index)
    s = math.sqrt(var / 2.0)
    return torch.complex(x * s, y * s)


def random_unit_vector(n: int, seed: int = SEED, stream: int = 7, device="cpu") -> torch.Tensor:
    """psi0 for the 'random normalised complex vector' configs (complex128)."""
    idx = torch.arange(n, dtype=torch.int64, device=device)
    z = complex_normal(seed, stream, idx)
    return z / torch.linalg.vector_norm(z)
