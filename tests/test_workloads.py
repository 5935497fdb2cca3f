"""Pins for the synthetic input generators (SURVEY.md 8(c) pin c-P12, readings g2, g3, g10, g11).

The generators hold none of the method's arithmetic; they are checked against
the textbook Kronecker-product definition of the spin operators (PAPER.md
eqs. (11)-(12), lines 241-248) and against closed-form counts.
"""
import math

import numpy as np
import pytest
import torch

import workloads as W
from workloads import dense, rng, xxz

SX = np.array([[0, 1], [1, 0]], dtype=complex)
SY = np.array([[0, -1j], [1j, 0]], dtype=complex)
SZ = np.array([[1, 0], [0, -1]], dtype=complex)
I2 = np.eye(2, dtype=complex)


def site_op(op, j, N):
    """sigma_j^alpha = I^(j-1) (x) op (x) I^(N-j), site 1 leftmost (eq. (12))."""
    out = np.array([[1.0 + 0j]])
    for s in range(1, N + 1):
        out = np.kron(out, op if s == j else I2)
    return out


def kron_xxz(N):
    H0 = np.zeros((1 << N, 1 << N), dtype=complex)
    H1 = np.zeros_like(H0)
    for j in range(1, N + 1):
        k = j % N + 1                       # periodic neighbour
        H0 += site_op(SX, j, N) @ site_op(SX, k, N) + site_op(SY, j, N) @ site_op(SY, k, N) \
            + 0.5 * site_op(SZ, j, N) @ site_op(SZ, k, N)
        H1 += site_op(SX, j, N)
    return H0, H1


@pytest.mark.parametrize("N", [3, 4, 5, 6])
def test_xxz_matches_kronecker_definition(N):
    H0k, H1k = kron_xxz(N)
    H0 = xxz.xxz_h0(N).to_scipy().toarray()
    H1 = xxz.xxz_h1(N).to_scipy().toarray()
    assert np.array_equal(H0, H0k)
    assert np.array_equal(H1, H1k)


@pytest.mark.parametrize("N", [4, 7, 10, 12])
def test_xxz_structure_and_counts(N):
    H0, H1 = xxz.xxz_h0(N), xxz.xxz_h1(N)
    n = 1 << N
    nnz0, nnz1 = xxz.xxz_nnz(N)
    assert H0.nnz == nnz0 == n + n * N // 2
    assert H1.nnz == nnz1 == n * N
    assert nnz0 + nnz1 == int(n * (1.5 * N + 1))
    for H in (H0, H1):
        assert H.row_ptr.dtype == torch.int32 and H.col_idx.dtype == torch.int32
        assert H.values.dtype == torch.complex128
        rp, ci = H.row_ptr.numpy(), H.col_idx.numpy()
        assert rp[0] == 0 and rp[-1] == H.nnz
        for r in range(0, n, max(1, n // 64)):
            row = ci[rp[r]:rp[r + 1]]
            assert np.all(np.diff(row) > 0)           # ascending, no duplicates
    # diagonal of H0 always stored and equal to 0.5 (N - 2k)
    rp, ci, v = H0.row_ptr.numpy(), H0.col_idx.numpy(), H0.values.numpy()
    for r in [0, 1, n - 1, xxz.neel_index(N), n // 3]:
        row = ci[rp[r]:rp[r + 1]]
        assert r in row
        bits = [(r >> b) & 1 for b in range(N)]
        k = sum(bits[b] != bits[(b + 1) % N] for b in range(N))
        assert v[rp[r] + list(row).index(r)] == 0.5 * (N - 2 * k)
        assert rp[r + 1] - rp[r] == 1 + k
    S1 = H1.to_scipy()
    assert abs(S1.diagonal()).max() == 0 and np.all(H1.values.numpy() == 1.0)
    S0 = H0.to_scipy()
    assert abs(S0 - S0.getH()).max() == 0 and abs(S1 - S1.getH()).max() == 0


def test_neel_state():
    assert xxz.neel_index(10) == 0b0101010101 == 341
    psi = xxz.neel_state(10)
    assert psi[341] == 1 and torch.linalg.vector_norm(psi) == 1
    # the Neel rows attain the Gershgorin extreme: all N bonds antiparallel
    H0 = xxz.xxz_h0(10)
    rp = H0.row_ptr.numpy()
    assert rp[342] - rp[341] == 11


def test_rng_is_counter_based_and_normal():
    idx = torch.arange(0, 200000, dtype=torch.int64)
    x, y = rng.normal_pair(rng.SEED, 3, idx)
    x2, _ = rng.normal_pair(rng.SEED, 3, idx[1000:1010])
    assert torch.equal(x[1000:1010], x2)              # value depends on the counter only
    z = torch.cat([x, y]).numpy()
    assert abs(z.mean()) < 0.01 and abs(z.std() - 1) < 0.01
    assert abs(np.mean(z ** 4) - 3) < 0.1
    xa, _ = rng.normal_pair(rng.SEED, 4, idx[:10])
    assert not torch.equal(xa, x[:10])                # streams differ
    # splitmix64 known-answer: first output of the reference generator seeded with 0
    assert rng._splitmix64_int(0) == 0xE220A8397B1DCDAF
    t = rng.splitmix64(torch.tensor([0], dtype=torch.int64))
    assert int(t[0]) & ((1 << 64) - 1) == 0xE220A8397B1DCDAF


def test_dense_hermitian_semicircle():
    n = 512
    H0, H1 = dense.dense_h0(n), dense.dense_h1(n)
    assert H0.dtype == torch.complex128 and H0.is_contiguous()
    assert torch.equal(H0, H0.conj().T) and torch.equal(H1, H1.conj().T)
    assert not torch.equal(H0, H1)
    off = H0.numpy()[np.triu_indices(n, 1)]
    assert abs(np.mean(abs(off) ** 2) * n - 1) < 0.02          # E|H_ij|^2 = 1/n (reading g10)
    ev = np.linalg.eigvalsh(H0.numpy())
    assert 1.85 < ev.max() < 2.15 and -2.15 < ev.min() < -1.85  # semicircle radius 2


def test_random_unit_vector_and_configs():
    v = rng.random_unit_vector(4096)
    assert abs(float(torch.linalg.vector_norm(v)) - 1) < 1e-14
    c = W.CONFIGS
    assert [c[k].n for k in ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5")] == [1024, 2048, 1 << 20, 16384, 1 << 24]
    assert math.isclose(c["cfg1"].tau, 0.01) and math.isclose(c["cfg2"].tau, 0.02)
    assert math.isclose(c["cfg3"].tau, 0.05) and math.isclose(c["cfg4"].tau, 0.1)
    assert math.isclose(c["cfg5"].tau, 0.05) and c["cfg5"].schemes == ("cf4",)
    s = W.scaled(c["cfg3"], 8, nsteps=3)
    assert s.n == 256 and math.isclose(s.tau, 0.05) and s.nsteps == 3
    assert xxz.f_cos2t(0.3) == math.cos(0.6) and dense.f_sin3t(0.3) == math.sin(3 * 0.3)


# ------------------------------------------------------------------ the paper's own Examples 1 and 2
@pytest.mark.parametrize("n", [3, 4, 5])
def test_paper_example1_matches_kronecker_definition(n):
    from workloads import paper_examples as pe
    H0k = np.zeros((1 << n, 1 << n), dtype=complex)
    H1k = np.zeros_like(H0k)
    for i in range(1, n + 1):
        for j in range(1, n + 1):
            if i != j:
                H0k -= (1.0 / abs(i - j)) * site_op(SZ, i, n) @ site_op(SZ, j, n)
        H1k -= site_op(SX, i, n)
    H0, H1 = pe.example1_dense(n)
    assert np.allclose(H0.numpy(), H0k, atol=1e-14) and np.array_equal(H1.numpy(), H1k)


@pytest.mark.parametrize("n", [3, 4, 5, 6])
def test_paper_example2_matches_kronecker_definition(n):
    from workloads import paper_examples as pe
    jx, jy, jz = 1.0, 2.0, 3.0
    H0k = np.zeros((1 << n, 1 << n), dtype=complex)
    H1k = np.zeros_like(H0k)
    for j in range(1, n + 1):
        k = j % n + 1                       # periodic reading of sigma_{n+1}
        H0k -= 0.5 * (jx * site_op(SX, j, n) @ site_op(SX, k, n) + jy * site_op(SY, j, n) @ site_op(SY, k, n)
                      + jz * site_op(SZ, j, n) @ site_op(SZ, k, n))
        H1k -= 0.5 * site_op(SZ, j, n)
    H0, H1 = pe.example2_csr(n)
    assert np.allclose(H0.to_scipy().toarray(), H0k, atol=1e-14)
    assert np.array_equal(H1.to_scipy().toarray(), H1k)
    assert H0.nnz == (1 << n) * (n + 1)                     # exactly n + 1 stored entries per row
    ci = H0.col_idx.view(1 << n, n + 1)
    assert bool((ci[:, 1:] > ci[:, :-1]).all())             # ascending, no duplicates


def test_paper_initial_value():
    from workloads import paper_examples as pe
    n = 6
    psi = pe.initial_value(n).numpy()
    assert abs(np.linalg.norm(psi) - 1) < 1e-14
    sz1 = site_op(SZ, 1, n)
    sz2 = site_op(SZ, 2, n)
    assert abs(np.vdot(psi, sz1 @ psi) - 1) < 1e-14 and abs(np.vdot(psi, sz2 @ psi) + 1) < 1e-14   # up, down
