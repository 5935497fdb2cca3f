"""GPU parity tests (-m gpu): the CUDA path, called through the C-ABI binding,
against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star):
  * integer work (iteration counts, CSR structure of the commutator): exact;
  * final psi: relative 2-norm error <= 1e-9 at Leja tol 1e-12;
  * a single fused iteration / mat-vec / GEMM: elementwise, tolerance derived
    from the summation length (n_terms * eps * magnitude).
"""
import math
import os

import numpy as np
import pytest
import torch

import workloads as W
from workloads import dense, rng, xxz

pytestmark = pytest.mark.gpu

DEV = "cuda"


@pytest.fixture(scope="module")
def M():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1709_06483_b200 as pkg
    pkg.lib()
    return pkg


def relerr(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def to_dev(x):
    return x.to(DEV) if hasattr(x, "to") else x


def host(x):
    return x.cpu().numpy()


def random_sparse_hermitian(n, density, seed, long_row=None):
    """General (not XXZ) Hermitian CSR: ragged rows, some empty rows, optionally one long row."""
    import scipy.sparse as sp
    r = np.random.default_rng(seed)
    k = int(density * n * n)
    A = sp.csr_matrix((r.normal(size=k) + 1j * r.normal(size=k), (r.integers(0, n, size=k), r.integers(0, n, size=k))),
                      shape=(n, n))          # duplicate positions are summed
    if long_row is not None:
        cols = r.choice(n, size=long_row[1], replace=False)
        vals = r.normal(size=len(cols)) + 1j * r.normal(size=len(cols))
        A = A + sp.csr_matrix((vals, (np.full(len(cols), long_row[0]), cols)), shape=(n, n))
    H = ((A + A.getH()) * 0.5).tocsr()
    empty = r.choice(n, size=max(1, n // 50), replace=False)
    keep = np.ones(n)
    keep[empty] = 0.0                       # empty rows (and, to stay Hermitian, columns)
    if long_row is not None:
        keep[long_row[0]] = 1.0
    D = sp.diags(keep)
    H = (D @ H @ D).tocsr()
    H.eliminate_zeros()
    H.sort_indices()
    return H


def csr_from_scipy(S, device=DEV):
    return xxz.CSR(S.shape[0], torch.from_numpy(S.indptr.astype(np.int32)).to(device),
                   torch.from_numpy(S.indices.astype(np.int32)).to(device),
                   torch.from_numpy(S.data.astype(np.complex128)).to(device))


def rand_vec(n, seed):
    r = np.random.default_rng(seed)
    v = r.normal(size=n) + 1j * r.normal(size=n)
    return v / np.linalg.norm(v)


# ------------------------------------------------------------------ Gershgorin (S3)
@pytest.mark.parametrize("N,g", [(6, 0.0), (10, 0.7), (12, -0.31), (16, 0.45), (18, -1.3)])   # N >= 15: staged kernel
def test_gershgorin_csr_xxz(M, oracle, N, g):
    H0, H1 = xxz.xxz_h0(N), xxz.xxz_h1(N)
    a, b = M.magnus_gershgorin(H0.to(DEV), H1.to(DEV), g)
    S = (H0.to_scipy() + g * H1.to_scipy()).tocsr()
    S.sort_indices()
    (ra, rb), _ = oracle.gershgorin(oracle.CsrHost(S.shape[0], S.indptr.astype(np.int32), S.indices.astype(np.int32),
                                                   S.data.astype(complex)))
    assert math.isclose(a, ra, rel_tol=1e-13) and math.isclose(b, rb, rel_tol=1e-13)
    assert math.isclose(a, -(2.5 + abs(g)) * N, rel_tol=1e-13) and math.isclose(b, (1.5 + abs(g)) * N, rel_tol=1e-13)


@pytest.mark.parametrize("n,density", [(700, 0.01), (40001, 0.0002)])   # small kernel / staged kernel with a ragged tail
def test_gershgorin_csr_overlapping_patterns(M, oracle, n, density):
    """H0 and H1 with overlapping patterns: the modulus is taken of the SUMMED entry (c4)."""
    A = random_sparse_hermitian(n, density, 1, long_row=(5, 2500) if n > 32768 else None)
    B = random_sparse_hermitian(n, density, 2) + 0.5 * A
    B = B.tocsr(); B.sort_indices()
    g = -0.83
    a, b = M.magnus_gershgorin(csr_from_scipy(A), csr_from_scipy(B), g)
    S = (A + g * B).tocsr(); S.sort_indices()
    (ra, rb), _ = oracle.gershgorin(oracle.CsrHost(n, S.indptr.astype(np.int32), S.indices.astype(np.int32),
                                                   S.data.astype(complex)))
    assert math.isclose(a, ra, rel_tol=1e-12) and math.isclose(b, rb, rel_tol=1e-12)


@pytest.mark.parametrize("n", [1, 7, 200, 777])
def test_gershgorin_dense(M, oracle, n):
    H0 = dense.random_hermitian(n, stream=11)
    H1 = dense.random_hermitian(n, stream=12)
    a, b = M.magnus_gershgorin(H0.to(DEV), H1.to(DEV), 0.37)
    (ra, rb), _ = oracle.gershgorin((H0 + 0.37 * H1).numpy())
    assert math.isclose(a, ra, rel_tol=1e-12, abs_tol=1e-14) and math.isclose(b, rb, rel_tol=1e-12, abs_tol=1e-14)
    a, b = M.magnus_gershgorin(H0.to(DEV))
    (ra, rb), _ = oracle.gershgorin(H0.numpy())
    assert math.isclose(a, ra, rel_tol=1e-12, abs_tol=1e-14) and math.isclose(b, rb, rel_tol=1e-12, abs_tol=1e-14)


# ------------------------------------------------------------------ one fused iteration (S6)
def expected_iteration(oracle, Mh, w, p, inv_gamma, shift, d):
    y = oracle.matvec(Mh, w)
    wn = inv_gamma * y - shift * w
    pn = p + d * wn
    return wn, pn


@pytest.mark.parametrize("N,kernel", [(8, 1), (12, 1), (12, 2), (15, 2), (16, 0), (8, 3), (12, 3), (16, 3), (16, 24001), (16, 27081), (16, 22040), (8, 4), (12, 4), (16, 4), (3, 5), (8, 5), (12, 5), (16, 5), (16, 5083), (16, 5045), (3, 6), (8, 6), (12, 6), (16, 6), (16, 6003), (16, 6104), (16, 6204), (16, 6016), (12, 6018),
                                      (8, 6504), (16, 6504), (16, 6515)])   # 65xx: real-part storage (shortcut) of the real chain
def test_fused_iteration_csr_xxz(M, oracle, N, kernel):
    n = 1 << N
    H0, H1 = xxz.xxz_h0(N), xxz.xxz_h1(N)
    g = 0.61
    w = rand_vec(n, 1)
    p = rand_vec(n, 2)
    S = (H0.to_scipy() + g * H1.to_scipy()).tocsr(); S.sort_indices()
    Mh = oracle.CsrHost(n, S.indptr.astype(np.int32), S.indices.astype(np.int32), S.data.astype(complex))
    inv_gamma, shift, d = 1.0 / (0.675 * N), -0.3 + 1.1547, 0.3 - 0.2j
    wn, pn = expected_iteration(oracle, Mh, w, p, inv_gamma, shift, d)
    wi, wo, pd = torch.from_numpy(w).to(DEV), torch.zeros(n, dtype=torch.complex128, device=DEV), torch.from_numpy(p).to(DEV)
    sw, sp, _ = M.magnus_leja_iteration(H0.to(DEV), H1.to(DEV), g, wi, wo, pd, inv_gamma, shift, d, csr_kernel=kernel)
    tol = 64 * N * np.finfo(float).eps
    assert np.max(np.abs(host(wo) - wn)) <= tol * np.max(np.abs(wn)) + 1e-300
    assert np.max(np.abs(host(pd) - pn)) <= tol * np.max(np.abs(pn))
    assert math.isclose(sw, np.sum(np.abs(wn) ** 2), rel_tol=1e-12)
    assert math.isclose(sp, np.sum(np.abs(pn) ** 2), rel_tol=1e-12)


@pytest.mark.parametrize("kernel,long_len", [(1, 1900), (2, 1900), (3, 1900), (3, 2990), (27001, 2990), (22030, 700), (23000, 40), (4, 1900), (4, 40), (5, 1900), (5, 40), (5045, 300), (6, 1900), (6, 40), (6003, 300)])
def test_fused_iteration_csr_general_ragged(M, oracle, kernel, long_len):
    """Non-power-of-two n, empty rows, one row longer than the row-block staging buffer / than a ring stage of
    the stream kernel (kernel 3 and its 2000+ variants: that unit is read straight from global memory), rows
    longer than 32 entries, an index array whose length is not a multiple of four (unaligned tail unit)."""
    n = 3001
    S = random_sparse_hermitian(n, 0.004, 5, long_row=(17, long_len))
    Mh = oracle.CsrHost(n, S.indptr.astype(np.int32), S.indices.astype(np.int32), S.data.astype(complex))
    w, p = rand_vec(n, 3), rand_vec(n, 4)
    inv_gamma, shift, d = 0.05, 0.7, -0.11 + 0.4j
    wn, pn = expected_iteration(oracle, Mh, w, p, inv_gamma, shift, d)
    wi, wo, pd = torch.from_numpy(w).to(DEV), torch.zeros(n, dtype=torch.complex128, device=DEV), torch.from_numpy(p).to(DEV)
    sw, sp, _ = M.magnus_leja_iteration(csr_from_scipy(S), None, 0.0, wi, wo, pd, inv_gamma, shift, d, csr_kernel=kernel)
    assert np.max(np.abs(host(wo) - wn)) <= 1e-13 * max(1.0, np.max(np.abs(wn)))
    assert np.max(np.abs(host(pd) - pn)) <= 1e-13 * max(1.0, np.max(np.abs(pn)))
    assert math.isclose(sw, np.sum(np.abs(wn) ** 2), rel_tol=1e-12)


@pytest.mark.parametrize("n", [1, 33, 500, 1237])
def test_fused_iteration_dense(M, oracle, n):
    H0 = dense.random_hermitian(n, stream=21)
    H1 = dense.random_hermitian(n, stream=22)
    g = -0.45
    Mh = (H0 + g * H1).numpy()
    w, p = rand_vec(n, 5), rand_vec(n, 6)
    inv_gamma, shift, d = 0.11, -0.9, 0.02 + 0.5j
    wn, pn = expected_iteration(oracle, Mh, w, p, inv_gamma, shift, d)
    wi, wo, pd = torch.from_numpy(w).to(DEV), torch.zeros(n, dtype=torch.complex128, device=DEV), torch.from_numpy(p).to(DEV)
    sw, sp, _ = M.magnus_leja_iteration(H0.to(DEV), H1.to(DEV), g, wi, wo, pd, inv_gamma, shift, d)
    tol = 8 * max(n, 16) * np.finfo(float).eps
    assert np.max(np.abs(host(wo) - wn)) <= tol * max(np.max(np.abs(wn)), np.max(np.abs(w)))
    assert np.max(np.abs(host(pd) - pn)) <= tol * max(np.max(np.abs(pn)), 1e-3)
    assert math.isclose(sw, np.sum(np.abs(wn) ** 2), rel_tol=1e-12)
    assert math.isclose(sp, np.sum(np.abs(pn) ** 2), rel_tol=1e-12)


# ------------------------------------------------------------------ leja_expmv (S3-S8)
@pytest.mark.parametrize("N,h", [(6, 0.3), (10, 0.05), (10, -0.4), (14, 0.1), (16, 0.05)])
def test_expmv_csr_vs_oracle(M, oracle, N, h):
    n = 1 << N
    S = (xxz.xxz_h0(N).to_scipy() + 0.77 * xxz.xxz_h1(N).to_scipy()).tocsr(); S.sort_indices()
    Mh = oracle.CsrHost(n, S.indptr.astype(np.int32), S.indices.astype(np.int32), S.data.astype(complex))
    v = rand_vec(n, 7)
    ref, rinfo = oracle.leja_expmv(Mh, v, h, 1e-12)
    vi = torch.from_numpy(v).to(DEV)
    vo = torch.empty_like(vi)
    info = M.leja_expmv(csr_from_scipy(S), vi, vo, h, 1e-12)
    assert info["iters"] == rinfo["iters"] and info["substeps"] == rinfo["substeps"]
    assert info["a"] == rinfo["a"] and info["b"] == rinfo["b"] and info["theta"] == rinfo["theta"]
    assert relerr(host(vo), ref) <= 1e-12
    assert abs(np.linalg.norm(host(vo)) - 1.0) < 1e-10
    # in place
    info2 = M.leja_expmv(csr_from_scipy(S), vi, vi, h, 1e-12)
    assert info2["iters"] == info["iters"] and torch.equal(vi, vo)


@pytest.mark.parametrize("n,h,scale", [(1, 0.7, 1.0), (2, 1.0, 1.0), (64, 0.3, 0.7), (300, 0.1, 1.0), (1111, -0.05, 1.0)])
def test_expmv_dense_vs_oracle_and_eigh(M, oracle, n, h, scale):
    H = (dense.random_hermitian(n, stream=31) * scale).contiguous()
    v = rand_vec(n, 8)
    ref, rinfo = oracle.leja_expmv(H.numpy(), v, h, 1e-12)
    vi = torch.from_numpy(v).to(DEV)
    vo = torch.empty_like(vi)
    info = M.leja_expmv(H.to(DEV), vi, vo, h, 1e-12)
    assert info["iters"] == rinfo["iters"] and info["a"] == rinfo["a"] and info["b"] == rinfo["b"]
    assert relerr(host(vo), ref) <= 1e-12
    lam, U = np.linalg.eigh(H.numpy())
    exact = U @ (np.exp(-1j * h * lam) * (U.conj().T @ v))
    assert np.linalg.norm(host(vo) - exact) <= 1e-11          # 10 tol (pin c-P3)


def test_expmv_degenerate_cases(M, oracle):
    # M = c I: gamma = 0, zero iterations, exact phase
    n = 5
    H = (2.5 * torch.eye(n, dtype=torch.complex128)).to(DEV)
    v = torch.from_numpy(rand_vec(n, 9)).to(DEV)
    out = torch.empty_like(v)
    info = M.leja_expmv(H, v, out, 0.4)
    assert info["iters"] == 0 and np.allclose(host(out), np.exp(-1j) * host(v), atol=1e-15)
    # h = 0: exactly two iterations (d_k = 0 for k >= 1), result == input
    H = dense.random_hermitian(40, stream=41).to(DEV)
    v = torch.from_numpy(rand_vec(40, 10)).to(DEV)
    info = M.leja_expmv(H, v, out := torch.empty_like(v), 0.0)
    assert info["iters"] == 2 and torch.equal(out, v)
    # theta > theta_max: sub-steps
    Hh = dense.random_hermitian(24, stream=42) * 3.0
    (_, _), (sa, sb) = oracle.gershgorin(Hh.numpy())
    hbig = 40.0 / ((sb - sa) / 4)
    vv = rand_vec(24, 11)
    ref, rinfo = oracle.leja_expmv(Hh.numpy(), vv, hbig, 1e-12)
    vi = torch.from_numpy(vv).to(DEV)
    info = M.leja_expmv(Hh.to(DEV), vi, vo := torch.empty_like(vi), hbig)
    assert info["substeps"] == rinfo["substeps"] == 3 and info["iters"] == rinfo["iters"]
    assert relerr(host(vo), ref) <= 1e-11
    # diagonal CSR (no off-diagonal entries): componentwise phases
    import scipy.sparse as sp
    x = np.array([-1.5, 0.2, 0.9, 3.0])
    D = sp.diags(x.astype(complex)).tocsr()
    vv = rand_vec(4, 12)
    vi = torch.from_numpy(vv).to(DEV)
    M.leja_expmv(csr_from_scipy(D), vi, vo := torch.empty_like(vi), 0.8)
    assert np.allclose(host(vo), np.exp(-0.8j * x) * vv, atol=1e-12)


def test_expmv_reports_nonconvergence(M):
    n = 64
    H = dense.random_hermitian(n, stream=43).to(DEV)
    v = torch.from_numpy(rand_vec(n, 13)).to(DEV)
    with pytest.raises(M.MagnusError) as e:
        # |d_k| decays like theta^k / k!, so the two-term estimate drops below any moderate tol well before
        # m_max = 128; only a tolerance under the size of d_128 (about 1e-100 at theta = 7) is unreachable
        M.leja_expmv(H, v, torch.empty_like(v), 2.0, 1e-300)
    assert e.value.code == -4


# ------------------------------------------------------------------ commutators (S0, D3)
@pytest.mark.parametrize("n", [8, 64, 130, 257, 600])
def test_zgemm_dmma_vs_oracle_product(M, oracle, n):
    A = dense.random_hermitian(n, stream=51)
    B = dense.random_hermitian(n, stream=52) + 0.1j * torch.triu(torch.ones(n, n, dtype=torch.complex128), 1)
    Cd = torch.empty(n, n, dtype=torch.complex128, device=DEV)
    M.magnus_zgemm(A.to(DEV), B.to(DEV), Cd)
    ref = oracle.matmul(A.numpy(), B.numpy())
    assert np.max(np.abs(host(Cd) - ref)) <= 8 * n * np.finfo(float).eps * np.max(np.abs(ref)) + 1e-300


@pytest.mark.parametrize("n", [2048, 2300, 2944, 3100])
def test_zgemm_stream_k_sampled_rows_and_columns(M, oracle, n):
    """Sizes whose 128 x 64 tile count leaves the last wave badly filled run the stream-K form of the DMMA GEMM
    (tiles split between two CTAs, partial tile parked and added): 2048 = CFG2, 2300 and 3100 with ragged edge tiles,
    2944 = 23 x 46 tiles.  Six whole rows and six whole columns of A B against the oracle's mat-vec, among them the
    first and last and rows / columns of split tiles."""
    A = dense.random_hermitian(n, stream=53)
    B = dense.random_hermitian(n, stream=54) + 0.1j * torch.triu(torch.ones(n, n, dtype=torch.complex128), 1)
    Cd = torch.empty(n, n, dtype=torch.complex128, device=DEV)
    M.magnus_zgemm(A.to(DEV), B.to(DEV), Cd)
    C = host(Cd)
    An, Bn = A.numpy(), B.numpy()
    idx = [0, n - 1, 127, 128, n // 2 + 3, (3 * n) // 4]
    tol = 8 * n * np.finfo(float).eps
    for j in idx:
        col = oracle.matvec(An, np.ascontiguousarray(Bn[:, j]))               # column j of A B = A (B e_j)
        assert np.max(np.abs(C[:, j] - col)) <= tol * np.max(np.abs(col))
        row = oracle.matvec(np.ascontiguousarray(Bn.T), np.ascontiguousarray(An[j, :]))   # row j of A B = B^T (A^T e_j)
        assert np.max(np.abs(C[j, :] - row)) <= tol * np.max(np.abs(row))
    assert np.isfinite(C).all()
    ref = An[5::97, :] @ Bn                                                         # a coarse sweep over all tiles
    assert np.max(np.abs(C[5::97, :] - ref)) <= tol * np.max(np.abs(ref))


@pytest.mark.parametrize("n", [48, 200, 333])
def test_dense_commutator_vs_oracle(M, oracle, n):
    A = dense.random_hermitian(n, stream=53)
    B = dense.random_hermitian(n, stream=54)
    K = torch.empty(n, n, dtype=torch.complex128, device=DEV)
    work = torch.empty_like(K)
    M.magnus_commutator_dense(A.to(DEV), B.to(DEV), K, work)
    ref = oracle.commutator(A.numpy(), B.numpy())           # plain definition AB - BA
    assert np.max(np.abs(host(K) - ref)) <= 16 * n * np.finfo(float).eps * max(np.max(np.abs(ref)), 1.0)
    assert np.max(np.abs(host(K) + host(K).conj().T)) == 0.0   # exactly anti-Hermitian by construction


@pytest.mark.parametrize("N", [4, 7, 10])
def test_sparse_commutator_vs_oracle(M, oracle, N):
    H0, H1 = xxz.xxz_h0(N), xxz.xxz_h1(N)
    rp, ci, v = M.magnus_commutator_csr(H0.to(DEV), H1.to(DEV))
    K = oracle.commutator(oracle.CsrHost.of(H0), oracle.CsrHost.of(H1))
    import scipy.sparse as sp
    n = 1 << N
    ref = sp.csr_matrix((K.values, K.col_idx, K.row_ptr), shape=(n, n)); ref.eliminate_zeros(); ref.sort_indices()
    got = sp.csr_matrix((host(v), host(ci), host(rp)), shape=(n, n))
    assert got.nnz == N * 2 ** (N - 1) == ref.nnz           # exact zeros dropped (pin c-P11)
    assert np.array_equal(got.indptr, ref.indptr) and np.array_equal(got.indices, ref.indices)
    assert np.array_equal(got.data, ref.data)               # small integers: exact


@pytest.mark.parametrize("n,density,long_row", [(400, 0.02, None), (1500, 0.002, (7, 300)), (900, 0.004, (11, 120))])
def test_sparse_commutator_general(M, oracle, n, density, long_row):
    """General CSR input.  Rows with more than 32 resulting entries (most rows of the first case), with more
    than 256 source rows (the long row of the second) or with more than 1024 candidate products leave the
    warp kernel through its worklist and are done by the CTA-wide kernel; the others stay with the warp."""
    A = random_sparse_hermitian(n, density, 21, long_row=long_row)
    B = random_sparse_hermitian(n, density, 22)
    rp, ci, v = M.magnus_commutator_csr(csr_from_scipy(A), csr_from_scipy(B))
    import scipy.sparse as sp
    got = sp.csr_matrix((host(v), host(ci), host(rp)), shape=(n, n)).toarray()
    K = oracle.commutator(oracle.CsrHost(n, A.indptr.astype(np.int32), A.indices.astype(np.int32), A.data.astype(complex)),
                          oracle.CsrHost(n, B.indptr.astype(np.int32), B.indices.astype(np.int32), B.data.astype(complex)))
    ref = sp.csr_matrix((K.values, K.col_idx, K.row_ptr), shape=(n, n)).toarray()
    assert np.max(np.abs(got - ref)) <= 1e-13 * max(1.0, np.max(np.abs(ref)))
    assert np.all(np.diff(host(ci)[host(rp)[7]:host(rp)[8]]) > 0)      # columns ascending inside a row


# ------------------------------------------------------------------ magnus_step / magnus_integrate
def run_config(M, oracle, cfg, scheme, device_inputs=None):
    H0, H1, psi0, f = W.build(cfg)
    if cfg.kind == "xxz":
        o0, o1 = oracle.CsrHost.of(H0), oracle.CsrHost.of(H1)
        d0, d1 = H0.to(DEV), H1.to(DEV)
    else:
        o0, o1 = H0.numpy(), H1.numpy()
        d0, d1 = H0.to(DEV), H1.to(DEV)
    ref, riters = oracle.magnus_integrate(o0, o1, f, scheme, cfg.t0, cfg.t_end, cfg.nsteps, psi0.numpy(), cfg.tol)
    psi = psi0.to(DEV).clone()
    with M.magnus_create(d0, d1, f, scheme, tol=cfg.tol) as h:
        st = h.integrate(cfg.t0, cfg.t_end, cfg.nsteps, psi)
    return host(psi), st, ref, riters


@pytest.mark.parametrize("scheme", ["cf4", "m4"])
def test_cfg1_full(M, oracle, scheme):
    """BASELINE config 1 at full size: XXZ N=10, Neel state, T=1, 100 steps."""
    psi, st, ref, riters = run_config(M, oracle, W.CONFIGS["cfg1"], scheme)
    assert np.array_equal(st["iters"], riters)              # identical Leja iteration counts
    assert relerr(psi, ref) <= 1e-9
    assert abs(np.linalg.norm(psi) - 1) < 1e-10


@pytest.mark.parametrize("scheme", ["cf4", "m4"])
@pytest.mark.parametrize("n,nsteps", [(96, 6), (515, 4)])
def test_cfg2_scaled(M, oracle, scheme, n, nsteps):
    """Config 2's recipe (dense random Hermitian, f = sin 3t, tau = 0.02) at sizes with ragged tiles."""
    cfg = W.scaled(W.CONFIGS["cfg2"], n, nsteps)
    psi, st, ref, riters = run_config(M, oracle, cfg, scheme)
    assert np.array_equal(st["iters"], riters)
    assert relerr(psi, ref) <= 1e-9
    assert abs(np.linalg.norm(psi) - 1) < 1e-10


def test_cfg2_full_cf4(M, oracle):
    cfg = W.CONFIGS["cfg2"]
    psi, st, ref, riters = run_config(M, oracle, cfg, "cf4")
    assert np.array_equal(st["iters"], riters)
    assert relerr(psi, ref) <= 1e-9


def test_cfg2_full_m4_three_steps(M, oracle):
    """Full n = 2048 with the DMMA commutator; 3 of the 50 steps (the oracle's plain-definition
    products cost 1.4e11 flop per step on the host)."""
    cfg = W.scaled(W.CONFIGS["cfg2"], 2048, 3)
    psi, st, ref, riters = run_config(M, oracle, cfg, "m4")
    assert np.array_equal(st["iters"], riters)
    assert relerr(psi, ref) <= 1e-9


@pytest.mark.parametrize("scheme", ["cf4", "m4"])
def test_cfg3_scaled(M, oracle, scheme):
    """Config 3's recipe (XXZ, random psi0, tau = 0.05) at N = 16: row-block CSR kernel, several waves."""
    cfg = W.scaled(W.CONFIGS["cfg3"], 16, 4)
    psi, st, ref, riters = run_config(M, oracle, cfg, scheme)
    assert np.array_equal(st["iters"], riters)
    assert relerr(psi, ref) <= 1e-9
    assert abs(np.linalg.norm(psi) - 1) < 1e-10


def test_cfg3_full_two_steps(M, oracle):
    """Config 3 at full size (N = 20, 32.5M stored entries), 2 of the 20 steps, CF4."""
    cfg = W.scaled(W.CONFIGS["cfg3"], 20, 2)
    psi, st, ref, riters = run_config(M, oracle, cfg, "cf4")
    assert np.array_equal(st["iters"], riters)
    assert relerr(psi, ref) <= 1e-9


def test_step_info_and_time_reversal(M):
    """Pin c-P10 on the GPU path: step(t, tau) then step(t + tau, -tau) returns psi."""
    cfg = W.scaled(W.CONFIGS["cfg1"], 8, 1)
    H0, H1, _, f = W.build(cfg)
    psi0 = rng.random_unit_vector(256)
    for scheme in ("cf4", "m4", "m2", "cf4:3"):
        psi = psi0.to(DEV).clone()
        with M.magnus_create(H0.to(DEV), H1.to(DEV), f, scheme) as h:
            infos = h.step(0.2, 0.1, psi)
            assert len(infos) == {"cf4": 2, "m4": 1, "m2": 1, "cf4:3": 3}[scheme]
            assert all(i["iters"] > 0 and i["status"] == 0 for i in infos)
            h.step(0.3, -0.1, psi)
        assert np.linalg.norm(host(psi) - psi0.numpy()) < 1e-11


def test_order_four_on_gpu_path(M):
    """Pin c-P8 through the CUDA path: step-halving slope 4 for CF4, M4 and CF4:3, 2 for M2."""
    N = 6
    H0, H1 = xxz.xxz_h0(N).to(DEV), xxz.xxz_h1(N).to(DEV)
    psi0 = xxz.neel_state(N)
    T = 0.5

    def run(scheme, ns, tol=1e-14):
        psi = psi0.to(DEV).clone()
        with M.magnus_create(H0, H1, xxz.f_cos2t, scheme, tol=tol) as h:
            h.integrate(0.0, T, ns, psi)
        return host(psi)

    for scheme, order in (("cf4", 4), ("m4", 4), ("cf4:3", 4), ("m2", 2)):
        ref = run(scheme, 512 if order == 4 else 4096)
        errs = [np.linalg.norm(run(scheme, ns) - ref) for ns in (4, 8, 16)]
        slopes = [math.log2(errs[i] / errs[i + 1]) for i in range(2)]
        assert all(order - 0.25 < s < order + 0.25 for s in slopes), (scheme, errs, slopes)


def test_integrate_host_end_to_end(M, oracle):
    cfg = W.CONFIGS["cfg1"]
    H0, H1, psi0, f = W.build(cfg)
    ref, riters = oracle.magnus_integrate(oracle.CsrHost.of(H0), oracle.CsrHost.of(H1), f, "cf4", 0.0, 0.1, 10,
                                          psi0.numpy(), 1e-12)
    pin = lambda t: t.pin_memory()
    H0p = xxz.CSR(H0.n, pin(H0.row_ptr), pin(H0.col_idx), pin(H0.values))
    H1p = xxz.CSR(H1.n, pin(H1.row_ptr), pin(H1.col_idx), pin(H1.values))
    psi = pin(psi0.clone())
    st = M.magnus_integrate_host(H0p, H1p, f, "cf4", 0.0, 0.1, 10, psi)
    assert np.array_equal(st["iters"], riters) and relerr(psi.numpy(), ref) <= 1e-9


@pytest.mark.parametrize("scheme", ["cf4", "m4"])
def test_step_csr_overlapping_patterns(M, oracle, scheme):
    """General CSR H0, H1 whose patterns OVERLAP: the handle must not use the cached separable row
    statistics for the Gershgorin bounds (modulus of the summed entry, c4) and must still match the oracle."""
    n = 900
    A = random_sparse_hermitian(n, 0.01, 31)
    B = (random_sparse_hermitian(n, 0.01, 32) + 0.5 * A).tocsr()
    B.sort_indices()
    f = lambda t: math.cos(1.3 * t) - 0.2
    psi0 = rand_vec(n, 33)
    oA = oracle.CsrHost(n, A.indptr.astype(np.int32), A.indices.astype(np.int32), A.data.astype(complex))
    oB = oracle.CsrHost(n, B.indptr.astype(np.int32), B.indices.astype(np.int32), B.data.astype(complex))
    ref, rinfo = oracle.magnus_step(oA, oB, f, scheme, 0.1, 0.05, psi0, 1e-12)
    psi = torch.from_numpy(psi0).to(DEV)
    with M.magnus_create(csr_from_scipy(A), csr_from_scipy(B), f, scheme) as h:
        info = h.step(0.1, 0.05, psi)
    assert [i["iters"] for i in info] == [i["iters"] for i in rinfo]
    assert all(i["a"] == r["a"] and i["b"] == r["b"] for i, r in zip(info, rinfo))
    assert relerr(host(psi), ref) <= 1e-9


# ------------------------------------------------------------------ M2 and Cf4:3 against the oracle
@pytest.mark.parametrize("scheme", ["m2", "cf4:3"])
@pytest.mark.parametrize("name,size,nsteps", [("cfg1", 10, 20), ("cfg3", 16, 3), ("cfg2", 515, 4)])
def test_m2_cf43_vs_oracle(M, oracle, scheme, name, size, nsteps):
    """The other two commutator-free schemes of the paper through the same kernels:
    identical iteration counts per exponential (1 resp. 3 per step), psi within 1e-9."""
    cfg = W.scaled(W.CONFIGS[name], size, nsteps)
    psi, st, ref, riters = run_config(M, oracle, cfg, scheme)
    assert len(riters) == nsteps * {"m2": 1, "cf4:3": 3}[scheme]
    assert np.array_equal(st["iters"], riters)
    assert relerr(psi, ref) <= 1e-9
    assert abs(np.linalg.norm(psi) - 1) < 1e-10


# ------------------------------------------------------------------ M6 against the oracle
@pytest.mark.parametrize("name,size,nsteps", [("cfg1", 10, 10), ("cfg3", 12, 3), ("cfg2", 515, 4), ("cfg2", 1024, 2)])
def test_m6_vs_oracle(M, oracle, name, size, nsteps):
    """The sixth-order scheme: three DMMA products per step built from Hermitian / anti-Hermitian factors
    (magnus.h at magnus_step) against the oracle's six plain-definition products; CSR input runs on dense copies
    on the GPU and as sparse matrices in the oracle.  Identical iteration counts, psi within 1e-9."""
    cfg = W.scaled(W.CONFIGS[name], size, nsteps)
    psi, st, ref, riters = run_config(M, oracle, cfg, "m6")
    assert len(riters) == nsteps
    assert np.array_equal(st["iters"], riters)
    assert relerr(psi, ref) <= 1e-9
    assert abs(np.linalg.norm(psi) - 1) < 1e-10


def test_m6_is_more_accurate_than_m4_and_refuses_large_csr(M):
    """Self-convergence at a coarse step: M6 is far closer to a fine-step solution than M4; CSR input beyond
    the dense-copy limit is refused with EINVAL instead of running out of memory."""
    cfg = W.scaled(W.CONFIGS["cfg2"], 256, 4)
    H0, H1, psi0, f = W.build(cfg, device=DEV)
    def run(scheme, ns):
        psi = psi0.clone()
        with M.magnus_create(H0, H1, f, scheme, tol=1e-13) as h:
            h.integrate(0.0, 0.4, ns, psi)
        return psi
    fine = run("m6", 64)
    e6 = float(torch.linalg.vector_norm(run("m6", 4) - fine))
    e4 = float(torch.linalg.vector_norm(run("m4", 4) - fine))
    assert e6 < 0.1 * e4 and e6 < 1e-6, (e6, e4)
    big = W.scaled(W.CONFIGS["cfg3"], 15, 1)
    B0, B1, _, fb = W.build(big, device=DEV)
    with pytest.raises(M.MagnusError) as ei:
        M.magnus_create(B0, B1, fb, "m6")
    assert ei.value.code == -1


def test_argument_errors_surface_as_einval_not_as_enoconv(M):
    """Three misuse cases that used to fail late or misleadingly: (1) MAGNUS_M6 on strided dense input is refused at
    create (it failed at every step); (2) an M6 step with tau = 0 (Omega_H divides by tau) is EINVAL; (3) a csr_kernel
    tuning code outside the launch tables launches nothing -- the call reports EINVAL naming the code instead of
    polling up to m_max and returning ENOCONV."""
    n = 96
    cfg = W.scaled(W.CONFIGS["cfg2"], n, 1)
    H0, H1, psi0, f = W.build(cfg, device=DEV)
    wide0 = torch.zeros((n, n + 3), dtype=torch.complex128, device=DEV)
    wide1 = torch.zeros_like(wide0)
    wide0[:, :n], wide1[:, :n] = H0, H1
    with pytest.raises(M.MagnusError) as e:
        M.magnus_create(wide0[:, :n], wide1[:, :n], f, "m6")
    assert e.value.code == -1 and "ld == n" in str(e.value)
    with M.magnus_create(H0, H1, f, "m6") as h:
        psi = psi0.clone()
        with pytest.raises(M.MagnusError) as e:
            h.step(0.0, 0.0, psi)
        assert e.value.code == -1 and "tau" in str(e.value)
        assert torch.equal(psi, psi0)
        h.step(0.0, 0.01, psi)                                   # the handle is still usable
        assert abs(float(torch.linalg.vector_norm(psi)) - 1) < 1e-10
    big = W.scaled(W.CONFIGS["cfg3"], 12, 1)
    B0, B1, p0, fb = W.build(big, device=DEV)
    w, wo, p = p0.clone(), torch.zeros_like(p0), p0.clone()
    for code in (6013, 5077):
        with pytest.raises(M.MagnusError) as e:
            M.magnus_leja_iteration(B0, B1, 0.3, w, wo, p, 0.1, 0.2, 0.5 + 0.1j, csr_kernel=code)
        assert e.value.code == -1 and str(code) in str(e.value)
        with M.magnus_create(B0, B1, fb, "cf4", csr_kernel=code) as h:
            psi = p0.clone()
            with pytest.raises(M.MagnusError) as e:
                h.step(0.0, 0.05, psi)
            assert e.value.code == -1 and str(code) in str(e.value)


# ------------------------------------------------------------------ shortcut: cached dense commutator
@pytest.mark.parametrize("n,nsteps", [(200, 5), (515, 3), (2048, 2)])
def test_shortcut_cached_dense_commutator_vs_oracle(M, oracle, n, nsteps):
    """Dense M4 with P0 = H0 H1 formed once at create ([H(t2), H(t1)] = (f1 - f2)[H0, H1]) against the oracle's
    per-step plain-definition commutator: identical counts and interval, psi within 1e-9; and it agrees with the
    mandated per-step-GEMM path of the library to rounding."""
    cfg = W.scaled(W.CONFIGS["cfg2"], n, nsteps)
    H0, H1, psi0, f = W.build(cfg)
    ref, riters = oracle.magnus_integrate(H0.numpy(), H1.numpy(), f, "m4", cfg.t0, cfg.t_end, nsteps, psi0.numpy(), cfg.tol)
    d0, d1 = H0.to(DEV), H1.to(DEV)
    out = {}
    for sc in (0, M.SHORTCUT_CACHED_COMMUTATOR):
        psi = psi0.to(DEV).clone()
        with M.magnus_create(d0, d1, f, "m4", tol=cfg.tol, shortcuts=sc) as h:
            st = h.integrate(cfg.t0, cfg.t_end, nsteps, psi)
        assert np.array_equal(st["iters"], riters)
        assert relerr(host(psi), ref) <= 1e-9
        out[sc] = (host(psi), st)
    assert relerr(out[1][0], out[0][0]) <= 1e-12
    assert out[1][1]["seconds_commutator"] == 0.0 and out[0][1]["seconds_commutator"] > 0.0


# ------------------------------------------------------------------ the paper's own workloads
@pytest.mark.parametrize("scheme", ["cf4", "m4", "cf4:3"])
def test_paper_example2_local_heisenberg(M, oracle, scheme):
    """Example 2: Jx, Jy, Jz = 1, 2, 3, z-field sin t, CSR with n + 1 entries per row, tau = 1e-3 as in the
    paper's runs, plus a larger step.  H1 is diagonal here, so H0 and H1 OVERLAP on the diagonal."""
    from workloads import paper_examples as pe
    n = 10
    H0, H1 = pe.example2_csr(n)
    psi0 = pe.initial_value(n)
    o0, o1 = oracle.CsrHost.of(H0), oracle.CsrHost.of(H1)
    for t_end, nsteps in ((0.005, 5), (0.3, 6)):
        ref, riters = oracle.magnus_integrate(o0, o1, pe.f_sin_t, scheme, 0.0, t_end, nsteps, psi0.numpy(), 1e-12)
        psi = psi0.to(DEV).clone()
        with M.magnus_create(H0.to(DEV), H1.to(DEV), pe.f_sin_t, scheme) as h:
            st = h.integrate(0.0, t_end, nsteps, psi)
        assert np.array_equal(st["iters"], riters)
        assert relerr(host(psi), ref) <= 1e-9


@pytest.mark.parametrize("scheme", ["cf4", "m4"])
def test_paper_example1_nonlocal_heisenberg(M, oracle, scheme):
    """Example 1: J_ij = 1/|i-j|, x-field sin t, stored dense (N = 2^8)."""
    from workloads import paper_examples as pe
    n = 8
    H0, H1 = pe.example1_dense(n)
    psi0 = pe.initial_value(n)
    ref, riters = oracle.magnus_integrate(H0.numpy(), H1.numpy(), pe.f_sin_t, scheme, 0.0, 0.2, 4, psi0.numpy(), 1e-12)
    psi = psi0.to(DEV).clone()
    with M.magnus_create(H0.to(DEV), H1.to(DEV), pe.f_sin_t, scheme) as h:
        st = h.integrate(0.0, 0.2, 4, psi)
    assert np.array_equal(st["iters"], riters)
    assert relerr(host(psi), ref) <= 1e-9


def test_small_csr_sweep_paths(M, oracle):
    """The single-launch sweep (n <= 4096): non-convergence is reported and leaves the vector untouched;
    sub-steps chain sweeps; forcing the per-iteration kernels (csr_kernel=1) gives the same counts and result."""
    N = 9
    n = 1 << N
    S = (xxz.xxz_h0(N).to_scipy() + 0.4 * xxz.xxz_h1(N).to_scipy()).tocsr(); S.sort_indices()
    Hd = csr_from_scipy(S)
    v = torch.from_numpy(rand_vec(n, 21)).to(DEV)
    keep = v.clone()
    with pytest.raises(M.MagnusError) as e:
        M.leja_expmv(Hd, v, v, 1.5, 1e-300)                  # in place: must not be overwritten on failure
    assert e.value.code == -4 and torch.equal(v, keep)
    Mh = oracle.CsrHost(n, S.indptr.astype(np.int32), S.indices.astype(np.int32), S.data.astype(complex))
    ref, rinfo = oracle.leja_expmv(Mh, host(keep), 2.0, 1e-25)   # two sub-steps, long sweeps (the oracle's
    out = torch.empty_like(v)                                    # __float128 table is exact to about 1e-32)
    info = M.leja_expmv(Hd, v, out, 2.0, 1e-25)
    assert info["substeps"] == rinfo["substeps"] == 2
    assert info["iters"] == rinfo["iters"] and relerr(host(out), ref) <= 1e-12
    H0, H1 = xxz.xxz_h0(N).to(DEV), xxz.xxz_h1(N).to(DEV)
    res = {}
    for ck in (0, 1):
        psi = keep.clone()
        with M.magnus_create(H0, H1, xxz.f_cos2t, "cf4", csr_kernel=ck) as h:
            st = h.integrate(0.0, 0.2, 4, psi)
        res[ck] = (st["iters"], host(psi))
    assert np.array_equal(res[0][0], res[1][0]) and relerr(res[0][1], res[1][1]) <= 1e-13


# ------------------------------------------------------------------ planned batches (whole-sweep kernels)
@pytest.mark.parametrize("scheme", ["cf4", "cf4:3"])
@pytest.mark.parametrize("n", [1, 2, 33, 150, 777, 1237])
def test_planned_dense_sweep_ragged_sizes(M, oracle, scheme, n):
    """Dense n <= 4096 with a commutator-free scheme runs planned batches on the persistent sweep kernel:
    sizes below the CTA count (CTAs without rows), ragged row/column tails, n = 1 (gamma = 0: that exponential
    takes the stepwise path inside the batch).  Against the oracle and against the per-iteration kernels."""
    cfg = W.scaled(W.CONFIGS["cfg2"], n, 5)
    H0, H1, psi0, f = W.build(cfg)
    ref, riters = oracle.magnus_integrate(H0.numpy(), H1.numpy(), f, scheme, cfg.t0, cfg.t_end, cfg.nsteps, psi0.numpy(), cfg.tol)
    res = {}
    for ck in (0, 1):
        psi = psi0.to(DEV).clone()
        with M.magnus_create(H0.to(DEV), H1.to(DEV), f, scheme, tol=cfg.tol, csr_kernel=ck) as h:
            if ck == 0 and n > 1:
                assert h.describe()["leja_kernel"] == "dense_leja_sweep_kernel"
            st = h.integrate(cfg.t0, cfg.t_end, cfg.nsteps, psi)
        res[ck] = (st["iters"], host(psi))
        assert np.array_equal(st["iters"], riters)
        assert relerr(host(psi), ref) <= 1e-9
    assert relerr(res[0][1], res[1][1]) <= 1e-13


@pytest.mark.parametrize("kind", ["xxz", "dense"])
def test_planned_batch_with_substeps_and_nonconvergence(M, oracle, kind):
    """A theta_max between the smallest and the largest theta of the run: some exponentials need sub-steps (the
    planner hands those to the stepwise path and resumes behind them), the rest run as jobs.  Same counts and
    psi as the all-stepwise run.  Then tol = 1e-300: the first job fails, the stepwise redo reports ENOCONV and
    psi is still the initial state."""
    cfg = W.scaled(W.CONFIGS["cfg1"], 8, 12) if kind == "xxz" else W.scaled(W.CONFIGS["cfg2"], 300, 12)
    H0, H1, psi0, f = W.build(cfg)
    d0, d1 = H0.to(DEV), H1.to(DEV)
    psi = psi0.to(DEV).clone()
    with M.magnus_create(d0, d1, f, "cf4", tol=cfg.tol, csr_kernel=1) as h:
        thetas = sorted(abs(i["theta"]) for s in range(cfg.nsteps) for i in h.step(cfg.t0 + s * cfg.tau, cfg.tau, psi))
    theta_max = 0.5 * (thetas[len(thetas) // 2 - 1] + thetas[len(thetas) // 2])
    assert thetas[0] < theta_max < thetas[-1]
    res = {}
    for ck in (0, 1):
        psi = psi0.to(DEV).clone()
        with M.magnus_create(d0, d1, f, "cf4", tol=cfg.tol, csr_kernel=ck, theta_max=theta_max) as h:
            infos = [i for s in range(0, cfg.nsteps, 4) for i in [h.integrate(cfg.t0 + s * cfg.tau, cfg.t0 + (s + 4) * cfg.tau, 4, psi)]]
        res[ck] = (np.concatenate([i["iters"] for i in infos]), host(psi))
    assert np.array_equal(res[0][0], res[1][0]) and relerr(res[0][1], res[1][1]) <= 1e-13
    o0, o1 = (oracle.CsrHost.of(H0), oracle.CsrHost.of(H1)) if kind == "xxz" else (H0.numpy(), H1.numpy())
    ref, _ = oracle.magnus_integrate(o0, o1, f, "cf4", cfg.t0, cfg.t_end, cfg.nsteps, psi0.numpy(), cfg.tol)
    assert relerr(res[0][1], ref) <= 1e-9          # sub-steps change the counts, not the result
    psi = psi0.to(DEV).clone()
    with M.magnus_create(d0, d1, f, "cf4", tol=1e-300) as h:   # planned path: the first job fails, then the stepwise redo
        with pytest.raises(M.MagnusError) as e:
            h.integrate(cfg.t0, cfg.t0 + 6.0, 3, psi)    # tau = 2: theta about 10, |d_128| about 1e-88 > tol
    assert e.value.code == -4 and torch.equal(psi, psi0.to(DEV))


def test_planned_batch_longer_than_the_plan_capacity(M, oracle):
    """1500 CF4 steps = 3000 exponentials > the ring of job slots (256) and two plans of 1365 steps: counts
    and psi against the oracle."""
    cfg = W.scaled(W.CONFIGS["cfg1"], 6, 1500)
    psi, st, ref, riters = run_config(M, oracle, cfg, "cf4")
    assert st["n_exp"] == 3000 and np.array_equal(st["iters"], riters)
    assert relerr(psi, ref) <= 1e-9


# ------------------------------------------------------------------ shortcut: matrix-free XXZ chain
def xxz_with_couplings(N, jxy, jz, hx):
    """The generator's H0, H1 rescaled to couplings (jxy, jz, hx): H0's diagonal is 0.5 (N - 2k), its off-diagonal 2."""
    H0, H1 = xxz.xxz_h0(N), xxz.xxz_h1(N)
    rows = torch.repeat_interleave(torch.arange(H0.n), (H0.row_ptr[1:] - H0.row_ptr[:-1]).long())
    diag = H0.col_idx.long() == rows
    v0 = torch.where(diag, H0.values * (jz / 0.5), H0.values * jxy)
    return xxz.CSR(H0.n, H0.row_ptr, H0.col_idx, v0), xxz.CSR(H1.n, H1.row_ptr, H1.col_idx, H1.values * hx)


@pytest.mark.parametrize("scheme", ["cf4", "cf4:3"])
@pytest.mark.parametrize("N,jxy,jz,hx,tau,nsteps", [(3, 1.0, 0.5, 1.0, 0.05, 3), (4, 1.0, 0.5, 1.0, 0.05, 3),
                                                    (5, -0.8, 0.4, 0.6, 0.05, 3), (6, 1.0, 0.5, 1.0, 0.05, 3),
                                                    (7, 0.7, -0.3, 1.3, 0.04, 3), (10, 1.0, 0.5, 1.0, 0.01, 10),
                                                    (13, 0.7, -0.3, 1.3, 0.03, 3), (16, 1.0, 0.5, 1.0, 0.05, 2)])
def test_shortcut_matrix_free_xxz(M, oracle, scheme, N, jxy, jz, hx, tau, nsteps):
    """`magnus_create_xxz`: the chain described by its couplings, no matrix in memory.  Against the oracle on the
    CSR matrices of the same model (identical counts, psi <= 1e-9) and against the library's own CSR path
    (psi <= 1e-12: same method, another summation order).  N <= 5: everything inside one warp (shuffles only)."""
    H0, H1 = xxz_with_couplings(N, jxy, jz, hx)
    psi0 = torch.from_numpy(rand_vec(1 << N, 31 + N))
    f = xxz.f_cos2t
    ref, riters = oracle.magnus_integrate(oracle.CsrHost.of(H0), oracle.CsrHost.of(H1), f, scheme, 0.1, 0.1 + tau * nsteps,
                                          nsteps, psi0.numpy(), 1e-12)
    psi = psi0.to(DEV).clone()
    with M.magnus_create_xxz(N, jxy, jz, hx, f, scheme, tol=1e-12) as h:
        d = h.describe()
        assert d["leja_kernel"] == "xxz_leja_iter_kernel" and d["bytes_per_iteration"] == 64 * (1 << N)
        st = h.integrate(0.1, 0.1 + tau * nsteps, nsteps, psi)
    assert np.array_equal(st["iters"], riters)
    assert relerr(host(psi), ref) <= 1e-9 and abs(np.linalg.norm(host(psi)) - 1) < 1e-10
    psi2 = psi0.to(DEV).clone()
    with M.magnus_create(H0.to(DEV), H1.to(DEV), f, scheme, tol=1e-12) as h:
        st2 = h.integrate(0.1, 0.1 + tau * nsteps, nsteps, psi2)
    assert np.array_equal(st["iters"], st2["iters"]) and relerr(host(psi), host(psi2)) <= 1e-12


def test_shortcut_matrix_free_xxz_refuses_commutator_schemes(M):
    for scheme in ("m4", "m6"):
        with pytest.raises(M.MagnusError) as e:
            M.magnus_create_xxz(10, 1.0, 0.5, 1.0, xxz.f_cos2t, scheme)
        assert e.value.code == -1
    with pytest.raises(M.MagnusError):
        M.magnus_create_xxz(2, 1.0, 0.5, 1.0, xxz.f_cos2t, "cf4")


# ------------------------------------------------------------------ shortcut: tight spectral interval
@pytest.mark.parametrize("name,size,nsteps,scheme,m", [("cfg2", 33, 3, "cf4", 8), ("cfg2", 300, 3, "cf4", 8),
                                                       ("cfg2", 300, 2, "m4", 6), ("cfg2", 1237, 2, "cf4:3", 8),
                                                       ("cfg2", 5000, 1, "cf4", 8), ("cfg1", 10, 5, "cf4", 8),
                                                       ("cfg1", 10, 5, "m4", 8), ("cfg3", 14, 2, "cf4", 12)])
def test_shortcut_tight_interval_vs_oracle(M, oracle, name, size, nsteps, scheme, m):
    """MAGNUS_SHORTCUT_TIGHT_INTERVAL: the interval of every exponential from m Lanczos steps started at psi.
    Against the oracle in the same mode (its own Lanczos, Jacobi eigenvalues): identical snapped intervals,
    identical iteration counts, psi <= 1e-9; on dense input fewer Leja iterations than with Gershgorin."""
    cfg = W.scaled(W.CONFIGS[name], size, nsteps)
    H0, H1, psi0, f = W.build(cfg)
    if cfg.kind == "xxz":
        o0, o1 = oracle.CsrHost.of(H0), oracle.CsrHost.of(H1)
    else:
        o0, o1 = H0.numpy(), H1.numpy()
    d0, d1 = H0.to(DEV), H1.to(DEV)
    with oracle.tight_interval(m):
        ref, riters = oracle.magnus_integrate(o0, o1, f, scheme, cfg.t0, cfg.t_end, cfg.nsteps, psi0.numpy(), cfg.tol)
        _, rinfo = oracle.magnus_step(o0, o1, f, scheme, cfg.t0, cfg.tau, psi0.numpy(), cfg.tol)
    psi = psi0.to(DEV).clone()
    with M.magnus_create(d0, d1, f, scheme, tol=cfg.tol, shortcuts=M.SHORTCUT_TIGHT_INTERVAL, lanczos_steps=m) as h:
        info = h.step(cfg.t0, cfg.tau, psi0.to(DEV).clone())
        st = h.integrate(cfg.t0, cfg.t_end, cfg.nsteps, psi)
    for gi, ri in zip(info, rinfo):
        assert gi["a"] == ri["a"] and gi["b"] == ri["b"] and gi["theta"] == ri["theta"] and gi["iters"] == ri["iters"]
    assert np.array_equal(st["iters"], riters) and st["lanczos_matvecs"] == m * len(riters)
    assert relerr(host(psi), ref) <= 1e-9 and abs(np.linalg.norm(host(psi)) - 1) < 1e-10
    if cfg.kind == "dense":
        psi2 = psi0.to(DEV).clone()
        with M.magnus_create(d0, d1, f, scheme, tol=cfg.tol) as h:
            st2 = h.integrate(cfg.t0, cfg.t_end, cfg.nsteps, psi2)
        assert st["total_matvecs"] < st2["total_matvecs"]
        assert relerr(host(psi), host(psi2)) <= 1e-9           # two intervals, one exponential


# ------------------------------------------------------------------ medium CSR: cooperative whole-sweep kernel
@pytest.mark.parametrize("scheme", ["cf4", "m4"])
@pytest.mark.parametrize("N,nsteps", [(11, 4), (13, 3), (15, 2), (16, 1)])
def test_medium_csr_sweep_kernel(M, oracle, scheme, N, nsteps):
    """1024 < n <= 65536: planned batches on the persistent cooperative CSR sweep kernel (rows partitioned over the SMs,
    w through L2 with one grid barrier per iteration).  Against the oracle (counts equal, psi <= 1e-9) and against the
    per-iteration kernels of the stepwise path (csr_kernel = 1)."""
    cfg = W.scaled(W.CONFIGS["cfg3"], N, nsteps)
    H0, H1, psi0, f = W.build(cfg)
    ref, riters = oracle.magnus_integrate(oracle.CsrHost.of(H0), oracle.CsrHost.of(H1), f, scheme, cfg.t0, cfg.t_end,
                                          cfg.nsteps, psi0.numpy(), cfg.tol)
    res = {}
    for ck in (0, 1):
        psi = psi0.to(DEV).clone()
        with M.magnus_create(H0.to(DEV), H1.to(DEV), f, scheme, tol=cfg.tol, csr_kernel=ck) as h:
            if ck == 0:
                assert h.describe()["leja_kernel"] == "csr_leja_sweep_mid_kernel"
            st = h.integrate(cfg.t0, cfg.t_end, cfg.nsteps, psi)
        assert np.array_equal(st["iters"], riters) and relerr(host(psi), ref) <= 1e-9
        res[ck] = host(psi)
    assert relerr(res[0], res[1]) <= 1e-13
    if N == 11:      # forced on a size the cluster kernel would take, and the cluster kernel forced... by size: N = 10
        cfg10 = W.scaled(W.CONFIGS["cfg1"], 10, 6)
        H0, H1, psi0, f = W.build(cfg10)
        out = {}
        for ck in (0, 7):
            psi = psi0.to(DEV).clone()
            with M.magnus_create(H0.to(DEV), H1.to(DEV), f, scheme, tol=cfg10.tol, csr_kernel=ck) as h:
                assert h.describe()["leja_kernel"] == ("csr_leja_sweep_mid_kernel" if ck == 7 else "csr_leja_sweep_small_kernel")
                st = h.integrate(cfg10.t0, cfg10.t_end, cfg10.nsteps, psi)
            out[ck] = (st["iters"], host(psi))
        assert np.array_equal(out[0][0], out[7][0]) and relerr(out[0][1], out[7][1]) <= 1e-13


def test_medium_csr_sweep_many_short_jobs_even_counts(M, oracle):
    """Stress of the job-to-job hand-over inside ONE cooperative launch: 1200 exponentials of a few iterations each
    (small tau), most of them stopping at an even degree -- the case in which the stop test of job e and the
    ||psi||^2 reduction of job e + 1 used to share a partials buffer with no grid barrier in between (a fast CTA could
    overwrite its slot while a slow one was still summing).  Counts equal to the oracle's, psi <= 1e-9, and three
    runs give the same bits."""
    N, nsteps = 11, 600
    cfg = W.scaled(W.CONFIGS["cfg3"], N, nsteps)
    H0, H1, psi0, f = W.build(cfg)
    t_end = cfg.t0 + nsteps * 1e-3          # 6 iterations per exponential at this tau
    ref, riters = oracle.magnus_integrate(oracle.CsrHost.of(H0), oracle.CsrHost.of(H1), f, "cf4", cfg.t0, t_end, nsteps,
                                          psi0.numpy(), cfg.tol)
    assert np.count_nonzero(np.asarray(riters) % 2 == 0) >= len(riters) // 2
    outs = []
    with M.magnus_create(H0.to(DEV), H1.to(DEV), f, "cf4", tol=cfg.tol) as h:
        assert h.describe()["leja_kernel"] == "csr_leja_sweep_mid_kernel"
        for _ in range(3):
            psi = psi0.to(DEV).clone()
            st = h.integrate(cfg.t0, t_end, nsteps, psi)
            assert np.array_equal(st["iters"], riters)
            outs.append(host(psi))
    assert relerr(outs[0], ref) <= 1e-9
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])


def test_medium_csr_sweep_general_matrix_and_expmv(M, oracle):
    """The same kernel on a general (non-XXZ) Hermitian CSR matrix with empty and long rows, through leja_expmv
    (one-job launch, out != in), and its non-convergence report (input untouched when in place)."""
    n = 9001
    S = random_sparse_hermitian(n, 0.0006, 9, long_row=(17, 1500))
    Mh = oracle.CsrHost(n, S.indptr.astype(np.int32), S.indices.astype(np.int32), S.data.astype(complex))
    v = rand_vec(n, 41)
    ref, rinfo = oracle.leja_expmv(Mh, v, 0.02, 1e-12)
    vi = torch.from_numpy(v).to(DEV)
    vo = torch.empty_like(vi)
    info = M.leja_expmv(csr_from_scipy(S), vi, vo, 0.02, 1e-12)
    assert info["iters"] == rinfo["iters"] and info["a"] == rinfo["a"] and info["b"] == rinfo["b"]
    assert relerr(host(vo), ref) <= 1e-12 and torch.equal(vi, torch.from_numpy(v).to(DEV))
    keep = vi.clone()
    with pytest.raises(M.MagnusError) as e:
        M.leja_expmv(csr_from_scipy(S), vi, vi, 3.0, 1e-300)
    assert e.value.code == -4 and torch.equal(vi, keep)


def test_runs_on_a_non_blocking_side_stream(M):
    """Everything a handle enqueues (workspace initialisation, layouts, interval kernels, job uploads, sweeps) is
    ordered on the caller's stream -- also a torch side stream, which does not synchronise with the legacy default
    stream.  Same bits as on the default stream (the path is deterministic), for the cluster kernel, the cooperative
    CSR and dense sweep kernels and the per-iteration kernels."""
    cases = [("cfg1", 10, 8, "cf4"), ("cfg1", 10, 8, "m4"), ("cfg3", 13, 3, "cf4"), ("cfg2", 300, 4, "cf4"),
             ("cfg2", 300, 3, "m4"), ("cfg3", 18, 2, "cf4")]
    side = torch.cuda.Stream()
    for name, size, nsteps, scheme in cases:
        cfg = W.scaled(W.CONFIGS[name], size, nsteps)
        H0, H1, psi0, f = W.build(cfg)
        d0, d1 = H0.to(DEV), H1.to(DEV)
        ref = psi0.to(DEV).clone()
        with M.magnus_create(d0, d1, f, scheme, tol=cfg.tol) as h:
            st0 = h.integrate(cfg.t0, cfg.t_end, cfg.nsteps, ref)
        torch.cuda.synchronize()
        with torch.cuda.stream(side):
            psi = psi0.to(DEV).clone()
            side.synchronize()
            for rep in range(3):                      # fresh handles: their initialisation must not race the first launch
                psi.copy_(psi0.to(DEV))
                with M.magnus_create(d0, d1, f, scheme, tol=cfg.tol, stream=side) as h:
                    st1 = h.integrate(cfg.t0, cfg.t_end, cfg.nsteps, psi)
                assert np.array_equal(st0["iters"], st1["iters"]) and torch.equal(psi, ref), (name, size, scheme, rep)


def test_shortcuts_combined_matrix_free_and_tight_interval(M, oracle):
    """The two shortcuts together: the matrix-free chain with its interval from Lanczos (the fused iteration kernel of
    the chain serves as the Lanczos mat-vec).  Same intervals and counts as the CSR path in the same mode, and as the
    oracle in the same mode."""
    N, m = 12, 10
    H0, H1 = xxz.xxz_h0(N), xxz.xxz_h1(N)
    psi0 = torch.from_numpy(rand_vec(1 << N, 77))
    f = xxz.f_cos2t
    with oracle.tight_interval(m):
        ref, riters = oracle.magnus_integrate(oracle.CsrHost.of(H0), oracle.CsrHost.of(H1), f, "cf4", 0.0, 0.15, 3, psi0.numpy(), 1e-12)
    out = {}
    for kind in ("xxz", "csr"):
        psi = psi0.to(DEV).clone()
        opts = dict(tol=1e-12, shortcuts=M.SHORTCUT_TIGHT_INTERVAL, lanczos_steps=m)
        h = M.magnus_create_xxz(N, 1.0, 0.5, 1.0, f, "cf4", **opts) if kind == "xxz" else \
            M.magnus_create(H0.to(DEV), H1.to(DEV), f, "cf4", **opts)
        with h:
            info = h.step(0.0, 0.05, psi0.to(DEV).clone())
            st = h.integrate(0.0, 0.15, 3, psi)
        out[kind] = (info, st["iters"], host(psi))
        assert np.array_equal(st["iters"], riters) and relerr(host(psi), ref) <= 1e-9 and st["lanczos_matvecs"] == 6 * m
    for a, b in zip(out["xxz"][0], out["csr"][0]):
        assert a["a"] == b["a"] and a["b"] == b["b"] and a["iters"] == b["iters"]
    assert relerr(out["xxz"][2], out["csr"][2]) <= 1e-12


@pytest.mark.parametrize("scheme", ["cf4", "m4"])
def test_shortcut_real_values(M, oracle, scheme):
    """MAGNUS_SHORTCUT_REAL_VALUES on a large CSR chain (N = 18: the offset-slot copy keeps the real parts only): the
    same bits as the mandated path, counts equal to the oracle's; on an operator WITH imaginary parts the flag changes
    nothing (complex storage stays)."""
    cfg = W.scaled(W.CONFIGS["cfg3"], 18, 2)
    H0, H1, psi0, f = W.build(cfg)
    ref, riters = oracle.magnus_integrate(oracle.CsrHost.of(H0), oracle.CsrHost.of(H1), f, scheme, cfg.t0, cfg.t_end,
                                          cfg.nsteps, psi0.numpy(), cfg.tol)
    d0, d1 = H0.to(DEV), H1.to(DEV)
    out = {}
    for sc in (0, M.SHORTCUT_REAL_VALUES):
        psi = psi0.to(DEV).clone()
        with M.magnus_create(d0, d1, f, scheme, tol=cfg.tol, shortcuts=sc) as h:
            d = h.describe()
            st = h.integrate(cfg.t0, cfg.t_end, cfg.nsteps, psi)
        out[sc] = (d, st["iters"], psi)
        assert np.array_equal(st["iters"], riters) and relerr(host(psi), ref) <= 1e-9
    assert torch.equal(out[0][2], out[M.SHORTCUT_REAL_VALUES][2])
    assert "real values" in out[M.SHORTCUT_REAL_VALUES][0]["leja_kernel"] and "real values" not in out[0][0]["leja_kernel"]
    assert out[0][0]["bytes_per_iteration"] - out[M.SHORTCUT_REAL_VALUES][0]["bytes_per_iteration"] == 8 * out[0][0]["entries"]
    # an operator with imaginary parts: i (|r><r'| - |r'><r|)-type entries from a complex phase on H1
    H1c = xxz.CSR(H1.n, H1.row_ptr, H1.col_idx, H1.values * torch.where(H1.col_idx.long() > torch.repeat_interleave(
        torch.arange(H1.n), (H1.row_ptr[1:] - H1.row_ptr[:-1]).long()), torch.tensor(1j), torch.tensor(-1j)))
    with M.magnus_create(d0, H1c.to(DEV), f, "cf4", tol=cfg.tol, shortcuts=M.SHORTCUT_REAL_VALUES) as h:
        assert "real values" not in h.describe()["leja_kernel"]
        psi = psi0.to(DEV).clone()
        st = h.integrate(cfg.t0, cfg.t0 + cfg.tau, 1, psi)
    refc, ritc = oracle.magnus_integrate(oracle.CsrHost.of(H0), oracle.CsrHost.of(H1c), f, "cf4", cfg.t0, cfg.t0 + cfg.tau, 1,
                                         psi0.numpy(), cfg.tol)
    assert np.array_equal(st["iters"], ritc) and relerr(host(psi), refc) <= 1e-9
