"""GPU test (-m gpu) of magnus_leja_iteration_dense_noalloc, the entry point for callers that cannot allocate.

Some users of this library run where a cudaMalloc is not an option: their process has handed all device memory to
a pool (PyTorch's caching allocator is the usual one), they work under a fixed memory budget inside somebody
else's CUDA context, or they sit in a loop with a latency bound that the driver-wide locks of cudaMalloc / cudaFree
would break.  For them the library keeps the scratch of the fused dense Leja iteration (per-block partial sums and
the last-block ticket) in a static device array of 65,792 bytes, which limits n to 32768 and forbids overlapping
calls on one GPU.

What is checked, against the EXISTING path (magnus_leja_iteration on the same dense matrix, which allocates its
workspace) and against the CPU oracle: w_out, p and the two norms on TWO calls in a row -- the second call finds the
first one's partial sums and ticket in the shared scratch, and a shorter problem after a longer one finds stale
partial slots beyond its own grid -- plus the size limit and argument errors.  The file name sorts last on purpose:
`pytest -x` stops at the first failure, and a failure here must not hide the parity tests.  The test does not depend
on what ran before it (it passes alone in a fresh process and after the whole suite): the entry point clears what it
needs itself.
"""
import numpy as np
import pytest
import torch

from workloads import dense

pytestmark = pytest.mark.gpu

DEV = "cuda"


@pytest.fixture(scope="module")
def M():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1709_06483_b200 as pkg
    pkg.lib()
    return pkg


def rand_vec(n, seed):
    r = np.random.default_rng(seed)
    v = r.normal(size=n) + 1j * r.normal(size=n)
    return v / np.linalg.norm(v)


def run_both(M, oracle, n, seed, inv_gamma, shift, d, strided=False):
    """One iteration through the allocating path and through the no-alloc entry point; asserts they agree with
    each other (bit for bit: same per-row arithmetic, same reduction order for n <= 32768) and with the oracle
    (tolerance of test_fused_iteration_dense: 8 max(n,16) eps elementwise, 1e-12 relative on the norms)."""
    H = dense.random_hermitian(n, stream=40 + seed)
    w, p = rand_vec(n, 100 + seed), rand_vec(n, 200 + seed)
    y = oracle.matvec(H.numpy(), w)
    wn = inv_gamma * y - shift * w
    pn = p + d * wn

    Hd = H.to(DEV)
    if strided:                       # rows with a leading dimension > n
        big = torch.zeros((n, n + 5), dtype=torch.complex128, device=DEV)
        big[:, :n] = Hd
        Hd = big[:, :n]
    wi = torch.from_numpy(w).to(DEV)
    wo_a, p_a = torch.zeros_like(wi), torch.from_numpy(p).to(DEV)
    sw_a, sp_a, _ = M.magnus_leja_iteration(Hd, None, 0.0, wi, wo_a, p_a, inv_gamma, shift, d)

    wo_b, p_b = torch.zeros_like(wi), torch.from_numpy(p).to(DEV)
    sums = torch.full((2,), float("nan"), dtype=torch.float64, device=DEV)
    M.magnus_leja_iteration_dense_noalloc(Hd, wi, wo_b, p_b, inv_gamma, shift, d, sums)
    torch.cuda.synchronize()
    sw_b, sp_b = sums.cpu().tolist()

    tol = 8 * max(n, 16) * np.finfo(float).eps
    for wo, pp, sw, sp in ((wo_a, p_a, sw_a, sp_a), (wo_b, p_b, sw_b, sp_b)):
        assert np.max(np.abs(wo.cpu().numpy() - wn)) <= tol * max(np.max(np.abs(wn)), np.max(np.abs(w)))
        assert np.max(np.abs(pp.cpu().numpy() - pn)) <= tol * max(np.max(np.abs(pn)), 1e-3)
        assert abs(sw - np.sum(np.abs(wn) ** 2)) <= 1e-12 * np.sum(np.abs(wn) ** 2)
        assert abs(sp - np.sum(np.abs(pn) ** 2)) <= 1e-12 * np.sum(np.abs(pn) ** 2)
    assert torch.equal(wo_a, wo_b) and torch.equal(p_a, p_b)
    assert sw_a == sw_b and sp_a == sp_b


def test_noalloc_two_calls_in_a_row_match_the_allocating_path(M, oracle):
    # a longer problem first, then a shorter one (stale partial slots beyond its grid), then a ragged size again
    run_both(M, oracle, 1237, 1, 0.11, -0.9, 0.02 + 0.5j)
    run_both(M, oracle, 33, 2, 0.7, 0.25, -0.3 + 0.1j)
    run_both(M, oracle, 500, 3, 0.05, 1.3, 0.4 - 0.2j, strided=True)
    run_both(M, oracle, 1, 4, 1.0, 0.0, 1.0)


def test_noalloc_same_buffers_twice_gives_the_next_iterate(M, oracle):
    """Two consecutive enqueues on one stream without a host synchronisation in between (the way the recurrence
    w <- Mw/gamma - shift w, p += d w runs): the second launch must wait for the first one's ticket and sums."""
    n = 777
    H = dense.random_hermitian(n, stream=51)
    w0, p0 = rand_vec(n, 7), rand_vec(n, 8)
    ig, sh, d1, d2 = 0.3, -0.4, 0.2 + 0.1j, -0.05 + 0.3j
    w1 = ig * oracle.matvec(H.numpy(), w0) - sh * w0
    p1 = p0 + d1 * w1
    w2 = ig * oracle.matvec(H.numpy(), w1) - sh * w1
    p2 = p1 + d2 * w2
    Hd = H.to(DEV)
    a, b, pd = torch.from_numpy(w0).to(DEV), torch.zeros(n, dtype=torch.complex128, device=DEV), torch.from_numpy(p0).to(DEV)
    s1 = torch.zeros(2, dtype=torch.float64, device=DEV)
    s2 = torch.zeros(2, dtype=torch.float64, device=DEV)
    M.magnus_leja_iteration_dense_noalloc(Hd, a, b, pd, ig, sh, d1, s1)
    M.magnus_leja_iteration_dense_noalloc(Hd, b, a, pd, ig, sh, d2, s2)
    torch.cuda.synchronize()
    tol = 16 * n * np.finfo(float).eps
    assert np.max(np.abs(b.cpu().numpy() - w1)) <= tol * np.max(np.abs(w1))
    assert np.max(np.abs(a.cpu().numpy() - w2)) <= tol * np.max(np.abs(w2))
    assert np.max(np.abs(pd.cpu().numpy() - p2)) <= tol * np.max(np.abs(p2))
    assert abs(s1[0].item() - np.sum(np.abs(w1) ** 2)) <= 1e-12 * np.sum(np.abs(w1) ** 2)
    assert abs(s2[0].item() - np.sum(np.abs(w2) ** 2)) <= 1e-12 * np.sum(np.abs(w2) ** 2)
    assert abs(s2[1].item() - np.sum(np.abs(p2) ** 2)) <= 1e-12 * np.sum(np.abs(p2) ** 2)


def test_noalloc_refuses_sizes_beyond_the_static_scratch(M):
    """n above NOALLOC_MAX_N must come back as EINVAL with a message that names the limit -- before any pointer is
    touched, so tiny stand-in buffers are enough here."""
    from paper_1709_06483_b200 import binding as B
    assert B.NOALLOC_MAX_N == 32768
    t = torch.zeros(4, dtype=torch.complex128, device=DEV)
    t2, t3 = torch.zeros_like(t), torch.zeros_like(t)
    sums = torch.zeros(2, dtype=torch.float64, device=DEV)
    rc = B.lib().magnus_leja_iteration_dense_noalloc(B.NOALLOC_MAX_N + 1, t.data_ptr(), 0, t.data_ptr(), t2.data_ptr(),
                                                     t3.data_ptr(), 1.0, 0.0, 1.0, 0.0, None, sums.data_ptr())
    assert rc == B.EINVAL
    msg = B.lib().magnus_last_error().decode()
    assert "32768" in msg and "MAGNUS_NOALLOC_MAX_N" in msg
    # aliased vectors and a missing output are refused as well
    rc = B.lib().magnus_leja_iteration_dense_noalloc(2, t.data_ptr(), 0, t2.data_ptr(), t2.data_ptr(), t3.data_ptr(),
                                                     1.0, 0.0, 1.0, 0.0, None, sums.data_ptr())
    assert rc == B.EINVAL
    rc = B.lib().magnus_leja_iteration_dense_noalloc(2, t.data_ptr(), 0, t.data_ptr(), t2.data_ptr(), t3.data_ptr(),
                                                     1.0, 0.0, 1.0, 0.0, None, None)
    assert rc == B.EINVAL
