"""Pins for the oracle's Leja machinery (SURVEY.md 8(c) pins c-P1..c-P5).

Nothing here re-types the oracle's formulas: Leja points are checked against
their defining extremal property, divided differences against a 60-digit mpmath
recurrence and against the interpolation property, leja_expmv against
numpy.linalg.eigh, Gershgorin against eigenvalues and closed forms.
PAPER.md lines 169-190 (section 3) define the operations.
"""
import math

import mpmath
import numpy as np
import pytest

import leja_check
import workloads as W
from workloads import xxz


def rand_herm(n, seed, scale=1.0):
    r = np.random.default_rng(seed)
    G = r.normal(size=(n, n)) + 1j * r.normal(size=(n, n))
    return scale * (G + G.conj().T) / 2


def rand_vec(n, seed):
    r = np.random.default_rng(seed)
    v = r.normal(size=n) + 1j * r.normal(size=n)
    return v / np.linalg.norm(v)


def expm_eigh(M, h, v):
    lam, U = np.linalg.eigh(M)
    return U @ (np.exp(-1j * h * lam) * (U.conj().T @ v))


# ------------------------------------------------------------------ c-P2
def test_leja_points_closed_form_and_extremal_property(oracle):
    m = oracle.max_degree() + 1
    l = oracle.leja_points(m)
    assert m == 129
    assert l[0] == 2.0 and l[1] == -2.0 and l[2] == 0.0
    assert abs(l[3] - 2 / math.sqrt(3)) < 1e-15
    assert np.all(np.abs(l) <= 2.0) and len(set(l.tolist())) == m
    # prefix property: asking for fewer points gives the same sequence
    assert np.array_equal(oracle.leja_points(17), l[:17])
    grid = np.linspace(-2, 2, 100001)
    for k in range(3, m):
        prev = l[:k]
        # stationary point of the log-product (interior maximum)
        g = np.sum(1.0 / (l[k] - prev))
        assert abs(g) < 1e-9 * np.sum(1.0 / np.abs(l[k] - prev)), k
        if k <= 40:   # global maximum of prod |x - l_j| over [-2,2] (100001-point grid)
            logp = np.sum(np.log(np.abs(grid[:, None] - prev[None, :]) + 1e-300), axis=1)
            mine = np.sum(np.log(np.abs(l[k] - prev)))
            assert mine >= logp.max() - 1e-9, k
    # every k up to m_max = 128: l_k is the maximiser of the WINNING gap (per-gap golden section + 40-digit polish,
    # tests/leja_check.py -- a route independent of the oracle's bisection), and no other gap comes within 1e-7
    # in log: a wrong gap choice anywhere in the sequence fails here
    worst = leja_check.check_sequence(l)
    assert worst > 1e-4


def test_leja_check_rejects_a_wrong_gap(oracle):
    """Negative control for the pin above: the runner-up gap's stationary point is refused."""
    l = oracle.leja_points(60).copy()
    x, fx = leja_check.gap_maxima(l[:50])
    order = np.argsort(fx)
    l[50] = x[order[-2]]          # stationary, interior, distinct -- but not the global maximum
    with pytest.raises(AssertionError):
        leja_check.check_sequence(l[:51], first=50)


# ------------------------------------------------------------------ c-P1
def mp_divided_differences(theta, l, dps=60):
    mpmath.mp.dps = dps
    x = [mpmath.mpf(float(t)) for t in l]
    d = [mpmath.exp(-1j * mpmath.mpf(theta) * t) for t in x]
    for k in range(1, len(x)):
        for j in range(len(x) - 1, k - 1, -1):
            d[j] = (d[j] - d[j - 1]) / (x[j] - x[j - k])
    return d


@pytest.mark.parametrize("theta", [0.05, 0.7, 3.3, -3.3, 8.0, 16.0])
def test_divided_differences_vs_mpmath(oracle, theta):
    m = 70
    l = oracle.leja_points(m)
    d = oracle.divided_differences(theta, m)
    ref = mp_divided_differences(theta, l, dps=80)
    for k in range(m):
        r = complex(ref[k])
        # __float128 recurrence: absolute error ~1e-32 (reading c3), i.e. correctly
        # rounded wherever |d_k| > 1e-16 -- far below any stopping threshold
        assert abs(d[k] - r) <= 4e-16 * abs(r) + 1e-30, (k, d[k], r)
    assert np.all(np.abs(d) <= 1.0 + 1e-15)          # no hump (reading c3)


@pytest.mark.parametrize("theta", [0.3, 2.0, 7.5])
def test_newton_polynomial_reproduces_exponential(oracle, theta):
    m = 80
    l = oracle.leja_points(m)
    d = oracle.divided_differences(theta, m)
    x = np.linspace(-2, 2, 1000)
    p = np.zeros_like(x, dtype=complex)
    w = np.ones_like(x, dtype=complex)
    for k in range(m):
        p += d[k] * w
        w = w * (x - l[k])
    assert np.max(np.abs(p - np.exp(-1j * theta * x))) < 1e-13


def test_divided_differences_theta_zero(oracle):
    d = oracle.divided_differences(0.0, 10)
    assert d[0] == 1.0 and np.all(d[1:] == 0.0)


# ------------------------------------------------------------------ matvec
def test_matvec_is_row_major_not_transposed(oracle):
    n = 37
    M = rand_herm(n, 1) + 0.3j * np.triu(np.ones((n, n)), 1)   # deliberately NOT Hermitian
    w = rand_vec(n, 2)
    assert np.allclose(oracle.matvec(M, w), M @ w, rtol=0, atol=1e-13)
    assert not np.allclose(oracle.matvec(M, w), M.T @ w, atol=1e-3)
    H0 = xxz.xxz_h0(6)
    v = rand_vec(64, 3)
    assert np.allclose(oracle.matvec(oracle.CsrHost.of(H0), v), H0.to_scipy() @ v, atol=1e-13)


# ------------------------------------------------------------------ c-P5
def test_gershgorin_contains_spectrum_and_snap(oracle):
    for seed, n in [(0, 8), (1, 33), (2, 64)]:
        M = rand_herm(n, seed)
        (a, b), (sa, sb) = oracle.gershgorin(M)
        ev = np.linalg.eigvalsh(M)
        assert a <= ev.min() and ev.max() <= b
        R = np.sum(np.abs(M), axis=1) - np.abs(np.diag(M))
        assert math.isclose(a, np.min(np.diag(M).real - R), rel_tol=1e-13)
        assert math.isclose(b, np.max(np.diag(M).real + R), rel_tol=1e-13)
        assert sa <= a and sb >= b
        width = b - a
        delta = 2.0 ** (math.ceil(math.log2(width)) - 12)
        assert a - sa < delta and sb - b < delta
        assert (sa / delta).is_integer() and (sb / delta).is_integer()
    # a perturbation far below the grid does not move the snapped interval
    assert oracle.snap_interval(-3.3000000000001, 5.1) == oracle.snap_interval(-3.3000000000002, 5.1)
    assert oracle.snap_interval(-4.0, 4.0) == (-4.0, 4.0)


@pytest.mark.parametrize("N,g", [(4, 0.0), (6, 0.7), (10, -1.0), (10, 0.25)])
def test_gershgorin_xxz_closed_form(oracle, N, g):
    """[-(2.5+|g|)N, (1.5+|g|)N] for even N (pin c-P5), attained at the Neel rows."""
    H0, H1 = xxz.xxz_h0(N).to_scipy(), xxz.xxz_h1(N).to_scipy()
    M = (H0 + g * H1).tocsr()
    M.sort_indices()
    C = oracle.CsrHost(M.shape[0], M.indptr.astype(np.int32), M.indices.astype(np.int32), M.data.astype(complex))
    (a, b), _ = oracle.gershgorin(C)
    assert math.isclose(a, -(2.5 + abs(g)) * N, rel_tol=1e-14)
    assert math.isclose(b, (1.5 + abs(g)) * N, rel_tol=1e-14)


# ------------------------------------------------------------------ c-P3
@pytest.mark.parametrize("n,h,scale", [(1, 0.7, 1.0), (2, 1.0, 1.0), (16, 0.5, 1.0), (40, 0.05, 3.0), (64, 0.3, 0.7), (64, -0.3, 0.7)])
def test_expmv_dense_vs_eigendecomposition(oracle, n, h, scale):
    M = rand_herm(n, 10 + n, scale)
    v = rand_vec(n, 20 + n)
    y, info = oracle.leja_expmv(M, v, h, 1e-12)
    ref = expm_eigh(M, h, v)
    assert np.linalg.norm(y - ref) <= 1e-11          # 10 tol (pin c-P3)
    assert abs(np.linalg.norm(y) - 1) < 1e-10        # c-P4, north_star
    assert info["status"] == 0 and info["substeps"] >= 1


def test_expmv_csr_vs_eigendecomposition(oracle):
    N = 6
    H = (xxz.xxz_h0(N).to_scipy() + 0.37 * xxz.xxz_h1(N).to_scipy()).tocsr()
    H.sort_indices()
    C = oracle.CsrHost(64, H.indptr.astype(np.int32), H.indices.astype(np.int32), H.data.astype(complex))
    v = rand_vec(64, 5)
    for h in (0.01, 0.2, 1.0):
        y, info = oracle.leja_expmv(C, v, h, 1e-12)
        assert np.linalg.norm(y - expm_eigh(H.toarray(), h, v)) <= 1e-11
        yd, infod = oracle.leja_expmv(H.toarray(), v, h, 1e-12)
        assert info["iters"] == infod["iters"] and np.linalg.norm(y - yd) < 1e-14


def test_expmv_substeps_large_theta(oracle):
    """theta > theta_max = 16 forces sub-steps (reading c6); result still exact."""
    M = rand_herm(24, 3, 2.0)
    v = rand_vec(24, 4)
    (a, b), (sa, sb) = oracle.gershgorin(M)
    gamma = (sb - sa) / 4
    h = 40.0 / gamma
    y, info = oracle.leja_expmv(M, v, h, 1e-12)
    assert info["substeps"] == 3 and abs(info["theta"] - 40.0 / 3) < 1e-12
    assert np.linalg.norm(y - expm_eigh(M, h, v)) <= 3e-11


def test_expmv_diagonal_and_trivial_paths(oracle):
    x = np.array([-1.5, 0.2, 0.9, 3.0])
    v = rand_vec(4, 1)
    y, info = oracle.leja_expmv(np.diag(x).astype(complex), v, 0.8, 1e-12)
    assert np.allclose(y, np.exp(-0.8j * x) * v, atol=1e-12)
    # M = c I: gamma = 0, exact, zero iterations
    y, info = oracle.leja_expmv(2.5 * np.eye(3, dtype=complex), rand_vec(3, 2), 0.4, 1e-12)
    assert info["iters"] == 0 and np.allclose(y, np.exp(-1j) * rand_vec(3, 2), atol=1e-15)
    # h = 0: d_k = 0 for k >= 1, the two-term test needs exactly 2 iterations (pin c-P4)
    M = rand_herm(8, 5)
    y, info = oracle.leja_expmv(M, rand_vec(8, 6), 0.0, 1e-12)
    assert info["iters"] == 2 and np.array_equal(y, rand_vec(8, 6))


# ------------------------------------------------------------------ c-P4
def test_expmv_group_property_and_inverse(oracle):
    M = rand_herm(48, 7)
    v = rand_vec(48, 8)
    y1, _ = oracle.leja_expmv(M, v, 0.3, 1e-12)
    y2, _ = oracle.leja_expmv(M, y1, 0.45, 1e-12)
    y12, _ = oracle.leja_expmv(M, v, 0.75, 1e-12)
    assert np.linalg.norm(y2 - y12) < 5e-12
    back, _ = oracle.leja_expmv(M, y12, -0.75, 1e-12)
    assert np.linalg.norm(back - v) < 5e-12


def test_iteration_count_sanity(oracle):
    """Counts are 'parity unpinned' by the paper; only monotonicity is checked."""
    M = rand_herm(32, 11)
    v = rand_vec(32, 12)
    its_tol = [oracle.leja_expmv(M, v, 0.2, tol)[1]["iters"] for tol in (1e-4, 1e-8, 1e-12)]
    assert its_tol == sorted(its_tol) and its_tol[0] < its_tol[-1]
    its_h = [oracle.leja_expmv(M, v, h, 1e-12)[1]["iters"] for h in (0.01, 0.1, 0.5, 1.0)]
    assert its_h == sorted(its_h) and its_h[0] < its_h[-1]
    _, info = oracle.leja_expmv(M, v, 1.0, 1e-12)
    assert info["iters"] <= info["substeps"] * (2 * abs(info["theta"]) + 40)
