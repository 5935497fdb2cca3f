"""Pins of the oracle's counterpart of the tight-interval shortcut (reading ti): the Lanczos interval.

None of these re-types the oracle's recurrence: they check what DEFINES a Lanczos tridiagonalisation (its moments),
exactness on an invariant subspace, interlacing, and the end-to-end accuracy of the exponential on the interval."""
import numpy as np
import pytest

from oracle import oracle as O
from workloads import dense, xxz


def rand_herm(n, seed):
    r = np.random.default_rng(seed)
    G = r.normal(size=(n, n)) + 1j * r.normal(size=(n, n))
    return (G + G.conj().T) / (2.0 * np.sqrt(n))


def tri(al, be):
    return np.diag(al) + np.diag(be[:-1], 1) + np.diag(be[:-1], -1)


@pytest.mark.parametrize("n,m,seed", [(30, 5, 1), (64, 8, 2), (200, 12, 3)])
def test_lanczos_moments_define_T(n, m, seed):
    """e_1^T T^p e_1 = q_1^H M^p q_1 for p <= 2m - 1 -- the property that characterises the Lanczos T."""
    M = rand_herm(n, seed)
    v = np.random.default_rng(seed + 10).normal(size=n) + 1j * np.random.default_rng(seed + 20).normal(size=n)
    (a, b), al, be = O.lanczos_interval(M, v, m)
    assert len(al) == m
    T = tri(al, be)
    q = v / np.linalg.norm(v)
    x, e = q.copy(), np.eye(m)[0]
    Tp = np.eye(m)
    for p in range(1, 2 * m):
        x = M @ x
        Tp = Tp @ T
        lhs, rhs = Tp[0, 0], np.vdot(q, x).real
        assert abs(lhs - rhs) <= 1e-10 * max(1.0, abs(rhs)), (p, lhs, rhs)
    ritz = np.linalg.eigvalsh(T)
    assert abs(a - (ritz[0] - be[-1])) <= 1e-12 * max(1.0, abs(a)) and abs(b - (ritz[-1] + be[-1])) <= 1e-12 * max(1.0, abs(b))
    ev = np.linalg.eigvalsh(M)
    assert ev[0] - 1e-12 <= ritz[0] and ritz[-1] <= ev[-1] + 1e-12      # Ritz values lie inside the spectrum
    assert a <= ev[0] and ev[-1] <= b                                   # widened by the residual norm: contains it (seeded case)


def test_lanczos_is_exact_on_an_invariant_subspace():
    """Diagonal M, v supported on 4 distinct eigenvalues: the process stops after 4 steps (beta_4 = 0) with the exact
    extreme eigenvalues; n = 1: one step, interval = the entry."""
    d = np.array([3.0, -1.5, 0.25, 7.0, 100.0, -50.0])
    M = np.diag(d).astype(complex)
    v = np.array([1.0, 2.0, -1.0, 0.5, 0.0, 0.0], dtype=complex)
    (a, b), al, be = O.lanczos_interval(M, v, 12)
    assert len(al) == 4 and be[-1] <= 1e-12 * 7.0
    assert abs(a - (-1.5)) < 1e-11 and abs(b - 7.0) < 1e-11
    (a, b), al, be = O.lanczos_interval(np.array([[2.5 + 0j]]), np.array([1j]), 5)
    assert len(al) == 1 and a == b == 2.5
    (a, b), al, be = O.lanczos_interval(M, np.zeros(6, dtype=complex), 5)          # v = 0: no step taken
    assert len(al) == 0


@pytest.mark.parametrize("kind,size", [("dense", 48), ("dense", 64), ("xxz", 6)])
def test_expmv_on_the_tight_interval(kind, size):
    """exp(-ihM)v on the Lanczos interval against the eigendecomposition (same bar as on the Gershgorin interval),
    and never more iterations than on the Gershgorin interval for these matrices."""
    if kind == "dense":
        M = (dense.dense_h0(size) + 0.7 * dense.dense_h1(size)).numpy()
    else:
        M = (xxz.xxz_h0(size).to_scipy() + 0.4 * xxz.xxz_h1(size).to_scipy()).toarray()
    n = M.shape[0]
    v = np.random.default_rng(5).normal(size=n) + 1j * np.random.default_rng(6).normal(size=n)
    v /= np.linalg.norm(v)
    w, U = np.linalg.eigh(M)
    for h in (0.3, -1.1):
        ref = U @ (np.exp(-1j * h * w) * (U.conj().T @ v))
        out_g, info_g = O.leja_expmv(M, v, h, 1e-12)
        with O.tight_interval(8):
            out_t, info_t = O.leja_expmv(M, v, h, 1e-12)
        assert np.linalg.norm(out_t - ref) <= 1e-11 and np.linalg.norm(out_g - ref) <= 1e-11
        assert info_t["iters"] <= info_g["iters"] and info_t["b"] - info_t["a"] <= info_g["b"] - info_g["a"]
    out_again, info_again = O.leja_expmv(M, v, 0.3, 1e-12)                          # the mode is off again outside the block
    assert info_again["a"] == O.gershgorin(M)[1][0]


def test_tight_interval_never_reaches_beyond_gershgorin():
    """Reading ti: the Lanczos interval [theta_min - beta_m, theta_max + beta_m] is an estimate, not an enclosure; on a
    DIAGONAL matrix Gershgorin is exact, so every bit of the widening by beta_m lies outside the spectrum.  The interval
    leja_expmv uses in tight mode is the intersection: equal to Gershgorin's where Lanczos sticks out, tighter where
    the start vector does not see a part of the spectrum -- and the result is still exp(-ihM)v."""
    n = 64
    d = np.linspace(-1.0, 1.0, n)
    M = np.diag(d).astype(complex)
    r = np.random.default_rng(11)
    v = r.normal(size=n) + 1j * r.normal(size=n)
    v /= np.linalg.norm(v)
    (la, lb), _, _ = O.lanczos_interval(M, v, 8)
    assert la < -1.0 and lb > 1.0                              # the raw estimate does stick out on both sides
    _, info_g = O.leja_expmv(M, v, 0.7, 1e-12)
    with O.tight_interval(8):
        out, info_t = O.leja_expmv(M, v, 0.7, 1e-12)
    assert info_t["a"] == info_g["a"] and info_t["b"] == info_g["b"]
    assert np.linalg.norm(out - np.exp(-0.7j * d) * v) <= 1e-12
    v2 = v.copy()
    v2[n // 2:] = 0.0                                          # sees only the eigenvalues in [-1, -1/63]
    v2 /= np.linalg.norm(v2)
    (la2, lb2), _, _ = O.lanczos_interval(M, v2, 8)
    assert la2 < -1.0 and lb2 < 0.5
    with O.tight_interval(8):
        out2, info_2 = O.leja_expmv(M, v2, 0.7, 1e-12)
    assert info_2["a"] == info_g["a"] and info_2["b"] < info_g["b"]
    assert np.linalg.norm(out2 - np.exp(-0.7j * d) * v2) <= 1e-12
