"""CPU tests of the product's host-side logic and of the C-ABI surface (-m "not gpu").

The shared library is built here by nvcc (cross-compiles without a GPU) and
loaded; only its host-side entry points are called.  They are checked against
mathematics (mpmath, defining properties, PAPER.md's printed coefficients) and
against the independent oracle.
"""
import ctypes
import math
import os
import re

import mpmath
import numpy as np
import pytest

import leja_check

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def M():
    from paper_1709_06483_b200 import build
    build.build()
    import paper_1709_06483_b200 as pkg
    pkg.lib()
    return pkg


def test_library_exports_every_declared_symbol(M):
    """Every function include/magnus.h declares is exported by the .so (no compute calls)."""
    hdr = open(os.path.join(ROOT, "include", "magnus.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(magnus_\w+|leja_expmv)\s*\(", hdr))
    names -= {"magnus_drive_fn"}
    assert {"magnus_create", "leja_expmv", "magnus_step", "magnus_integrate", "magnus_destroy"} <= names
    L = ctypes.CDLL(os.path.join(ROOT, "paper_1709_06483_b200", "libmagnus_b200.so"))
    for n in sorted(names):
        assert hasattr(L, n), n
    assert "sm_100a" in M.magnus_version()


def test_no_gpu_means_loud_failure_not_fallback(M):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    H = torch.eye(4, dtype=torch.complex128)
    v = torch.ones(4, dtype=torch.complex128)
    with pytest.raises(M.MagnusError) as e:
        M.leja_expmv(H, v, v.clone(), 0.1)
    assert e.value.code == -3 and "no CPU fallback" in str(e.value)
    with pytest.raises(M.MagnusError):
        M.magnus_create(H, H, lambda t: 1.0, "cf4")


def test_product_does_not_import_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_1709_06483_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".h", ".cuh")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "magnus_oracle" not in src, f


# ------------------------------------------------------------------ Leja points (c2)
def test_leja_points_defining_property(M):
    l = M.magnus_host_leja_points(129)
    assert l[0] == 2.0 and l[1] == -2.0 and l[2] == 0.0 and abs(l[3] - 2 / math.sqrt(3)) < 1e-15
    assert np.all(np.abs(l) <= 2.0) and len(set(l.tolist())) == 129
    grid = np.linspace(-2, 2, 40001)
    for k in range(4, 129):
        prev = l[:k]
        g = np.sum(1.0 / (l[k] - prev))
        assert abs(g) < 1e-9 * np.sum(1.0 / np.abs(l[k] - prev)), k
        if k <= 32:
            logp = np.sum(np.log(np.abs(grid[:, None] - prev[None, :]) + 1e-300), axis=1)
            assert np.sum(np.log(np.abs(l[k] - prev))) >= logp.max() - 1e-9, k
    # all k <= 128: the winning gap and its maximiser, by a route independent of the library's Newton iteration
    assert leja_check.check_sequence(l) > 1e-4


def test_leja_points_agree_with_oracle(M, oracle):
    assert np.max(np.abs(M.magnus_host_leja_points(129) - oracle.leja_points(129))) < 1e-14


# ------------------------------------------------------------------ divided differences (c3)
def mp_dd(theta, l, dps=80):
    mpmath.mp.dps = dps
    x = [mpmath.mpf(float(t)) for t in l]
    d = [mpmath.exp(-1j * mpmath.mpf(theta) * t) for t in x]
    for k in range(1, len(x)):
        for j in range(len(x) - 1, k - 1, -1):
            d[j] = (d[j] - d[j - 1]) / (x[j] - x[j - k])
    return d


@pytest.mark.parametrize("theta", [0.05, 0.7, -3.3, 8.0, 16.0])
def test_divided_differences_vs_mpmath(M, theta):
    m = 64
    l = M.magnus_host_leja_points(m)
    d = M.magnus_host_divided_differences(theta, m)
    ref = mp_dd(theta, l)
    for k in range(m):
        r = complex(ref[k])
        if abs(r) > 1e-17:      # full relative accuracy down to far below any stopping threshold
            assert abs(d[k] - r) <= 5e-16 * abs(r), (k, d[k], r)


@pytest.mark.parametrize("theta", [0.0, 0.1, 2.5, 12.0])
def test_divided_differences_prefix_and_oracle(M, oracle, theta):
    full = M.magnus_host_divided_differences(theta, 129)
    short = M.magnus_host_divided_differences(theta, 40)
    assert np.array_equal(full[:40], short)      # d_k depends on l_0..l_k only
    ref = oracle.divided_differences(theta, 129)
    big = np.abs(ref) > 1e-16
    assert np.max(np.abs(full - ref)[big] / np.abs(ref)[big]) < 1e-15
    if theta == 0.0:
        assert full[0] == 1.0 and np.all(full[1:] == 0.0)


def test_newton_polynomial_reproduces_exponential(M):
    theta, m = 5.0, 90
    l = M.magnus_host_leja_points(m)
    d = M.magnus_host_divided_differences(theta, m)
    x = np.linspace(-2, 2, 1000)
    p = np.zeros_like(x, dtype=complex)
    w = np.ones_like(x, dtype=complex)
    for k in range(m):
        p += d[k] * w
        w = w * (x - l[k])
    assert np.max(np.abs(p - np.exp(-1j * theta * x))) < 1e-13


# ------------------------------------------------------------------ interval snapping (c4)
def test_snap_interval(M, oracle):
    r = np.random.default_rng(0)
    for _ in range(2000):
        a = r.normal() * 10 ** r.uniform(-3, 3)
        b = a + 10 ** r.uniform(-3, 3)
        sa, sb = M.magnus_host_snap_interval(a, b)
        assert (sa, sb) == oracle.snap_interval(a, b)
        delta = 2.0 ** (math.ceil(math.log2(b - a)) - 12)
        assert sa <= a < sa + delta and sb - delta < b <= sb
    assert M.magnus_host_snap_interval(-4.0, 4.0) == (-4.0, 4.0)
    assert M.magnus_host_snap_interval(0.0, 1.0) == (0.0, 1.0)
    assert M.magnus_host_snap_interval(1.0, 1.0) == (1.0, 1.0)       # gamma = 0 passes through


# ------------------------------------------------------------------ scheme scalars (c1)
def test_step_coefficients_against_printed_formulas(M):
    f = lambda t: math.sin(3 * t) + 0.2 * t
    t, tau = 0.3, 0.07
    s3, s15 = math.sqrt(3), math.sqrt(15)
    f1, f2 = f(t + (0.5 - s3 / 6) * tau), f(t + (0.5 + s3 / 6) * tau)
    a1, a2 = (3 - 2 * s3) / 12, (3 + 2 * s3) / 12
    coef, hs, _ = M.magnus_host_step_coefficients("cf4", f, t, tau)
    # exp(tau(a1 A1 + a2 A2)) exp(tau(a2 A1 + a1 A2)) Y: the right factor acts first, H-weight a1+a2 = 1/2
    assert hs == [0.5, 0.5]
    assert math.isclose(coef[0], (a2 * f1 + a1 * f2) / 0.5, rel_tol=1e-15)
    assert math.isclose(coef[1], (a1 * f1 + a2 * f2) / 0.5, rel_tol=1e-15)
    coef, hs, kappa = M.magnus_host_step_coefficients("m4", f, t, tau)
    assert coef == [f1, f2] and hs == [1.0]
    assert math.isclose(kappa, s3 * tau / 12 * (f1 - f2), rel_tol=1e-15)
    coef, hs, _ = M.magnus_host_step_coefficients("m2", f, t, tau)
    assert coef == [f(t + tau / 2)] and hs == [1.0]
    coef, hs, _ = M.magnus_host_step_coefficients("cf4:3", f, t, tau)
    fn = [f(t + (0.5 - s15 / 10) * tau), f(t + 0.5 * tau), f(t + (0.5 + s15 / 10) * tau)]
    al = np.array([[37 / 240 - 10 * s15 / 261, -1 / 30, 37 / 240 + 10 * s15 / 261],
                   [-11 / 360, 23 / 45, -11 / 360],
                   [37 / 240 + 10 * s15 / 261, -1 / 30, 37 / 240 - 10 * s15 / 261]])
    assert math.isclose(sum(hs), 1.0, rel_tol=1e-15)
    for e in range(3):                  # exponential e acts e-th: row 3 first
        row = al[2 - e]
        assert math.isclose(hs[e], row.sum(), rel_tol=1e-14)
        assert math.isclose(coef[e] * hs[e], row @ np.array(fn), rel_tol=1e-13)


def test_bad_arguments_are_rejected_before_any_cuda_call(M):
    with pytest.raises(M.MagnusError):
        M.magnus_host_leja_points(500)
    with pytest.raises(M.MagnusError):
        M.magnus_host_divided_differences(1.0, 0)


def test_tridiag_extremes_against_numpy(M):
    """The host piece of the tight-interval shortcut (Sturm bisection) against numpy.linalg.eigvalsh: random
    tridiagonals, k = 1, a zero off-diagonal (decoupled blocks), equal eigenvalues, huge and tiny scales."""
    r = np.random.default_rng(7)
    cases = [(r.normal(size=k), np.abs(r.normal(size=k - 1))) for k in (2, 3, 8, 12, 40, 64)]
    cases += [(np.array([2.5]), np.array([])), (np.array([1.0, -3.0, 2.0]), np.array([0.0, 0.5])),
              (np.ones(6), np.zeros(5)), (1e150 * r.normal(size=5), 1e150 * np.abs(r.normal(size=4))),
              (1e-150 * r.normal(size=5), 1e-150 * np.abs(r.normal(size=4)))]
    for al, be in cases:
        k = len(al)
        T = np.diag(al) + (np.diag(be, 1) + np.diag(be, -1) if k > 1 else 0.0)
        ev = np.linalg.eigvalsh(T)
        lo, hi = M.magnus_host_tridiag_extremes(al, be)
        scale = max(np.max(np.abs(al)), np.max(np.abs(be)) if k > 1 else 0.0)
        assert abs(lo - ev[0]) <= 1e-13 * scale and abs(hi - ev[-1]) <= 1e-13 * scale, (al, be, lo, hi, ev[0], ev[-1])
