"""Pins for the oracle's Magnus steps (SURVEY.md 8(c) pins c-P6..c-P11).

References are independent of the oracle: numpy.linalg.eigh exponentials, a
brute-force fine-step propagator, closed forms for commuting operators, and the
convergence order the paper states (PAPER.md lines 97-101 Method 2 "order
four", lines 130-134 Method 4 "order 4", line 156 Figure 1).
"""
import math

import numpy as np
import pytest

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


def expm_h(M, h):
    lam, U = np.linalg.eigh(M)
    return (U * np.exp(-1j * h * lam)) @ U.conj().T


def brute_force(H0, H1, f, t0, t1, psi, nfine=4000):
    """psi(t1) by the exponential midpoint rule with exact small exponentials on a very
    fine grid (error O(dt^2) ~ 1e-8 * const): an integrator that shares nothing with
    the Gauss-node schemes under test."""
    dt = (t1 - t0) / nfine
    for k in range(nfine):
        psi = expm_h(H0 + f(t0 + (k + 0.5) * dt) * H1, dt) @ psi
    return psi


def csr_pair(oracle, N):
    return oracle.CsrHost.of(xxz.xxz_h0(N)), oracle.CsrHost.of(xxz.xxz_h1(N))


# ------------------------------------------------------------------ c-P6
@pytest.mark.parametrize("scheme", ["cf4", "m4"])
@pytest.mark.parametrize("nsteps", [1, 3, 8])
def test_time_independent_hamiltonian_is_exact(oracle, scheme, nsteps):
    n = 24
    H0, H1 = rand_herm(n, 1, 0.5), rand_herm(n, 2, 0.5)
    psi0 = rand_vec(n, 3)
    fc = 0.37
    psi, iters = oracle.magnus_integrate(H0, H1, lambda t: fc, scheme, 0.0, 0.9, nsteps, psi0)
    ref = expm_h(H0 + fc * H1, 0.9) @ psi0
    assert np.linalg.norm(psi - ref) < 2e-11
    assert len(iters) == nsteps * (2 if scheme == "cf4" else 1) and np.all(iters > 0)


# ------------------------------------------------------------------ c-P7
def test_commuting_operators(oracle):
    n = 20
    U = np.linalg.qr(rand_herm(n, 4))[0]
    r = np.random.default_rng(5)
    H0 = (U * r.normal(size=n)) @ U.conj().T
    H1 = (U * r.normal(size=n)) @ U.conj().T
    H0, H1 = (H0 + H0.conj().T) / 2, (H1 + H1.conj().T) / 2
    K = oracle.commutator(H0, H1)
    assert np.abs(K).max() < 1e-14
    f = lambda t: math.cos(2 * t)
    psi0 = rand_vec(n, 6)
    T, ns = 0.8, 4
    tau = T / ns
    c1, c2 = 0.5 - math.sqrt(3) / 6, 0.5 + math.sqrt(3) / 6
    Q = sum(tau / 2 * (f(s * tau + c1 * tau) + f(s * tau + c2 * tau)) for s in range(ns))
    ref = expm_h(H0 * T + H1 * Q, 1.0) @ psi0
    a, _ = oracle.magnus_integrate(H0, H1, f, "cf4", 0.0, T, ns, psi0)
    b, _ = oracle.magnus_integrate(H0, H1, f, "m4", 0.0, T, ns, psi0)
    assert np.linalg.norm(a - ref) < 1e-11 and np.linalg.norm(b - ref) < 1e-11
    assert np.linalg.norm(a - b) < 1e-11


# ------------------------------------------------------------------ c-P8
def observed_order(oracle, H0, H1, f, scheme, psi0, T, ref, steps=(4, 8, 16)):
    errs = []
    for ns in steps:
        psi, _ = oracle.magnus_integrate(H0, H1, f, scheme, 0.0, T, ns, psi0, tol=1e-14)
        errs.append(np.linalg.norm(psi - ref))
    slopes = [math.log2(errs[i] / errs[i + 1]) for i in range(len(errs) - 1)]
    return errs, slopes


def test_fourth_order_dense_and_negative_control(oracle):
    n = 12
    H0, H1 = rand_herm(n, 7, 0.6), rand_herm(n, 8, 0.6)
    f = lambda t: math.sin(3 * t)
    psi0 = rand_vec(n, 9)
    T = 1.0
    ref = brute_force(H0, H1, f, 0.0, T, psi0, nfine=20000)   # error ~1e-9, below the errors measured
    for scheme in ("cf4", "m4"):
        errs, slopes = observed_order(oracle, H0, H1, f, scheme, psi0, T, ref, steps=(8, 16, 32))
        assert all(3.7 < s < 4.4 for s in slopes), (scheme, errs, slopes)
    errs, slopes = observed_order(oracle, H0, H1, f, "m4_wrong_sign", psi0, T, ref, steps=(8, 16, 32))
    assert all(1.7 < s < 2.3 for s in slopes), ("flipped commutator must drop to order 2", errs, slopes)


def test_fourth_order_xxz_csr_self_convergence(oracle):
    """Order on the sparse path; reference = same scheme at a 16x finer step (pin c-P8)."""
    N = 6
    H0, H1 = csr_pair(oracle, N)
    psi0 = xxz.neel_state(N).numpy()
    f = xxz.f_cos2t
    T = 0.5
    for scheme in ("cf4", "m4"):
        ref, _ = oracle.magnus_integrate(H0, H1, f, scheme, 0.0, T, 256, psi0, tol=1e-14)
        errs, slopes = observed_order(oracle, H0, H1, f, scheme, psi0, T, ref, steps=(4, 8, 16))
        assert all(3.8 < s < 4.2 for s in slopes), (scheme, errs, slopes)
    # and both schemes converge to the SAME solution (brute force, dense copy of the chain)
    D0, D1 = xxz.xxz_h0(N).to_scipy().toarray(), xxz.xxz_h1(N).to_scipy().toarray()
    bf = brute_force(D0, D1, f, 0.0, T, psi0, nfine=8000)
    for scheme in ("cf4", "m4"):
        psi, _ = oracle.magnus_integrate(H0, H1, f, scheme, 0.0, T, 64, psi0)
        assert np.linalg.norm(psi - bf) < 5e-8


# ------------------------------------------------------------------ c-P9
def test_cf4_vs_m4_and_error_constant(oracle):
    n = 16
    H0, H1 = rand_herm(n, 11, 0.5), rand_herm(n, 12, 0.5)
    f = lambda t: math.sin(3 * t)
    psi0 = rand_vec(n, 13)
    ref = brute_force(H0, H1, f, 0.0, 1.0, psi0, nfine=20000)
    d = []
    for ns in (4, 8):
        a, _ = oracle.magnus_integrate(H0, H1, f, "cf4", 0.0, 1.0, ns, psi0)
        b, _ = oracle.magnus_integrate(H0, H1, f, "m4", 0.0, 1.0, ns, psi0)
        d.append(np.linalg.norm(a - b))
        # "Cf4 ... is somewhat more accurate compared to the M4 method"
        assert np.linalg.norm(a - ref) < np.linalg.norm(b - ref)
    assert 3.5 < math.log2(d[0] / d[1]) < 4.5          # the two differ by O(tau^4)


# ------------------------------------------------------------------ c-P10
@pytest.mark.parametrize("scheme", ["cf4", "m4"])
def test_time_reversal_symmetry(oracle, scheme):
    n = 16
    H0, H1 = rand_herm(n, 14, 0.5), rand_herm(n, 15, 0.5)
    f = lambda t: math.sin(3 * t)
    psi0 = rand_vec(n, 16)
    psi1, _ = oracle.magnus_step(H0, H1, f, scheme, 0.2, 0.1, psi0)
    back, _ = oracle.magnus_step(H0, H1, f, scheme, 0.3, -0.1, psi1)
    assert np.linalg.norm(back - psi0) < 1e-11
    assert abs(np.linalg.norm(psi1) - 1) < 1e-10


# ------------------------------------------------------------------ c-P11
def test_commutator_identities(oracle):
    n = 18
    A, B = rand_herm(n, 17), rand_herm(n, 18)
    K = oracle.commutator(A, B)
    assert np.allclose(K, A @ B - B @ A, atol=1e-13)
    P = A @ B
    assert np.allclose(K, P - P.conj().T, atol=1e-13)          # Hermitian operands
    assert np.allclose(K, -K.conj().T, atol=1e-13) and abs(np.trace(K)) < 1e-12
    # [H(t2), H(t1)] = (f1 - f2) [H0, H1]
    f1, f2 = 0.3, -0.8
    K21 = oracle.commutator(A + f2 * B, A + f1 * B)
    assert np.allclose(K21, (f1 - f2) * oracle.commutator(A, B), atol=1e-12)


def test_dense_product_is_not_transposed(oracle):
    n = 23
    A = rand_herm(n, 30) + 0.2j * np.triu(np.ones((n, n)), 2)     # not Hermitian: A@B != (B@A)^H
    B = rand_herm(n, 31) - 0.4 * np.tril(np.ones((n, n)), -1)
    assert np.allclose(oracle.matmul(A, B), A @ B, rtol=0, atol=1e-13)
    assert not np.allclose(oracle.matmul(A, B), B @ A, atol=1e-3)
    assert not np.allclose(oracle.matmul(A, B), A.T @ B.T, atol=1e-3)


def test_sparse_commutator_matches_dense(oracle):
    N = 5
    H0, H1 = csr_pair(oracle, N)
    K = oracle.commutator(H0, H1)
    import scipy.sparse as sp
    Ks = sp.csr_matrix((K.values, K.col_idx, K.row_ptr), shape=(K.n, K.n)).toarray()
    D0, D1 = xxz.xxz_h0(N).to_scipy().toarray(), xxz.xxz_h1(N).to_scipy().toarray()
    assert np.array_equal(Ks, D0 @ D1 - D1 @ D0)
    assert np.all(Ks.imag == 0) and np.array_equal(Ks, -Ks.T)   # real antisymmetric
    nz = Ks != 0
    assert np.all(D1[nz] != 0)                                   # pattern inside H1's
    assert nz.sum() == N * 2 ** (N - 1)


def test_sparse_and_dense_steps_agree(oracle):
    N = 5
    H0, H1 = csr_pair(oracle, N)
    D0, D1 = xxz.xxz_h0(N).to_scipy().toarray(), xxz.xxz_h1(N).to_scipy().toarray()
    psi0 = rand_vec(32, 19)
    for scheme in ("cf4", "m4"):
        a, ia = oracle.magnus_step(H0, H1, xxz.f_cos2t, scheme, 0.1, 0.05, psi0)
        b, ib = oracle.magnus_step(D0, D1, xxz.f_cos2t, scheme, 0.1, 0.05, psi0)
        assert np.linalg.norm(a - b) < 1e-13
        assert [i["iters"] for i in ia] == [i["iters"] for i in ib]
        assert [i["a"] for i in ia] == [i["a"] for i in ib]


def test_single_step_matches_scheme_formula_with_exact_exponentials(oracle):
    """One step against the printed formulas evaluated with
    eigendecomposition exponentials of A = -iH."""
    n = 10
    H0, H1 = rand_herm(n, 20, 0.5), rand_herm(n, 21, 0.5)
    f = lambda t: math.sin(3 * t)
    psi0 = rand_vec(n, 22)
    t, tau = 0.4, 0.2
    c1, c2 = 0.5 - math.sqrt(3) / 6, 0.5 + math.sqrt(3) / 6
    Ha, Hb = H0 + f(t + c1 * tau) * H1, H0 + f(t + c2 * tau) * H1    # H(t1), H(t2)
    A1, A2 = -1j * Ha, -1j * Hb
    a1, a2 = (3 - 2 * math.sqrt(3)) / 12, (3 + 2 * math.sqrt(3)) / 12

    def expm_general(X):            # X = -i * Hermitian
        return expm_h(1j * X, 1.0)

    ref_cf4 = expm_general(tau * (a1 * A1 + a2 * A2)) @ (expm_general(tau * (a2 * A1 + a1 * A2)) @ psi0)
    Om = tau / 2 * (A1 + A2) + math.sqrt(3) * tau ** 2 / 12 * (A2 @ A1 - A1 @ A2)
    ref_m4 = expm_general(Om) @ psi0
    got_cf4, _ = oracle.magnus_step(H0, H1, f, "cf4", t, tau, psi0)
    got_m4, _ = oracle.magnus_step(H0, H1, f, "m4", t, tau, psi0)
    assert np.linalg.norm(got_cf4 - ref_cf4) < 1e-11
    assert np.linalg.norm(got_m4 - ref_m4) < 1e-11


def test_single_step_cf43_and_m2_match_printed_products_with_exact_exponentials(oracle):
    """One Cf4:3 step against the printed product (nodes 1/2, 1/2 -+ sqrt(15)/10, the 3 x 3
    alpha table, the factor of row 3 acting first) and one M2 step against exp(tau A(t + tau/2)) (lines 87-95), both
    with eigendecomposition exponentials of A = -iH.  A swapped row order, a transposed alpha or a wrong node fails
    here at O(tau^3) ~ 1e-3, far above the bar."""
    n = 10
    H0, H1 = rand_herm(n, 23, 0.5), rand_herm(n, 24, 0.5)
    f = lambda t: math.sin(3 * t)
    psi0 = rand_vec(n, 25)
    t, tau = 0.4, 0.2
    s15 = math.sqrt(15.0)
    c = (0.5 - s15 / 10, 0.5, 0.5 + s15 / 10)
    A = [-1j * (H0 + f(t + ci * tau) * H1) for ci in c]
    p, m = 37 / 240 + 10 * s15 / 261, 37 / 240 - 10 * s15 / 261
    alpha = np.array([[m, -1 / 30, p], [-11 / 360, 23 / 45, -11 / 360], [p, -1 / 30, m]])

    def expm_general(X):            # X = -i * Hermitian
        return expm_h(1j * X, 1.0)

    y = psi0
    for row in (2, 1, 0):           # exp(Omega^(1)) exp(Omega^(2)) exp(Omega^(3)) Y_n: the third factor acts first
        y = expm_general(tau * sum(alpha[row, j] * A[j] for j in range(3))) @ y
    got, infos = oracle.magnus_step(H0, H1, f, "cf4:3", t, tau, psi0)
    assert len(infos) == 3 and np.linalg.norm(got - y) < 1e-11
    wrong = psi0
    for row in (0, 1, 2):           # negative control: the factors in the other order differ at O(tau^3)
        wrong = expm_general(tau * sum(alpha[row, j] * A[j] for j in range(3))) @ wrong
    assert np.linalg.norm(wrong - y) > 1e-6
    ref_m2 = expm_general(tau * (-1j) * (H0 + f(t + tau / 2) * H1)) @ psi0
    got_m2, infos = oracle.magnus_step(H0, H1, f, "m2", t, tau, psi0)
    assert len(infos) == 1 and np.linalg.norm(got_m2 - ref_m2) < 1e-11


def test_cfg1_totals_are_stable(oracle):
    """CFG1 end to end on the oracle: norm conserved to 1e-10 (north_star), CF4 and M4
    agree to O(tau^4); the iteration totals are recorded in tests/golden by
    tests/golden/make_golden.py (oracle-only) and must not drift silently."""
    import json, os
    cfg = W.CONFIGS["cfg1"]
    H0, H1, psi0, f = W.build(cfg)
    H0, H1 = oracle.CsrHost.of(H0), oracle.CsrHost.of(H1)
    out = {}
    for scheme in cfg.schemes:
        psi, iters = oracle.magnus_integrate(H0, H1, f, scheme, cfg.t0, cfg.t_end, cfg.nsteps, psi0.numpy(), cfg.tol)
        assert abs(np.linalg.norm(psi) - 1) < 1e-10
        out[scheme] = (psi, int(iters.sum()))
    assert 1e-10 < np.linalg.norm(out["cf4"][0] - out["m4"][0]) < 1e-8
    gold = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "cfg1_oracle.json")))
    assert out["cf4"][1] == gold["cf4"]["total_matvecs"] and out["m4"][1] == gold["m4"]["total_matvecs"]


# ------------------------------------------------------------------ M2 and Cf4:3
def _exact_propagator_reference(H0, H1, f, t0, T, fine=30000):
    """Brute force: exponential midpoint with EXACT (eigh) exponentials on a very fine grid."""
    psi = None
    tau = (T - t0) / fine
    U = np.eye(H0.shape[0], dtype=complex)
    for s in range(fine):
        lam, V = np.linalg.eigh(H0 + f(t0 + (s + 0.5) * tau) * H1)
        U = (V * np.exp(-1j * tau * lam)) @ V.conj().T @ U
    return U


@pytest.mark.parametrize("scheme,order", [("m2", 2), ("cf4:3", 4)])
def test_order_of_m2_and_cf43(oracle, scheme, order):
    """P:95 "which is of order two"; "optimized commutator-free method of order 4": step-halving slope
    against a brute-force reference that does not use the oracle."""
    n = 12
    r = np.random.default_rng(3)
    def herm():
        G = r.normal(size=(n, n)) + 1j * r.normal(size=(n, n))
        return (G + G.conj().T) / 2
    H0, H1 = herm(), herm()
    f = lambda t: math.sin(3 * t) + 0.3 * t
    psi0 = r.normal(size=n) + 1j * r.normal(size=n); psi0 /= np.linalg.norm(psi0)
    T = 0.4
    exact = _exact_propagator_reference(H0, H1, f, 0.0, T) @ psi0
    errs = []
    for ns in (4, 8, 16):      # the order-2 brute-force reference is good to about 1e-10
        psi, _ = oracle.magnus_integrate(H0, H1, f, scheme, 0.0, T, ns, psi0, 1e-14)
        errs.append(np.linalg.norm(psi - exact))
    slopes = [math.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert all(order - 0.3 < s < order + 0.35 for s in slopes), (errs, slopes)


def test_cf43_smaller_error_constant_than_cf4(oracle):
    """Cf4:3 has a smaller error constant than Cf4 (same order)."""
    n = 10
    r = np.random.default_rng(4)
    G = r.normal(size=(n, n)) + 1j * r.normal(size=(n, n)); H0 = (G + G.conj().T) / 2
    G = r.normal(size=(n, n)) + 1j * r.normal(size=(n, n)); H1 = (G + G.conj().T) / 2
    f = lambda t: math.cos(2 * t)
    psi0 = np.zeros(n, complex); psi0[0] = 1
    exact = _exact_propagator_reference(H0, H1, f, 0.0, 0.5) @ psi0
    e = {}
    for scheme in ("cf4", "cf4:3"):
        psi, _ = oracle.magnus_integrate(H0, H1, f, scheme, 0.0, 0.5, 10, psi0, 1e-14)
        e[scheme] = np.linalg.norm(psi - exact)
    assert e["cf4:3"] < e["cf4"]


@pytest.mark.parametrize("scheme", ["m2", "cf4:3"])
def test_m2_cf43_time_independent_and_reversal(oracle, scheme):
    """f = const: every scheme is the exact exponential (row sums of alpha add up to 1); and
    step(t, tau) followed by step(t + tau, -tau) is the identity (both schemes are self-adjoint)."""
    n = 16
    r = np.random.default_rng(6)
    G = r.normal(size=(n, n)) + 1j * r.normal(size=(n, n)); H0 = (G + G.conj().T) / 2
    G = r.normal(size=(n, n)) + 1j * r.normal(size=(n, n)); H1 = (G + G.conj().T) / 2
    psi0 = r.normal(size=n) + 1j * r.normal(size=n); psi0 /= np.linalg.norm(psi0)
    psi, _ = oracle.magnus_integrate(H0, H1, lambda t: 0.7, scheme, 0.0, 0.6, 3, psi0, 1e-13)
    lam, V = np.linalg.eigh(H0 + 0.7 * H1)
    assert np.linalg.norm(psi - V @ (np.exp(-0.6j * lam) * (V.conj().T @ psi0))) < 1e-11
    f = lambda t: math.sin(3 * t)
    a, _ = oracle.magnus_step(H0, H1, f, scheme, 0.2, 0.1, psi0, 1e-13)
    b, _ = oracle.magnus_step(H0, H1, f, scheme, 0.3, -0.1, a, 1e-13)
    assert np.linalg.norm(b - psi0) < 1e-11


# ------------------------------------------------------------------ M6 (Method 3)
def _herm_pair(n, seed):
    r = np.random.default_rng(seed)
    def herm():
        G = r.normal(size=(n, n)) + 1j * r.normal(size=(n, n))
        return (G + G.conj().T) / 2
    H0, H1 = herm(), herm()
    psi0 = r.normal(size=n) + 1j * r.normal(size=n)
    return H0, H1, psi0 / np.linalg.norm(psi0)


def test_m6_order_six_and_printed_coefficient_is_order_two(oracle):
    """P:103 "the following scheme of order six": step-halving slope 6 against a brute-force propagator that does not
    use the oracle.  Reading m6: with the coefficient of B3 as PAPER.md l.105 prints it (1/2) the same test gives
    order 2 -- the first Magnus term int A = tau a0 + tau^3 a2/12 needs 1/12."""
    n = 10
    H0, H1, psi0 = _herm_pair(n, 11)
    H0, H1 = 0.6 * H0, 0.6 * H1
    f = lambda t: math.sin(3 * t) + 0.3 * t
    T = 0.6
    # reference: the oracle-independent exact-exponential midpoint rule, Richardson-extrapolated twice (errors
    # O(dt^2), O(dt^4) removed) so that it is good to ~1e-13, below the order-6 errors measured here
    U1 = _exact_propagator_reference(H0, H1, f, 0.0, T, fine=1500) @ psi0
    U2 = _exact_propagator_reference(H0, H1, f, 0.0, T, fine=3000) @ psi0
    U4 = _exact_propagator_reference(H0, H1, f, 0.0, T, fine=6000) @ psi0
    R1, R2 = (4 * U2 - U1) / 3, (4 * U4 - U2) / 3
    exact = (16 * R2 - R1) / 15
    assert np.linalg.norm(R2 - exact) < 1e-11
    errs = []
    for ns in (2, 4, 8):
        psi, _ = oracle.magnus_integrate(H0, H1, f, "m6", 0.0, T, ns, psi0, 1e-15)
        errs.append(np.linalg.norm(psi - exact))
    slopes = [math.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert errs[-1] > 3e-12, errs                         # still above the reference's own accuracy
    assert all(5.5 < s < 6.6 for s in slopes), (errs, slopes)
    bad = []
    for ns in (4, 8, 16):
        psi, _ = oracle.magnus_integrate(H0, H1, f, "m6_as_printed", 0.0, T, ns, psi0, 1e-14)
        bad.append(np.linalg.norm(psi - exact))
    bslopes = [math.log2(bad[i] / bad[i + 1]) for i in range(2)]
    assert all(1.7 < s < 2.3 for s in bslopes), (bad, bslopes)
    # and M6 beats the fourth-order schemes at the same step (Figure 1)
    p4, _ = oracle.magnus_integrate(H0, H1, f, "m4", 0.0, T, 8, psi0, 1e-15)
    assert errs[-1] < 0.05 * np.linalg.norm(p4 - exact)


def test_m6_time_independent_commuting_and_reversal(oracle):
    n = 14
    H0, H1, psi0 = _herm_pair(n, 12)
    # f = const: B2 = B3 = 0, Omega = tau A: exact exponential
    psi, iters = oracle.magnus_integrate(H0, H1, lambda t: -0.4, "m6", 0.0, 0.7, 3, psi0, 1e-13)
    lam, V = np.linalg.eigh(H0 - 0.4 * H1)
    assert np.linalg.norm(psi - V @ (np.exp(-0.7j * lam) * (V.conj().T @ psi0))) < 1e-11 and len(iters) == 3
    # time reversal: step(t, tau) then step(t + tau, -tau) is the identity (the scheme is self-adjoint)
    f = lambda t: math.cos(2 * t) + t * t
    a, _ = oracle.magnus_step(H0, H1, f, "m6", 0.1, 0.2, psi0, 1e-13)
    b, _ = oracle.magnus_step(H0, H1, f, "m6", 0.3, -0.2, a, 1e-13)
    assert np.linalg.norm(b - psi0) < 1e-11 and np.linalg.norm(a - psi0) > 1e-2
    # commuting H0, H1: every commutator vanishes, Omega_H = H0 + Q3 H1 with Q3 the three-point Gauss rule of f
    U = np.linalg.qr(H0)[0]
    r = np.random.default_rng(13)
    D0 = (U * r.normal(size=n)) @ U.conj().T; D0 = (D0 + D0.conj().T) / 2
    D1 = (U * r.normal(size=n)) @ U.conj().T; D1 = (D1 + D1.conj().T) / 2
    t, tau = 0.3, 0.25
    s15 = math.sqrt(15) / 10
    fn = [f(t + (0.5 - s15) * tau), f(t + 0.5 * tau), f(t + (0.5 + s15) * tau)]
    Om = oracle.m6_omega(D0, D1, fn, tau)
    Q3 = (5 * fn[0] + 8 * fn[1] + 5 * fn[2]) / 18
    assert np.abs(Om - (D0 + Q3 * D1)).max() < 1e-13


def test_m6_omega_structure_and_csr_agrees_with_dense(oracle):
    """Omega_H is Hermitian; its leading terms are the ones the formula prints: H0 + Q3 H1 + (commutator terms of
    relative size tau); and the CSR implementation of the same formulas gives the same step as the dense one."""
    N = 6
    H0s, H1s = xxz.xxz_h0(N), xxz.xxz_h1(N)
    H0d, H1d = H0s.to_scipy().toarray(), H1s.to_scipy().toarray()
    f = xxz.f_cos2t
    t, tau = 0.4, 0.05
    s15 = math.sqrt(15) / 10
    fn = [f(t + (0.5 - s15) * tau), f(t + 0.5 * tau), f(t + (0.5 + s15) * tau)]
    Om = oracle.m6_omega(H0d, H1d, fn, tau)
    assert np.abs(Om - Om.conj().T).max() < 1e-13
    Q3 = (5 * fn[0] + 8 * fn[1] + 5 * fn[2]) / 18
    C = H0d @ H1d - H1d @ H0d
    # leading commutator term: (1/240)[-20 B1, B2] = -(1/12)[B1, B2], and with A = -iH
    # [B1, B2] = -(sqrt(15)/3) tau^2 (f3 - f1) [H0, H1], so
    # Omega_H = (i/tau) Omega = H0 + Q3 H1 + i (sqrt(15)/36) tau (f3 - f1) [H0, H1] + O(tau^3)
    # (the counterpart of M4's -i (sqrt(3) tau/12)(f1 - f2)[H0, H1], on the three-point nodes)
    lead = H0d + Q3 * H1d + 1j * (math.sqrt(15) / 36) * tau * (fn[2] - fn[0]) * C
    assert np.abs(Om - lead).max() < 5e-3 * tau and np.abs(Om - (H0d + Q3 * H1d)).max() > 1e-4
    psi0 = rand_vec(1 << N, 7)
    a, ia = oracle.magnus_step(oracle.CsrHost.of(H0s), oracle.CsrHost.of(H1s), f, "m6", t, tau, psi0)
    b, ib = oracle.magnus_step(H0d, H1d, f, "m6", t, tau, psi0)
    assert np.linalg.norm(a - b) < 1e-12 and ia[0]["iters"] == ib[0]["iters"]
