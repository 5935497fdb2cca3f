"""ctypes front end of the C++ oracle (TEST INFRASTRUCTURE ONLY).

numpy in, numpy out; all arithmetic happens in magnus_oracle.cpp.  This file
only marshals arguments.  It must never be imported by the product path.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass
from typing import Callable, Optional, Sequence, Tuple

import numpy as np

from . import build as _build

CF4, M4, M2, CF4_3, M6, M4_WRONG_SIGN, M6_AS_PRINTED = 0, 1, 2, 3, 4, 101, 104
SCHEMES = {"cf4": CF4, "m4": M4, "m2": M2, "cf4:3": CF4_3, "m6": M6, "m4_wrong_sign": M4_WRONG_SIGN,
           "m6_as_printed": M6_AS_PRINTED}
N_EXP = {CF4: 2, M4: 1, M2: 1, CF4_3: 3, M6: 1, M4_WRONG_SIGN: 1, M6_AS_PRINTED: 1}

DRIVE = C.CFUNCTYPE(C.c_double, C.c_double, C.c_void_p)


class ExpmvInfo(C.Structure):
    _fields_ = [("iters", C.c_int32), ("substeps", C.c_int32), ("status", C.c_int32), ("_pad", C.c_int32),
                ("a", C.c_double), ("b", C.c_double), ("theta", C.c_double), ("err_est", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "_pad"}


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.oracle_max_degree.restype = C.c_int
        L.oracle_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _c(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


@dataclass
class CsrHost:
    n: int
    row_ptr: np.ndarray
    col_idx: np.ndarray
    values: np.ndarray

    @staticmethod
    def of(m) -> "CsrHost":
        """From a workloads.xxz.CSR (torch) or anything with the same fields."""
        def h(x):
            return x.cpu().numpy() if hasattr(x, "cpu") else np.asarray(x)
        return CsrHost(int(m.n), _c(h(m.row_ptr), np.int32), _c(h(m.col_idx), np.int32), _c(h(m.values), np.complex128))

    def args(self):
        return (_p(self.row_ptr), _p(self.col_idx), _p(self.values))


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(t: int) -> None:
    lib().oracle_set_num_threads(C.c_int(t))


def max_degree() -> int:
    return int(lib().oracle_max_degree())


def leja_points(m: int) -> np.ndarray:
    out = np.empty(m, dtype=np.float64)
    lib().oracle_leja_points(C.c_int(m), _p(out))
    return out


def divided_differences(theta: float, m: int) -> np.ndarray:
    out = np.empty(m, dtype=np.complex128)
    lib().oracle_divided_differences(C.c_double(theta), C.c_int(m), _p(out))
    return out


def snap_interval(a: float, b: float) -> Tuple[float, float]:
    ca, cb = C.c_double(a), C.c_double(b)
    lib().oracle_snap_interval(C.byref(ca), C.byref(cb))
    return ca.value, cb.value


def gershgorin(M):
    """Returns ((a_raw, b_raw), (a_snapped, b_snapped)) for dense ndarray or CsrHost."""
    raw, snp = np.empty(2), np.empty(2)
    if isinstance(M, CsrHost):
        lib().oracle_gershgorin_csr(C.c_int64(M.n), *M.args(), _p(raw), _p(snp))
    else:
        M = _c(M, np.complex128)
        lib().oracle_gershgorin_dense(C.c_int64(M.shape[0]), _p(M), _p(raw), _p(snp))
    return tuple(raw), tuple(snp)


def lanczos_interval(M, v, m: int):
    """Shortcut "tight interval" (reading ti): raw interval from m Lanczos steps started at v.
    Returns ((a, b), alpha, beta) with the steps actually taken."""
    v = _c(v, np.complex128)
    ab = np.zeros(2); al = np.zeros(m); be = np.zeros(m)
    if isinstance(M, CsrHost):
        k = lib().oracle_lanczos_interval_csr(C.c_int64(M.n), *M.args(), _p(v), C.c_int(m), _p(ab), _p(al), _p(be))
    else:
        M = _c(M, np.complex128)
        k = lib().oracle_lanczos_interval_dense(C.c_int64(M.shape[0]), _p(M), _p(v), C.c_int(m), _p(ab), _p(al), _p(be))
    return (float(ab[0]), float(ab[1])), al[:k].copy(), be[:k].copy()


class tight_interval:
    """Context manager: inside, every leja_expmv / magnus_step / magnus_integrate takes its interval from m
    Lanczos steps (the shortcut) instead of Gershgorin (the mandated path)."""

    def __init__(self, m: int):
        self.m = int(m)

    def __enter__(self):
        self.old = int(lib().oracle_get_lanczos_steps())
        lib().oracle_set_lanczos_steps(C.c_int(self.m))
        return self

    def __exit__(self, *exc):
        lib().oracle_set_lanczos_steps(C.c_int(self.old))


def matvec(M, w) -> np.ndarray:
    w = _c(w, np.complex128)
    y = np.empty_like(w)
    if isinstance(M, CsrHost):
        lib().oracle_matvec_csr(C.c_int64(M.n), *M.args(), _p(w), _p(y))
    else:
        M = _c(M, np.complex128)
        lib().oracle_matvec_dense(C.c_int64(M.shape[0]), _p(M), _p(w), _p(y))
    return y


def leja_expmv(M, v, h: float, tol: float = 1e-12):
    """exp(-i h M) v.  Returns (result, info dict); raises on ENOCONV."""
    v = _c(v, np.complex128)
    out = np.empty_like(v)
    info = ExpmvInfo()
    if isinstance(M, CsrHost):
        rc = lib().oracle_leja_expmv_csr(C.c_int64(M.n), *M.args(), _p(v), _p(out), C.c_double(h), C.c_double(tol), C.byref(info))
    else:
        M = _c(M, np.complex128)
        rc = lib().oracle_leja_expmv_dense(C.c_int64(M.shape[0]), _p(M), _p(v), _p(out), C.c_double(h), C.c_double(tol), C.byref(info))
    if rc != 0:
        raise RuntimeError(f"oracle leja_expmv failed rc={rc} info={info.as_dict()}")
    return out, info.as_dict()


def matmul(A, B) -> np.ndarray:
    """Dense A @ B by the i-k-j definition loop (the product inside the commutator)."""
    A = _c(A, np.complex128); B = _c(B, np.complex128)
    out = np.empty_like(A)
    lib().oracle_matmul_dense(C.c_int64(A.shape[0]), _p(A), _p(B), _p(out))
    return out


def commutator(A, B):
    """A B - B A by the plain definition; dense ndarray or CsrHost (returns the same kind)."""
    if isinstance(A, CsrHost):
        nnz = C.c_int64(0)
        lib().oracle_commutator_csr(C.c_int64(A.n), *A.args(), *B.args(), C.c_int64(0), C.byref(nnz), None, None, None)
        rp = np.empty(A.n + 1, np.int32); ci = np.empty(nnz.value, np.int32); v = np.empty(nnz.value, np.complex128)
        rc = lib().oracle_commutator_csr(C.c_int64(A.n), *A.args(), *B.args(), C.c_int64(nnz.value), C.byref(nnz), _p(rp), _p(ci), _p(v))
        assert rc == 0
        return CsrHost(A.n, rp, ci, v)
    A = _c(A, np.complex128); B = _c(B, np.complex128)
    K = np.empty_like(A)
    lib().oracle_commutator_dense(C.c_int64(A.shape[0]), _p(A), _p(B), _p(K))
    return K


def m6_omega(H0, H1, fn, tau: float) -> np.ndarray:
    """Omega_H of one M6 step on dense H0, H1 at the node values fn = (f(t1), f(t2), f(t3))."""
    H0 = _c(H0, np.complex128); H1 = _c(H1, np.complex128)
    fn = _c(fn, np.float64)
    out = np.empty_like(H0)
    lib().oracle_m6_omega_dense(C.c_int64(H0.shape[0]), _p(H0), _p(H1), _p(fn), C.c_double(tau), _p(out))
    return out


def _drive(f: Callable[[float], float]):
    return DRIVE(lambda t, _u: float(f(t)))


def magnus_step(H0, H1, f, scheme: str, t: float, tau: float, psi, tol: float = 1e-12):
    psi = _c(psi, np.complex128).copy()
    infos = (ExpmvInfo * 3)()
    cb = _drive(f)
    sc = C.c_int(SCHEMES[scheme])
    if isinstance(H0, CsrHost):
        rc = lib().oracle_magnus_step_csr(C.c_int64(H0.n), *H0.args(), *H1.args(), cb, None, sc, C.c_double(t), C.c_double(tau), _p(psi), C.c_double(tol), infos)
    else:
        H0 = _c(H0, np.complex128); H1 = _c(H1, np.complex128)
        rc = lib().oracle_magnus_step_dense(C.c_int64(H0.shape[0]), _p(H0), _p(H1), cb, None, sc, C.c_double(t), C.c_double(tau), _p(psi), C.c_double(tol), infos)
    if rc != 0:
        raise RuntimeError(f"oracle magnus_step failed rc={rc}")
    nexp = N_EXP[SCHEMES[scheme]]
    return psi, [infos[i].as_dict() for i in range(nexp)]


def magnus_integrate(H0, H1, f, scheme: str, t0: float, t_end: float, nsteps: int, psi, tol: float = 1e-12):
    """Returns (psi_final, iteration counts per exponential in call order)."""
    psi = _c(psi, np.complex128).copy()
    nexp = N_EXP[SCHEMES[scheme]] * nsteps
    iters = np.zeros(nexp, dtype=np.int32)
    cb = _drive(f)
    sc = C.c_int(SCHEMES[scheme])
    tail = (sc, C.c_double(t0), C.c_double(t_end), C.c_int64(nsteps), _p(psi), C.c_double(tol), _p(iters), C.c_int64(nexp))
    if isinstance(H0, CsrHost):
        rc = lib().oracle_magnus_integrate_csr(C.c_int64(H0.n), *H0.args(), *H1.args(), cb, None, *tail)
    else:
        H0 = _c(H0, np.complex128); H1 = _c(H1, np.complex128)
        rc = lib().oracle_magnus_integrate_dense(C.c_int64(H0.shape[0]), _p(H0), _p(H1), cb, None, *tail)
    if rc != 0:
        raise RuntimeError(f"oracle magnus_integrate failed rc={rc}")
    return psi, iters
