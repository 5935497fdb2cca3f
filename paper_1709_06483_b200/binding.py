"""ctypes binding of libmagnus_b200.so -- argument marshalling only.

Same names as include/magnus.h.  Every step of the path runs inside the CUDA
kernels of the shared library; nothing here computes.  torch tensors are used
only as owners of device (or pinned host) memory: their data_ptr() is passed
through.  If the library cannot be loaded the import fails loudly -- there is
no fallback of any kind.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Callable, List, Optional, Sequence, Tuple

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libmagnus_b200.so")

OK, EINVAL, ENOMEM, ECUDA, ENOCONV, ENOTHERMITIAN = 0, -1, -2, -3, -4, -5
DENSE, CSR = 0, 1
CF4, M4, M2, CF4_3, M6 = 0, 1, 2, 3, 4
SCHEMES = {"cf4": CF4, "m4": M4, "m2": M2, "cf4:3": CF4_3, "m6": M6}
MAX_EXP_PER_STEP = 3


class MagnusError(RuntimeError):
    def __init__(self, code: int, detail: str):
        super().__init__(f"magnus error {code}: {detail}")
        self.code = code


class MatrixStruct(C.Structure):
    _fields_ = [("format", C.c_int32), ("reserved", C.c_int32), ("n", C.c_int64), ("nnz", C.c_int64),
                ("values", C.c_void_p), ("col_idx", C.c_void_p), ("row_ptr", C.c_void_p), ("ld", C.c_int64)]


class Options(C.Structure):
    _fields_ = [("tol", C.c_double), ("theta_max", C.c_double), ("m_max", C.c_int32), ("check_hermitian", C.c_int32),
                ("stream", C.c_void_p), ("csr_kernel", C.c_int32), ("shortcuts", C.c_int32), ("lanczos_steps", C.c_int32)]


class ExpmvInfo(C.Structure):
    _fields_ = [("iters", C.c_int32), ("substeps", C.c_int32), ("status", C.c_int32), ("reserved", C.c_int32),
                ("a", C.c_double), ("b", C.c_double), ("theta", C.c_double), ("err_est", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "reserved"}


class StepInfo(C.Structure):
    _fields_ = [("n_exp", C.c_int32), ("reserved", C.c_int32), ("exp", ExpmvInfo * MAX_EXP_PER_STEP)]


class Stats(C.Structure):
    _fields_ = [("total_matvecs", C.c_int64), ("n_exp", C.c_int64), ("iters", C.c_void_p), ("iters_cap", C.c_int64),
                ("seconds_device", C.c_double), ("seconds_leja", C.c_double), ("seconds_commutator", C.c_double),
                ("kernel_launches", C.c_int64), ("lanczos_matvecs", C.c_int64)]


class PathInfo(C.Structure):
    _fields_ = [("leja_kernel", C.c_char * 64), ("bytes_per_iteration", C.c_int64),
                ("csr_bytes_per_iteration", C.c_int64), ("slices", C.c_int64), ("slots", C.c_int64),
                ("entries", C.c_int64)]


class XxzModel(C.Structure):
    _fields_ = [("nspins", C.c_int32), ("reserved", C.c_int32), ("jxy", C.c_double), ("jz", C.c_double),
                ("hx", C.c_double)]


DRIVE = C.CFUNCTYPE(C.c_double, C.c_double, C.c_void_p)

EXPORTS = [
    "magnus_create", "magnus_create_xxz", "magnus_destroy", "magnus_describe", "leja_expmv", "magnus_step", "magnus_integrate", "magnus_integrate_host",
    "magnus_gershgorin", "magnus_leja_iteration", "magnus_leja_iteration_dense_noalloc", "magnus_zgemm", "magnus_commutator_dense", "magnus_commutator_csr", "magnus_omega_dense",
    "magnus_fp64_peaks", "magnus_host_leja_points", "magnus_host_divided_differences", "magnus_host_snap_interval", "magnus_host_tridiag_extremes",
    "magnus_host_step_coefficients", "magnus_strerror", "magnus_last_error", "magnus_version",
]

_lib = None


def lib():
    """Load the shared library (raises if it is missing: no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1709_06483_b200.build` "
                              "(there is no fallback path)")
        L = C.CDLL(LIB_PATH)
        for name in EXPORTS:
            getattr(L, name)          # AttributeError if a declared symbol is not exported
        for name in ("magnus_strerror", "magnus_last_error", "magnus_version"):
            getattr(L, name).restype = C.c_char_p
        L.magnus_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(MatrixStruct), C.POINTER(MatrixStruct), DRIVE,
                                    C.c_void_p, C.c_int, C.POINTER(Options)]
        L.magnus_destroy.argtypes = [C.c_void_p]
        L.magnus_create_xxz.argtypes = [C.POINTER(C.c_void_p), C.POINTER(XxzModel), DRIVE, C.c_void_p, C.c_int,
                                        C.POINTER(Options)]
        L.magnus_describe.argtypes = [C.c_void_p, C.POINTER(PathInfo)]
        L.leja_expmv.argtypes = [C.POINTER(MatrixStruct), C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_void_p,
                                 C.POINTER(ExpmvInfo)]
        L.magnus_step.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_void_p, C.POINTER(StepInfo)]
        L.magnus_integrate.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int64, C.c_void_p, C.POINTER(Stats)]
        L.magnus_integrate_host.argtypes = [C.POINTER(MatrixStruct), C.POINTER(MatrixStruct), DRIVE, C.c_void_p,
                                            C.c_int, C.POINTER(Options), C.c_double, C.c_double, C.c_int64,
                                            C.c_void_p, C.POINTER(Stats)]
        L.magnus_gershgorin.argtypes = [C.POINTER(MatrixStruct), C.POINTER(MatrixStruct), C.c_double, C.c_void_p,
                                        C.POINTER(C.c_double)]
        L.magnus_leja_iteration.argtypes = [C.POINTER(MatrixStruct), C.POINTER(MatrixStruct), C.c_double, C.c_void_p,
                                            C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_double,
                                            C.c_void_p, C.c_int, C.c_int, C.POINTER(C.c_double),
                                            C.POINTER(C.c_float)]
        L.magnus_leja_iteration_dense_noalloc.argtypes = [C.c_int64, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p,
                                                          C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_double,
                                                          C.c_void_p, C.c_void_p]
        L.magnus_zgemm.argtypes = [C.c_int64, C.c_void_p, C.c_int64, C.c_void_p, C.c_int64, C.c_void_p, C.c_int64,
                                   C.c_void_p, C.POINTER(C.c_float)]
        L.magnus_commutator_dense.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.magnus_commutator_csr.argtypes = [C.POINTER(MatrixStruct), C.POINTER(MatrixStruct), C.c_int64,
                                            C.POINTER(C.c_int64), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.magnus_omega_dense.argtypes = [C.c_int64, C.c_void_p, C.c_int64, C.c_void_p, C.c_int64, C.c_double, C.c_double,
                                         C.c_double, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                         C.POINTER(C.c_double)]
        L.magnus_fp64_peaks.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_void_p]
        L.magnus_host_leja_points.argtypes = [C.c_int, C.c_void_p]
        L.magnus_host_divided_differences.argtypes = [C.c_double, C.c_int, C.c_void_p]
        L.magnus_host_snap_interval.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.magnus_host_tridiag_extremes.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.POINTER(C.c_double),
                                                   C.POINTER(C.c_double)]
        L.magnus_host_step_coefficients.argtypes = [C.c_int, DRIVE, C.c_void_p, C.c_double, C.c_double,
                                                    C.POINTER(C.c_double), C.POINTER(C.c_double),
                                                    C.POINTER(C.c_double)]
        _lib = L
    return _lib


def _check(rc: int):
    if rc < 0:
        raise MagnusError(rc, lib().magnus_last_error().decode() or lib().magnus_strerror(rc).decode())
    return rc


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        import torch
        if torch.cuda.is_available():
            return int(torch.cuda.current_stream().cuda_stream) or None
        return None
    if hasattr(stream, "cuda_stream"):
        return int(stream.cuda_stream) or None
    return int(stream) or None


def _ptr(t) -> int:
    return int(t.data_ptr())


@dataclass
class Matrix:
    """A magnus_matrix plus the tensors that own its memory (kept alive here)."""
    struct: MatrixStruct
    keep: tuple

    @property
    def n(self) -> int:
        return int(self.struct.n)

    def ref(self):
        return C.byref(self.struct)


def as_matrix(M) -> Matrix:
    """torch complex128 2-D tensor (row-major) -> DENSE; object with row_ptr/col_idx/values -> CSR."""
    if isinstance(M, Matrix):
        return M
    s = MatrixStruct()
    if hasattr(M, "row_ptr"):
        s.format = CSR
        s.n = int(M.n)
        s.nnz = int(M.col_idx.numel())
        s.values, s.col_idx, s.row_ptr = _ptr(M.values), _ptr(M.col_idx), _ptr(M.row_ptr)
        s.ld = 0
        return Matrix(s, (M.values, M.col_idx, M.row_ptr))
    if M.dim() != 2 or M.shape[0] != M.shape[1] or M.stride(1) != 1:
        raise ValueError("dense matrix must be square and row-major")
    s.format = DENSE
    s.n = int(M.shape[0])
    s.nnz = 0
    s.values = _ptr(M)
    s.ld = int(M.stride(0)) if M.shape[0] > 1 else int(M.shape[0])
    return Matrix(s, (M,))


def _drive(f: Callable[[float], float]):
    return DRIVE(lambda t, _user: float(f(t)))


SHORTCUT_CACHED_COMMUTATOR = 1
SHORTCUT_TIGHT_INTERVAL = 2
SHORTCUT_REAL_VALUES = 4


def _options(tol=None, theta_max=None, m_max=None, check_hermitian=False, stream=None, csr_kernel=0,
             shortcuts=0, lanczos_steps=0) -> Options:
    o = Options()
    o.tol = tol or 0.0
    o.theta_max = theta_max or 0.0
    o.m_max = m_max or 0
    o.check_hermitian = 1 if check_hermitian else 0
    o.stream = _stream_ptr(stream)
    o.csr_kernel = csr_kernel
    o.shortcuts = shortcuts
    o.lanczos_steps = lanczos_steps
    return o


class Handle:
    """magnus_handle with RAII-style close()."""

    def __init__(self, H0, H1, f: Callable[[float], float], scheme, **opts):
        self.H0, self.H1 = as_matrix(H0), as_matrix(H1)
        self._cb = _drive(f)
        self.scheme = SCHEMES[scheme] if isinstance(scheme, str) else int(scheme)
        self._opt = _options(**opts)
        self._h = C.c_void_p()
        _check(lib().magnus_create(C.byref(self._h), self.H0.ref(), self.H1.ref(), self._cb, None, self.scheme,
                                   C.byref(self._opt)))

    @classmethod
    def xxz(cls, nspins: int, jxy: float, jz: float, hx: float, f: Callable[[float], float], scheme, **opts) -> "Handle":
        """Shortcut handle: matrix-free periodic XXZ chain (magnus_create_xxz); commutator-free schemes only."""
        self = cls.__new__(cls)
        self.H0 = self.H1 = None
        self._cb = _drive(f)
        self.scheme = SCHEMES[scheme] if isinstance(scheme, str) else int(scheme)
        self._opt = _options(**opts)
        self._h = C.c_void_p()
        model = XxzModel(int(nspins), 0, float(jxy), float(jz), float(hx))
        _check(lib().magnus_create_xxz(C.byref(self._h), C.byref(model), self._cb, None, self.scheme,
                                       C.byref(self._opt)))
        return self

    def step(self, t: float, tau: float, psi) -> List[dict]:
        info = StepInfo()
        _check(lib().magnus_step(self._h, t, tau, _ptr(psi), C.byref(info)))
        return [info.exp[i].as_dict() for i in range(info.n_exp)]

    def integrate(self, t0: float, t_end: float, nsteps: int, psi, max_exp: Optional[int] = None) -> dict:
        import numpy as np
        cap = max_exp if max_exp is not None else MAX_EXP_PER_STEP * nsteps
        iters = np.zeros(cap, dtype=np.int32)
        st = Stats()
        st.iters = iters.ctypes.data
        st.iters_cap = cap
        _check(lib().magnus_integrate(self._h, t0, t_end, nsteps, _ptr(psi), C.byref(st)))
        return {"total_matvecs": int(st.total_matvecs), "n_exp": int(st.n_exp), "iters": iters[:int(st.n_exp)].copy(),
                "seconds_device": st.seconds_device, "seconds_leja": st.seconds_leja,
                "seconds_commutator": st.seconds_commutator, "kernel_launches": int(st.kernel_launches),
                "lanczos_matvecs": int(st.lanczos_matvecs)}

    def describe(self) -> dict:
        """The kernel that runs the fused Leja iteration for this handle and its algorithmic bytes per launch."""
        info = PathInfo()
        _check(lib().magnus_describe(self._h, C.byref(info)))
        return {"leja_kernel": info.leja_kernel.decode(), "bytes_per_iteration": int(info.bytes_per_iteration),
                "csr_bytes_per_iteration": int(info.csr_bytes_per_iteration), "slices": int(info.slices),
                "slots": int(info.slots), "entries": int(info.entries)}

    def close(self):
        if self._h:
            lib().magnus_destroy(self._h)
            self._h = C.c_void_p()

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def magnus_create(H0, H1, f, scheme, **opts) -> Handle:
    return Handle(H0, H1, f, scheme, **opts)


def magnus_create_xxz(nspins: int, jxy: float, jz: float, hx: float, f, scheme, **opts) -> Handle:
    return Handle.xxz(nspins, jxy, jz, hx, f, scheme, **opts)


def magnus_step(handle: Handle, t: float, tau: float, psi) -> List[dict]:
    return handle.step(t, tau, psi)


def magnus_integrate(handle: Handle, t0: float, t_end: float, nsteps: int, psi) -> dict:
    return handle.integrate(t0, t_end, nsteps, psi)


def magnus_destroy(handle: Handle) -> None:
    handle.close()


def leja_expmv(H, v_in, v_out, h: float, tol: float = 1e-12, stream=None) -> dict:
    Hm = as_matrix(H)
    info = ExpmvInfo()
    rc = lib().leja_expmv(Hm.ref(), _ptr(v_in), _ptr(v_out), h, tol, _stream_ptr(stream), C.byref(info))
    _check(rc)
    return info.as_dict()


def magnus_integrate_host(H0_host, H1_host, f, scheme, t0: float, t_end: float, nsteps: int, psi_host, **opts) -> dict:
    """End to end with HOST tensors (ideally pinned); psi_host is updated in place."""
    import numpy as np
    A, B = as_matrix(H0_host), as_matrix(H1_host)
    cb = _drive(f)
    sc = SCHEMES[scheme] if isinstance(scheme, str) else int(scheme)
    opt = _options(**opts)
    cap = MAX_EXP_PER_STEP * nsteps
    iters = np.zeros(cap, dtype=np.int32)
    st = Stats()
    st.iters = iters.ctypes.data
    st.iters_cap = cap
    _check(lib().magnus_integrate_host(A.ref(), B.ref(), cb, None, sc, C.byref(opt), t0, t_end, nsteps,
                                       _ptr(psi_host), C.byref(st)))
    return {"total_matvecs": int(st.total_matvecs), "n_exp": int(st.n_exp), "iters": iters[:int(st.n_exp)].copy(),
            "seconds_device": st.seconds_device, "seconds_leja": st.seconds_leja,
            "seconds_commutator": st.seconds_commutator, "kernel_launches": int(st.kernel_launches)}


def magnus_gershgorin(H0, H1=None, g: float = 0.0, stream=None) -> Tuple[float, float]:
    A = as_matrix(H0)
    B = as_matrix(H1) if H1 is not None else None
    ab = (C.c_double * 2)()
    _check(lib().magnus_gershgorin(A.ref(), B.ref() if B else None, g, _stream_ptr(stream), ab))
    return ab[0], ab[1]


def magnus_leja_iteration(H0, H1, g: float, w_in, w_out, p, inv_gamma: float, shift: float, d: complex, stream=None,
                          csr_kernel: int = 0, reps: int = 1) -> Tuple[float, float, float]:
    """Returns (sum |w_out|^2, sum |p|^2, ms per launch)."""
    A = as_matrix(H0)
    B = as_matrix(H1) if H1 is not None else None
    sums = (C.c_double * 2)()
    ms = C.c_float()
    _check(lib().magnus_leja_iteration(A.ref(), B.ref() if B else None, g, _ptr(w_in), _ptr(w_out), _ptr(p), inv_gamma,
                                       shift, complex(d).real, complex(d).imag, _stream_ptr(stream), csr_kernel, reps,
                                       sums, C.byref(ms)))
    return sums[0], sums[1], ms.value


NOALLOC_MAX_N = 32768


def magnus_leja_iteration_dense_noalloc(M, w_in, w_out, p, inv_gamma: float, shift: float, d: complex, sums,
                                        stream=None) -> None:
    """The fused dense Leja iteration for callers that must not allocate device memory (a process whose GPU
    memory is owned by a pool, a latency-bound loop): the library's static scratch replaces the workspace, n is
    limited to NOALLOC_MAX_N, calls must not overlap on one GPU.  `M` is an n x n complex128 device tensor (rows
    may be strided), `sums` a device tensor of 2 float64 that receives (sum |w_out|^2, sum |p|^2).  Enqueues only:
    read `sums` after synchronising the stream.  See include/magnus.h."""
    _check(lib().magnus_leja_iteration_dense_noalloc(int(M.shape[0]), _ptr(M), int(M.stride(0)), _ptr(w_in),
                                                     _ptr(w_out), _ptr(p), inv_gamma, shift, complex(d).real,
                                                     complex(d).imag, _stream_ptr(stream), _ptr(sums)))


def magnus_zgemm(A, B, Cout, stream=None) -> float:
    """Cout = A @ B (row-major complex128 device tensors); returns the kernel time in ms."""
    n = int(A.shape[0])
    ms = C.c_float()
    _check(lib().magnus_zgemm(n, _ptr(A), int(A.stride(0)), _ptr(B), int(B.stride(0)), _ptr(Cout),
                              int(Cout.stride(0)), _stream_ptr(stream), C.byref(ms)))
    return ms.value


def magnus_commutator_dense(A, B, K, work, stream=None) -> None:
    _check(lib().magnus_commutator_dense(int(A.shape[0]), _ptr(A), _ptr(B), _ptr(K), _ptr(work), _stream_ptr(stream)))


def magnus_omega_dense(H0, H1, f1: float, f2: float, tau: float, Omega, work_a2, work_p, stream=None) -> Tuple[float, float]:
    """Omega_H of one dense M4 step into `Omega`; returns its raw Gershgorin interval."""
    ab = (C.c_double * 2)()
    _check(lib().magnus_omega_dense(int(H0.shape[0]), _ptr(H0), int(H0.stride(0)), _ptr(H1), int(H1.stride(0)), f1, f2,
                                    tau, _ptr(Omega), _ptr(work_a2), _ptr(work_p), _stream_ptr(stream), ab))
    return ab[0], ab[1]


def magnus_commutator_csr(A, B, stream=None):
    """Returns (row_ptr, col_idx, values) torch tensors on A's device."""
    import torch
    Am, Bm = as_matrix(A), as_matrix(B)
    nnz = C.c_int64(0)
    _check(lib().magnus_commutator_csr(Am.ref(), Bm.ref(), 0, C.byref(nnz), None, None, None, _stream_ptr(stream)))
    dev = A.values.device
    rp = torch.zeros(Am.n + 1, dtype=torch.int32, device=dev)
    ci = torch.zeros(max(1, nnz.value), dtype=torch.int32, device=dev)
    v = torch.zeros(max(1, nnz.value), dtype=torch.complex128, device=dev)
    if nnz.value > 0:
        _check(lib().magnus_commutator_csr(Am.ref(), Bm.ref(), nnz.value, C.byref(nnz), _ptr(rp), _ptr(ci), _ptr(v),
                                           _stream_ptr(stream)))
    return rp, ci[:nnz.value], v[:nnz.value]


def magnus_host_tridiag_extremes(alpha, beta) -> Tuple[float, float]:
    """Extreme eigenvalues of tridiag(alpha; beta) (host; the Sturm bisection of the tight-interval shortcut)."""
    import numpy as np
    al = np.ascontiguousarray(alpha, dtype=np.float64)
    be = np.ascontiguousarray(beta if len(al) > 1 else [0.0], dtype=np.float64)
    lo, hi = C.c_double(), C.c_double()
    _check(lib().magnus_host_tridiag_extremes(al.ctypes.data, be.ctypes.data, len(al), C.byref(lo), C.byref(hi)))
    return lo.value, hi.value


def magnus_fp64_peaks(stream=None) -> Tuple[float, float]:
    a, b = C.c_double(), C.c_double()
    _check(lib().magnus_fp64_peaks(C.byref(a), C.byref(b), _stream_ptr(stream)))
    return a.value, b.value


# ---- host-side pieces (no GPU needed) -----------------------------------------------
def magnus_host_leja_points(m: int):
    import numpy as np
    out = np.empty(m, dtype=np.float64)
    _check(lib().magnus_host_leja_points(m, out.ctypes.data))
    return out


def magnus_host_divided_differences(theta: float, m: int):
    import numpy as np
    out = np.empty(m, dtype=np.complex128)
    _check(lib().magnus_host_divided_differences(theta, m, out.ctypes.data))
    return out


def magnus_host_snap_interval(a: float, b: float) -> Tuple[float, float]:
    ca, cb = C.c_double(a), C.c_double(b)
    _check(lib().magnus_host_snap_interval(C.byref(ca), C.byref(cb)))
    return ca.value, cb.value


def magnus_host_step_coefficients(scheme, f, t: float, tau: float):
    """Returns (coef_h1[:n_exp], h_scale[:n_exp], kappa)."""
    sc = SCHEMES[scheme] if isinstance(scheme, str) else int(scheme)
    coef = (C.c_double * MAX_EXP_PER_STEP)()
    hs = (C.c_double * MAX_EXP_PER_STEP)()
    kappa = C.c_double()
    cb = _drive(f)
    n = _check(lib().magnus_host_step_coefficients(sc, cb, None, t, tau, coef, hs, C.byref(kappa)))
    m = 2 if sc == M4 else (3 if sc == M6 else n)
    return list(coef)[:m], list(hs)[:n], kappa.value


def magnus_version() -> str:
    return lib().magnus_version().decode()
