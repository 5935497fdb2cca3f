"""B200-native hot path of arXiv 1709.06483 (Magnus integrators Cf4 / M4 with
Leja-point interpolation of the matrix exponential).

The product is the C-ABI library libmagnus_b200.so (include/magnus.h), built
from csrc/ by `python -m paper_1709_06483_b200.build`; this package is its
thin ctypes binding.  It never imports `oracle/` and has no CPU fallback.
"""
from .binding import (  # noqa: F401
    CF4, CF4_3, CSR, DENSE, M2, M4, M6, SCHEMES, SHORTCUT_CACHED_COMMUTATOR, SHORTCUT_TIGHT_INTERVAL, SHORTCUT_REAL_VALUES, Handle, MagnusError, leja_expmv, lib, magnus_commutator_csr,
    magnus_commutator_dense, magnus_create, magnus_create_xxz, magnus_destroy, magnus_fp64_peaks, magnus_gershgorin,
    magnus_host_divided_differences, magnus_host_leja_points, magnus_host_snap_interval, magnus_host_tridiag_extremes,
    magnus_host_step_coefficients, magnus_integrate, magnus_integrate_host, magnus_leja_iteration, magnus_leja_iteration_dense_noalloc, magnus_step,
    magnus_omega_dense, magnus_version, magnus_zgemm,
)
