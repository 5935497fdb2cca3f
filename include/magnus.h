/* magnus.h -- C-ABI of the B200-native Magnus/Leja library (libmagnus_b200.so).
 *
 * Hot path of arXiv 1709.06483 ("Magnus integrators on multicore CPUs and
 * GPUs"): one time step of the 4th-order Magnus integrators Cf4 and M4 for
 *     i dpsi/dt = H(t) psi,   H(t) = H0 + f(t) H1            (eq. (1), l.17; l.237)
 * with exp(-i h M) v computed by Newton interpolation at Leja points
 * (section 3, l.169-190) on a Gershgorin spectral interval.
 *
 * "P:n" below = /root/reference/PAPER.md line n.  "c1..c7" = the readings of
 * the paper listed in DESIGN.md section 3.
 *
 * Conventions common to every call
 *   - complex128 everywhere: interleaved (re, im) doubles == cuDoubleComplex ==
 *     torch.complex128.  Indices are int32, 0-based.
 *   - "device" pointers are CUDA device pointers of the current device (e.g. a
 *     torch tensor's data_ptr()); "host" pointers are ordinary host memory.
 *     Unless a call says otherwise, matrix and vector pointers are DEVICE.
 *   - Every call returns an int: MAGNUS_OK (0) or a negative MAGNUS_E* code.
 *     No exception or abort crosses the ABI.  magnus_last_error() returns a
 *     thread-local human-readable detail for the last failure.
 *   - Ownership: the caller owns H0, H1, psi, v; the library never frees,
 *     reallocates or writes H0/H1.  A handle owns only its own workspace.
 *   - Work is enqueued on the options' stream (0 = the legacy default stream;
 *     pass torch.cuda.current_stream().cuda_stream).  Calls synchronise that
 *     stream where a scalar must reach the host (spectral interval, stop test).
 *   - Calls on one handle are not thread-safe.  There is no CPU fallback: with
 *     no usable CUDA device every compute call returns MAGNUS_ECUDA.
 */
#ifndef MAGNUS_B200_H
#define MAGNUS_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MAGNUS_OK             0
#define MAGNUS_EINVAL        -1   /* bad argument (null pointer, n <= 0, format mismatch, ...) */
#define MAGNUS_ENOMEM        -2   /* device or host allocation failed */
#define MAGNUS_ECUDA         -3   /* a CUDA runtime call or kernel launch failed */
#define MAGNUS_ENOCONV       -4   /* m_max reached without meeting tol; psi / v_out unspecified */
#define MAGNUS_ENOTHERMITIAN -5   /* magnus_create's sampled Hermitian check failed */

#define MAGNUS_DENSE 0            /* row-major n x n, leading dimension ld >= n (in elements) */
#define MAGNUS_CSR   1            /* row_ptr[n+1], col_idx[nnz] ascending within a row, values[nnz] */

#define MAGNUS_CF4   0            /* commutator-free, two exponentials  (Method 4) */
#define MAGNUS_M4    1            /* classical, one commutator          (Method 2) */
#define MAGNUS_M2    2            /* exponential midpoint rule          (Method 1) */
#define MAGNUS_CF4_3 3            /* optimised commutator-free, three exponentials (Method 5) */
#define MAGNUS_M6    4            /* sixth order, nested commutators     (Method 3; reading m6) */

#define MAGNUS_MAX_EXP_PER_STEP 3

/* Matrix descriptor.  The matrix must be Hermitian: the dense storage is read
 * ROW-major (reading the same buffer column-major would give conj(H)).
 * CSR: row_ptr[0] == 0, row_ptr[n] == nnz < 2^31, columns sorted ascending and
 * unique within a row.  An absent diagonal entry counts as 0. */
typedef struct magnus_matrix {
  int32_t format;          /* MAGNUS_DENSE or MAGNUS_CSR */
  int32_t reserved;
  int64_t n;               /* dimension */
  int64_t nnz;             /* CSR: stored entries; dense: ignored */
  const void* values;      /* complex128: dense n*ld, CSR nnz */
  const int32_t* col_idx;  /* CSR only */
  const int32_t* row_ptr;  /* CSR only */
  int64_t ld;              /* dense only: row stride in elements (0 means n) */
} magnus_matrix;

/* f(t) of H(t) = H0 + f(t) H1.  Called on the calling host thread, once per
 * quadrature node per step ("computed sequentially (on the CPU)"). */
typedef double (*magnus_drive_fn)(double t, void* user);

/* Options; a NULL pointer or a zero field selects the default. */
typedef struct magnus_options {
  double tol;          /* Leja stopping tolerance, relative 2-norm (c6); default 1e-12 */
  double theta_max;    /* |h gamma| per sub-step (c6); default 16 */
  int32_t m_max;       /* maximal interpolation degree per sub-step (c6); default and maximum 128 */
  int32_t check_hermitian; /* 1: sampled check in magnus_create (costs a device pass); default 0 */
  void* stream;        /* cudaStream_t; NULL = legacy default stream */
  int32_t csr_kernel;  /* 0 auto: CSR n <= 65536 (an 8-CTA cluster up to n = 1024, a cooperative grid above) / dense n <= 4096:
                          whole sweeps per launch and steps planned ahead (magnus_step, below); CSR n > 65536: a handle re-stores the operator once in the offset-slot
                          layout (kernels_csr_slice.cu: 16 B per entry + 8 B per slot, no column array; kept if a slot
                          holds >= 8 entries on average, about 50% more device memory than the caller's CSR) and runs the
                          slice kernel, else the row-block kernel; in between the generic kernel.
                          Non-zero values force a per-iteration kernel and the stepwise control flow:
                          1 generic, 2 row-block, 3 warp-specialised TMA ring, 4 row-block with TMA staging (3 and 4 need
                          16-byte aligned value and index arrays, else the row-block kernel runs), 5 slices with a
                          column array, 6 offset-slot slices; 7 forces the cooperative whole-sweep kernel (n <= 65536);
                          values >= 1000 select tuning variants (kernel sources) */
  int32_t shortcuts;   /* bit mask of beyond-paper shortcuts, default 0 = the mandated path only:
                          MAGNUS_SHORTCUT_CACHED_COMMUTATOR (dense M4), MAGNUS_SHORTCUT_TIGHT_INTERVAL,
                          MAGNUS_SHORTCUT_REAL_VALUES (large CSR) */
  int32_t lanczos_steps; /* MAGNUS_SHORTCUT_TIGHT_INTERVAL: Lanczos steps per exponential; default 8, at most 64 */
} magnus_options;

/* Shortcut (reported separately from the mandated path): for H(t) = H0 + f(t) H1 the commutator of
 * an M4 step is [H(t2), H(t1)] = (f1 - f2) [H0, H1], so on dense H the product P0 = H0 H1 is formed ONCE in
 * magnus_create and a step assembles Omega_H = H0 + fbar H1 - i kappa (P0 - P0^H) without any GEMM (the paper
 * recomputes A2 A1 and A1 A2 every step, P:262 l.6-7; the CSR path always caches [H0, H1], row S0). */
#define MAGNUS_SHORTCUT_CACHED_COMMUTATOR 1

/* Shortcut (SURVEY 8f-4 "tighter spectral interval", reported separately from the mandated path): P:190 only asks
 * for "an estimate on the spectrum"; NS fixes Gershgorin, which over-estimates the radius of a dense random Hermitian
 * matrix 20x to 57x and so costs 1.6-3x more Leja iterations.  With this bit the interval of every exponential of
 * magnus_step / magnus_integrate comes from lanczos_steps steps of the Lanczos process on the exponentiated matrix,
 * started at the current psi:  [theta_min(T) - beta_m, theta_max(T) + beta_m]  (extreme Ritz values widened by the
 * norm of the last residual), intersected with the Gershgorin interval (the estimate is not an enclosure and may
 * stick out of it), then snapped as usual (reading ti).  If it undershoots the spectrum badly the interpolation can
 * fail with MAGNUS_ENOCONV; there is no automatic retry -- repeat the step on a handle without this bit.  Costs lanczos_steps extra mat-vecs per
 * exponential (magnus_stats.lanczos_matvecs); the interval now depends on psi, so steps are not planned ahead. */
#define MAGNUS_SHORTCUT_TIGHT_INTERVAL 2

/* Shortcut (beyond the paper, reported separately from the mandated path, which moves the complex128 values it is
 * given): for a large CSR operator none of whose stored values has an imaginary part -- a real symmetric H0, H1 and
 * therefore [H0, H1], as on the spin chains -- the handle's offset-slot copy keeps the real parts only (8 B per entry
 * instead of 16) and the fused iteration multiplies by them.  Checked exactly in magnus_create; results are identical
 * to the bit (the products left out are multiplications by an exact zero).  No effect on other operators. */
#define MAGNUS_SHORTCUT_REAL_VALUES 4

/* Shortcut (SURVEY 8f-4 "matrix-free XXZ apply", reported separately from the mandated CSR path): the periodic
 * XXZ chain in a transverse field -- the structure of the paper's Example 2 and of BASELINE configs
 * 1, 3, 5 -- described by its couplings instead of by matrices:
 *   H0 = sum over the N periodic nearest-neighbour bonds of  jxy (sx sx + sy sy) + jz sz sz,   H1 = hx sum_i sx_i,
 * n = 2^nspins, sz basis, site j on bit nspins - j (the layout of workloads/xxz.py).  magnus_create_xxz returns a
 * handle for magnus_step / magnus_integrate / magnus_describe / magnus_destroy whose fused Leja iteration
 * recomputes the matrix entries from the row bits and moves vector bytes only; the Gershgorin bounds come from
 * their closed form.  Commutator-free schemes only (MAGNUS_CF4, MAGNUS_M2, MAGNUS_CF4_3; others: MAGNUS_EINVAL);
 * 3 <= nspins <= 30.  Results agree with the CSR path on the same model to rounding (different summation order),
 * iteration counts are equal. */
typedef struct magnus_xxz_model {
  int32_t nspins;
  int32_t reserved;
  double jxy, jz, hx;
} magnus_xxz_model;

/* What one exponential did (reading c4-c7). */
typedef struct magnus_expmv_info {
  int32_t iters;       /* mat-vecs used, summed over sub-steps */
  int32_t substeps;    /* s = max(1, ceil(|h gamma| / theta_max)) */
  int32_t status;      /* MAGNUS_OK or MAGNUS_ENOCONV */
  int32_t reserved;
  double a, b;         /* snapped Gershgorin interval used */
  double theta;        /* (h/s) * gamma */
  double err_est;      /* e_k + e_{k-1} at the stop */
} magnus_expmv_info;

typedef struct magnus_step_info {
  int32_t n_exp;       /* exponentials in this step: CF4 2, M4 1, M2 1, CF4:3 3 */
  int32_t reserved;
  magnus_expmv_info exp[MAGNUS_MAX_EXP_PER_STEP];
} magnus_step_info;

typedef struct magnus_stats {
  int64_t total_matvecs;   /* Leja iterations over the whole call */
  int64_t n_exp;           /* exponentials computed */
  int32_t* iters;          /* caller-provided HOST array (nullable): iterations per exponential, call order */
  int64_t iters_cap;       /* capacity of iters */
  double seconds_device;   /* CUDA-event time of the whole call on the stream */
  double seconds_leja;     /* CUDA-event time spent inside fused Leja-iteration kernels (init..stop) */
  double seconds_commutator; /* CUDA-event time inside the dense commutator GEMM (M4 dense), else 0 */
  int64_t kernel_launches; /* kernels this call enqueued */
  int64_t lanczos_matvecs; /* MAGNUS_SHORTCUT_TIGHT_INTERVAL: mat-vecs spent on interval estimates (not in total_matvecs) */
} magnus_stats;

typedef struct magnus_context* magnus_handle;

/* magnus_create -- set up an integrator for H(t) = H0 + f(t) H1.
 *   H0, H1  device matrices of the same format and n; BORROWED until magnus_destroy
 *           (kept alive and unmodified by the caller).
 *   f,user  the scalar drive; called on the host.
 *   scheme  MAGNUS_CF4 / MAGNUS_M4 / MAGNUS_M2 / MAGNUS_CF4_3 / MAGNUS_M6.
 * Allocates every workspace once (w ping-pong, p, partial-norm buffers; CSR: per-term row
 * statistics for the Gershgorin bounds, 24 n bytes per term, and a test whether the terms'
 * patterns overlap -- c4 takes the modulus of the SUMMED entry, which separates only if
 * they do not; dense: the
 * assembled matrix, and for M4 the node matrices A1, A2 and the product P; CSR
 * M4: computes and owns the sparse commutator C = [H0, H1] -- row S0 of the
 * scope table -- so that a step only rescales it, since
 * [H(t2), H(t1)] = (f1 - f2) [H0, H1]).
 * M6 runs on dense matrices (three FP64 tensor-core GEMMs per step, see magnus_step); CSR input of n <= 16384 --
 * the range the paper runs sparse M6 on -- is expanded into handle-owned dense copies, larger CSR
 * input is refused (EINVAL): the nested commutators fill in.
 * Errors: EINVAL, ENOMEM, ECUDA, ENOTHERMITIAN (only with check_hermitian). */
int magnus_create(magnus_handle* out, const magnus_matrix* H0, const magnus_matrix* H1,
                  magnus_drive_fn f, void* user, int scheme, const magnus_options* opt);

/* magnus_destroy -- frees handle-owned memory only.  NULL is allowed. */
int magnus_destroy(magnus_handle h);

/* leja_expmv -- v_out = exp(-i h H) v_in by Newton interpolation at Leja points
 * (w = Aw - xi w; p = p + d_i w), on the Gershgorin interval of H
 * (c4), with the two-term relative stopping test (c6) and
 * sub-stepping (c6).  H: device matrix (dense or CSR); v_in, v_out: device,
 * n complex128; v_in == v_out allowed; h may be negative or zero.  Standalone:
 * allocates and frees a transient workspace.  stream: cudaStream_t or NULL.
 * info nullable.  Errors: EINVAL, ENOMEM, ECUDA, ENOCONV. */
int leja_expmv(const magnus_matrix* H, const void* v_in, void* v_out, double h, double tol,
               void* stream, magnus_expmv_info* info);

/* magnus_step -- one step t -> t + tau of the handle's scheme, psi (device,
 * n complex128) updated in place.  CF4 (c1): exp(-i tau/2 (H0+g_a H1))
 * then exp(-i tau/2 (H0+g_b H1)).  M4 (c1): one exponential of
 * Omega_H = (H(t1)+H(t2))/2 - i (sqrt(3) tau/12) [H(t2),H(t1)] with h = tau; on dense
 * H the commutator is one FP64 tensor-core complex GEMM per step.  M6 (reading m6): with H2 = H(t2),
 * b2 = (sqrt(15)/3) tau (f3 - f1), b3 = (10/3) tau (f3 - 2 f2 + f1) and A = -iH every nested commutator reduces to a
 * product of Hermitian / anti-Hermitian factors, three GEMMs in all:  G = [H2, H1] = P1 - P1^H (P1 = H2 H1),
 * S = [H2, G] = P2 + P2^H (P2 = H2 G),  L = 20 i tau H2 + i b3 H1 - tau b2 G,
 * R = -i b2 H1 + (tau b3/30) G - (i tau^2 b2/60) S,  Omega_H = H2 + (b3/(12 tau)) H1 + (i/(240 tau)) (P3 - P3^H),
 * P3 = L R;  one exponential with h = tau.  info nullable. */
int magnus_step(magnus_handle h, double t, double tau, void* psi, magnus_step_info* info);

/* magnus_integrate -- nsteps steps of size tau = (t_end - t0)/nsteps from
 * t_n = t0 + n tau (a product, not an accumulated sum).  psi device, in place.
 * Synchronises the stream before returning so that stats (nullable) is valid.  Up to 1365 steps are planned at a
 * time where planning applies (see magnus_step). */
int magnus_integrate(magnus_handle h, double t0, double t_end, int64_t nsteps, void* psi,
                     magnus_stats* stats);

/* magnus_integrate_host -- the same end to end with HOST buffers: H0, H1 (their
 * values / col_idx / row_ptr pointers are HOST memory, ideally pinned) and
 * psi_host (n complex128, in place) are copied to the device, a handle is
 * created, the integration runs, psi is copied back, everything is freed.
 * This is the call bench.py times for its "e2e" number. */
int magnus_integrate_host(const magnus_matrix* H0_host, const magnus_matrix* H1_host,
                          magnus_drive_fn f, void* user, int scheme, const magnus_options* opt,
                          double t0, double t_end, int64_t nsteps, void* psi_host,
                          magnus_stats* stats);

/* ---- single kernels of the path, exposed for parity tests and roofline timing ---- */

/* Gershgorin interval of M = H0 + g*H1 (H1 may be NULL: M = H0), raw (unsnapped):
 * ab_host[0] = min_i(Re M_ii - R_i), ab_host[1] = max_i(Re M_ii + R_i),
 * R_i = sum_{j != i} |M_ij| over the SUMMED entries (c4).  Device matrices. */
int magnus_gershgorin(const magnus_matrix* H0, const magnus_matrix* H1, double g, void* stream,
                      double* ab_host);

/* One fused Leja iteration (row S6 of the scope table) on device vectors:
 *   w_out = inv_gamma * (H0 + g*H1) w_in - shift * w_in;   p += d * w_out;
 *   sums_host[0] = sum |w_out|^2, sums_host[1] = sum |p|^2   (after the update).
 * H1 may be NULL.  w_in and w_out must not alias.  reps >= 1 repeats the launch
 * (ping-ponging nothing: same inputs) and returns the mean kernel time in
 * ms_per_launch (nullable), measured with CUDA events on the stream. */
int magnus_leja_iteration(const magnus_matrix* H0, const magnus_matrix* H1, double g,
                          const void* w_in, void* w_out, void* p, double inv_gamma, double shift,
                          double d_re, double d_im, void* stream, int csr_kernel, int reps,
                          double* sums_host, float* ms_per_launch);

/* magnus_leja_iteration_dense_noalloc -- the same fused iteration (row S6) on a dense row-major matrix,
 * for callers that are not allowed to allocate: a process whose GPU memory already belongs to a pool (a PyTorch
 * caching allocator that has taken the device, a service with a fixed memory budget, a plug-in inside another
 * program's CUDA context) cannot rely on cudaMalloc succeeding, and a latency-bound loop cannot afford it --
 * cudaMalloc / cudaFree take driver-wide locks and cudaFree waits for the device.  Every other reducing entry point
 * here allocates a workspace for its per-block partial sums; this one keeps them in a fixed array inside the library
 * image and calls no cudaMalloc, cudaMallocHost, cudaFree, event/stream creation or allocating library routine.
 *   w_out = inv_gamma * M w_in - shift * w_in;   p += (d_re + i d_im) * w_out;
 *   sums_dev[0] = sum |w_out|^2,  sums_dev[1] = sum |p|^2   (after the update).
 * All pointers are DEVICE pointers owned by the caller: M (n rows of ld >= n complex128, ld = 0 means n), w_in, w_out,
 * p (n complex128, pairwise distinct, 16-byte aligned), sums_dev (2 doubles, written by the kernel).  The call only
 * ENQUEUES on `stream` (a memset of 256 bytes and one kernel) and returns; results are valid in stream order.
 * For n <= MAGNUS_NOALLOC_MAX_N the results equal magnus_leja_iteration's on the same dense matrix bit for bit.
 * Limits and rules:
 *   - n <= MAGNUS_NOALLOC_MAX_N; anything larger returns MAGNUS_EINVAL with a message (nothing is launched).
 *   - The scratch is 65,792 bytes of device memory that every GPU on which this library is loaded holds until the
 *     process exits, used or not.
 *   - One scratch per device, shared by all calls and all threads: calls that may overlap on the GPU (different
 *     streams without an ordering between them) race on it and return wrong sums.  Order them.
 *   - It keeps the previous call's contents; the call itself re-zeroes the one word that has to start at zero.
 *   - The first call on each device (with that device current) resolves the scratch address with
 *     cudaGetSymbolAddress, which can trigger module loading: make it before any stream capture begins.
 * Errors: EINVAL (sizes, null / aliased / misaligned pointers), ECUDA (no device, address lookup or enqueue failed). */
#define MAGNUS_NOALLOC_MAX_N 32768
int magnus_leja_iteration_dense_noalloc(int64_t n, const void* M, int64_t ld, const void* w_in, void* w_out, void* p,
                                        double inv_gamma, double shift, double d_re, double d_im, void* stream,
                                        double* sums_dev);

/* C = A * B, dense row-major complex128 n x n (device), by the FP64 tensor-core
 * (DMMA m8n8k4) kernel used for the M4 commutator (P:262 l.6-7).  C must not
 * alias A or B.  ms (nullable): CUDA-event time of the launch. */
int magnus_zgemm(int64_t n, const void* A, int64_t lda, const void* B, int64_t ldb, void* C,
                 int64_t ldc, void* stream, float* ms);

/* K = A B - B A for Hermitian dense A, B (device): one GEMM P = A B and
 * K = P - P^H (P:262 l.6-8; exact identity for Hermitian operands).
 * work: device scratch of n*n complex128. */
int magnus_commutator_dense(int64_t n, const void* A, const void* B, void* K, void* work,
                            void* stream);

/* Omega_H of one M4 step on dense H (rows S2, D3, D4, S3 of the scope table; P:99, P:262 l.3-9 with A = -iH; c1):
 *   A1 = H0 + f1 H1, A2 = H0 + f2 H1, P = A2 A1 (FP64 tensor-core GEMM),
 *   Omega = (A1 + A2)/2 - i (sqrt(3) tau / 12) (P - P^H),
 * exactly the launches magnus_step makes, exposed so that the assembled matrix can be compared entry by entry with
 * the plain definition.  H0, H1 device, row-major, leading dimensions ld0, ld1 (0 = n), Hermitian.  Omega, work_a2,
 * work_p: device, n*n complex128 each, pairwise distinct; Omega receives the result.  ab_host (nullable): raw
 * Gershgorin interval of Omega.  Errors: EINVAL, ENOMEM, ECUDA. */
int magnus_omega_dense(int64_t n, const void* H0, int64_t ld0, const void* H1, int64_t ld1, double f1, double f2,
                       double tau, void* Omega, void* work_a2, void* work_p, void* stream, double* ab_host);

/* C = A B - B A for CSR A, B (device), exact zeros dropped.  Two-call protocol:
 * with cap_nnz == 0 only *nnz_out is written; otherwise row_ptr_out[n+1],
 * col_idx_out, values_out (device, capacity cap_nnz) are filled.
 * Limits (also for magnus_create with MAGNUS_M4 on CSR input, which calls this): a row i is built from
 * the rows B_k (k in A's row i) and A_k (k in B's row i); up to 256 such source rows with at most 1024
 * entries in total and 32 resulting entries are handled by a warp, anything beyond by a CTA that holds at
 * most 2048 candidate products -- a row that needs more returns MAGNUS_EINVAL (spin chains need 2 N^2).
 * Needs temporary device memory of 640 bytes per row. */
int magnus_commutator_csr(const magnus_matrix* A, const magnus_matrix* B, int64_t cap_nnz,
                          int64_t* nnz_out, int32_t* row_ptr_out, int32_t* col_idx_out,
                          void* values_out, void* stream);

int magnus_create_xxz(magnus_handle* out, const magnus_xxz_model* model, magnus_drive_fn f, void* user, int scheme,
                      const magnus_options* opt);

/* What the handle will run for the fused Leja iteration (row S6) and what that kernel moves per launch.
 * Measurement support (bench.py reports the roofline against THESE bytes: "never count bytes a
 * variant does not move").  leja_kernel is the kernel's name; bytes_per_iteration its algorithmic HBM bytes for
 * one iteration of the handle's operator (CSR: all terms of the scheme -- H0, H1 and, for M4, C; dense:
 * 16 n^2 + 64 n); csr_bytes_per_iteration the same for plain CSR storage, 20 nnz + 4 (n + 1) terms + 64 n
 * (0 for dense).  slices / slots / entries describe the slice-major copy when one was built (else 0):
 * the offset-slot layout moves 16 B per entry + 8 B per slot + 24 B per slice + 64 B per row. */
typedef struct magnus_path_info {
  char leja_kernel[64];
  int64_t bytes_per_iteration;
  int64_t csr_bytes_per_iteration;
  int64_t slices, slots, entries;
} magnus_path_info;
int magnus_describe(magnus_handle h, magnus_path_info* out);

/* Register-resident micro-benchmarks that fix the ALU-side roofline denominators
 * (no FP64 peak is in MEASURED_PEAKS.json): DMMA m8n8k4 and plain DFMA, TFLOP/s. */
int magnus_fp64_peaks(double* dmma_tflops, double* dfma_tflops, void* stream);

/* ---- host-side pieces of the path (no GPU needed; used by the CPU tests) ---- */

/* The first m Leja points of [-2, 2] (c2).  out_host: m doubles, m <= 129. */
int magnus_host_leja_points(int m, double* out_host);

/* d_k = exp(-i theta x)[l_0..l_k], k < m (c3), out_host: m complex128. */
int magnus_host_divided_differences(double theta, int m, double* out_host);

/* Widen [a,b] outward to the grid of spacing 2^(ceil(log2(b-a)) - 12) (c4). */
int magnus_host_snap_interval(double* a, double* b);
/* Extreme eigenvalues of the symmetric tridiagonal matrix with diagonal alpha[0..k) and off-diagonal beta[0..k-1)
 * (HOST arrays; Sturm-count bisection): the host piece of MAGNUS_SHORTCUT_TIGHT_INTERVAL (reading ti). */
int magnus_host_tridiag_extremes(const double* alpha_host, const double* beta_host, int k, double* lo, double* hi);

/* Per-exponential scalars of one step (c1).  coef_h1[e] multiplies H1 in the e-th
 * exponential's matrix, h_scale[e]*tau is its h; for M4 kappa_out receives
 * (sqrt(3) tau / 12) (f1 - f2), the factor of -i [H0, H1].  Returns n_exp. */
int magnus_host_step_coefficients(int scheme, magnus_drive_fn f, void* user, double t, double tau,
                                  double* coef_h1, double* h_scale, double* kappa_out);

const char* magnus_strerror(int code);
const char* magnus_last_error(void);
const char* magnus_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MAGNUS_B200_H */
