// C-ABI entry points (include/magnus.h) and the host-side step driver:
// rows S1, S4 and the control flow of S5-S8 ("The control structures are
// executed in sequence (on the CPU), while the vector and matrix operations ...
// are parallelized").  Every arithmetic step on vectors and matrices runs in the
// CUDA kernels of this library; there is no CPU fallback.
#include "magnus_internal.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <vector>

namespace magnus {

const int kM6DenseMaxN = 16384;
const int64_t kSliceAutoMinN = 32768;     // csr_kernel 0: from this n on, try the offset-slot layout (kernels_csr_slice.cu)
const double kSliceAutoMinFill = 8.0;     // ... and keep it if a slot holds at least this many entries on average   // CSR input of MAGNUS_M6 is expanded into dense copies up to this n

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
}

#define CU_TRY(expr)                                                                        \
  do {                                                                                      \
    cudaError_t _e = (expr);                                                                \
    if (_e != cudaSuccess) {                                                                \
      set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
      return MAGNUS_ECUDA;                                                                  \
    }                                                                                       \
  } while (0)

static int require_device() {
  int count = 0;
  const cudaError_t e = cudaGetDeviceCount(&count);
  if (e != cudaSuccess || count <= 0) {
    set_error("no usable CUDA device (%s); this library has no CPU fallback",
              e == cudaSuccess ? "device count 0" : cudaGetErrorString(e));
    cudaGetLastError();
    return MAGNUS_ECUDA;
  }
  return MAGNUS_OK;
}

static int check_matrix(const magnus_matrix* M, const char* name) {
  if (!M) { set_error("%s is NULL", name); return MAGNUS_EINVAL; }
  if (M->n <= 0) { set_error("%s: n must be positive", name); return MAGNUS_EINVAL; }
  if (!M->values) { set_error("%s: values is NULL", name); return MAGNUS_EINVAL; }
  if (M->format == MAGNUS_CSR) {
    if (!M->col_idx || !M->row_ptr) { set_error("%s: CSR needs col_idx and row_ptr", name); return MAGNUS_EINVAL; }
    if (M->nnz < 0 || M->nnz >= (int64_t)1 << 31) { set_error("%s: nnz must be in [0, 2^31)", name); return MAGNUS_EINVAL; }
    if (M->n >= (int64_t)1 << 31) { set_error("%s: n must be < 2^31", name); return MAGNUS_EINVAL; }
  } else if (M->format == MAGNUS_DENSE) {
    if (M->ld != 0 && M->ld < M->n) { set_error("%s: ld < n", name); return MAGNUS_EINVAL; }
  } else {
    set_error("%s: unknown format %d", name, M->format);
    return MAGNUS_EINVAL;
  }
  return MAGNUS_OK;
}

static int64_t dense_ld(const magnus_matrix* M) { return M->ld ? M->ld : M->n; }

static CsrTerm csr_term(const magnus_matrix* M, double re, double im) {
  CsrTerm t;
  t.rp = M->row_ptr;
  t.ci = M->col_idx;
  t.v = (const cplx*)M->values;
  t.coef = make_double2(re, im);
  t.nnz = M->nnz;
  return t;
}

// Either a CSR operator formed on the fly or a dense (assembled) matrix.
struct OpRef {
  bool dense;
  CsrOp csr;
  DenseOp dns;
  bool xxz = false;     // matrix-free XXZ chain (shortcut): csr and dns unused
  XxzOp xx;
};

static int read_interval(int nblk, Workspace* ws, cudaStream_t st, double* a, double* b) {
  (void)nblk;   // the min/max over blocks is taken by the last block of the producing kernel
  CU_TRY(cudaGetLastError());   // a failed launch of the producing kernel must not turn into a garbage interval
  CU_TRY(cudaMemcpyAsync(ws->ab_host, ws->gersh + 2 * kMaxPartials, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
  CU_TRY(cudaStreamSynchronize(st));
  *a = ws->ab_host[0];
  *b = ws->ab_host[1];
  return MAGNUS_OK;
}

static int op_interval(const OpRef& op, Workspace* ws, cudaStream_t st, double* a, double* b) {
  const int nblk = op.dense ? launch_dense_gershgorin(op.dns, ws, st) : launch_csr_gershgorin(op.csr, ws, st);
  return read_interval(nblk, ws, st, a, b);
}

static int launch_iter(const OpRef& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma, double shift,
                       cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st) {
  if (op.xxz) return launch_xxz_leja_iter(op.xx, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws, st);
  return op.dense ? launch_dense_leja_iter(op.dns, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws, st)
                  : launch_csr_leja_iter(op.csr, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws, st);
}

// Divided differences of one exponential (c3), computed lazily: first the terms a sweep can possibly need
// for this theta, the rest (up to m_max) only if the stop test asks for more.
struct LejaTable {
  double theta;
  int full, have;
  double tol;
  int m_max;
  std::vector<std::complex<double>> d;
  LejaTable(double theta_, const LejaParams& prm)
      : theta(theta_), full(prm.m_max + 1), tol(prm.tol), m_max(prm.m_max), d((size_t)prm.m_max + 1) {
    have = std::min(full, std::max(16, (int)std::ceil(2.5 * std::fabs(theta)) + 20));
    divided_differences(theta, have, d.data());
  }
  void need(int k) {   // grows geometrically: a longer table costs O(length^2) host work
    if (k < have) return;
    while (k >= have) have = std::min(full, 2 * have);
    divided_differences(theta, have, d.data());
  }
  // a-priori length of the first chunk: first k with |d_k| + |d_{k-1}| <= tol, plus 2
  int first_chunk() {
    for (int k = 1; k <= m_max; ++k) {
      need(k);
      if (std::abs(d[k]) + std::abs(d[k - 1]) <= tol) return std::min(m_max, k + 2);
    }
    return m_max;
  }
};

// ---------------------------------------------------------------------------
// exp(-i h M) v on the RAW Gershgorin interval [a_raw, b_raw] of M (S4-S8).
//   B = (M - cI)/gamma, theta = (h/s) gamma, d_k = exp(-i theta x)[l_0..l_k]        (c3)
//   w_0 = v, p_0 = d_0 v;  w_k = (1/gamma) M w_{k-1} - (c/gamma + l_{k-1}) w_{k-1};
//   p_k = p_{k-1} + d_k w_k                                                          (c5)
//   stop at the first k >= 1 with e_k + e_{k-1} <= tol ||p_k||, e_k = |d_k| ||w_k||    (c6)
// The stop test is evaluated on the device by the last block of every iteration
// kernel; iteration kernels launched after it fired return immediately.  The host launches a
// first chunk sized from the table alone (|d_k| + |d_{k-1}| <= tol) plus two,
// then polls the device status every four iterations.
// ---------------------------------------------------------------------------
static int expmv_on_interval(const OpRef& op, double a_raw, double b_raw, const cplx* v_in, cplx* v_out, double h,
                             const LejaParams& prm, Workspace* ws, cudaStream_t st, magnus_expmv_info* info) {
  const int64_t n = op.xxz ? (int64_t)1 << op.xx.nspins : op.dense ? op.dns.n : op.csr.n;
  double a = a_raw, b = b_raw;
  if (!std::isfinite(a) || !std::isfinite(b)) {
    set_error("Gershgorin interval is not finite (NaN/Inf in the matrix?)");
    return MAGNUS_EINVAL;
  }
  snap_interval(&a, &b);
  const double c = 0.5 * (a + b), gamma = 0.25 * (b - a);
  magnus_expmv_info loc;
  std::memset(&loc, 0, sizeof loc);
  loc.a = a;
  loc.b = b;
  if (!(gamma > 0.0)) {   // M = c I: exact, no iterations (c4)
    launch_scale_copy(v_in, v_out, n, make_double2(std::cos(h * c), -std::sin(h * c)), st, ws);
    loc.substeps = 1;
    if (info) *info = loc;
    return MAGNUS_OK;
  }
  const int s = std::max(1, (int)std::ceil(std::fabs(h * gamma) / prm.theta_max));
  const double hs = h / s, theta = hs * gamma;
  loc.substeps = s;
  loc.theta = theta;

  const double* l = leja_points();
  LejaTable T(theta, prm);
  std::vector<std::complex<double>>& d = T.d;
  int& have = T.have;
  auto need = [&](int k) { T.need(k); };
  const int first_chunk = T.first_chunk();

  const double inv_gamma = 1.0 / gamma, c_over_gamma = c / gamma;
  const cplx phase = make_double2(std::cos(hs * c), -std::sin(hs * c));
  float ms = 0.f;
  const bool mid_csr = !op.xxz && !op.dense && csr_mid_sweep_supported(n, ws->csr_kernel);
  const bool small_csr = !op.xxz && !op.dense && n <= kSmallSweepMaxN && ws->csr_kernel == 0 && !mid_csr;
  const bool mid_dense = !op.xxz && op.dense && dense_sweep_supported(n) && op.dns.ld == n && ws->csr_kernel == 0;
  if (small_csr || mid_dense || mid_csr) {
    // small CSR / medium dense problem: each sub-step sweep is ONE launch (kernels_csr_small.cu,
    // kernels_dense_sweep.cu) on an already assembled operator; the table first covers `have` terms and is
    // extended only if the sweep asks for more
    SweepTable tab;
    for (int sub = 0; sub < s; ++sub) {
      const cplx* src = sub == 0 ? v_in : v_out;
      int m_try = std::min(prm.m_max, std::max(have - 1, first_chunk));
      while (true) {
        need(m_try);
        for (int k = 0; k <= m_try; ++k) {
          tab.d[k] = make_double2(d[k].real(), d[k].imag());
          tab.l[k] = l[k];
        }
        CU_TRY(cudaMemsetAsync(ws->status, 0, sizeof(LejaStatus), st));
        if (ws->time_leja) CU_TRY(cudaEventRecord(ws->ev[0], st));
        const int lrc = small_csr ? launch_csr_leja_sweep_small(op.csr, src, v_out, inv_gamma, c_over_gamma, prm.tol, m_try,
                                                                phase, tab, ws, st)
                        : mid_csr ? launch_csr_leja_sweep_mid(op.csr, src, v_out, inv_gamma, c_over_gamma, prm.tol, m_try, phase,
                                                              tab, ws, st)
                                  : launch_dense_leja_sweep(op.dns, src, v_out, inv_gamma, c_over_gamma, prm.tol, m_try,
                                                            phase, tab, ws, st);
        if (lrc) {
          set_error("whole-sweep launch failed: %s", cudaGetErrorString(cudaGetLastError()));
          return MAGNUS_ECUDA;
        }
        if (ws->time_leja) CU_TRY(cudaEventRecord(ws->ev[1], st));
        CU_TRY(cudaMemcpyAsync(ws->status_host, ws->status, sizeof(LejaStatus), cudaMemcpyDeviceToHost, st));
        CU_TRY(cudaStreamSynchronize(st));
        if (ws->time_leja) {
          CU_TRY(cudaEventElapsedTime(&ms, ws->ev[0], ws->ev[1]));
          ws->leja_ms += ms;
        }
        loc.err_est = ws->status_host->err_est;
        if (ws->status_host->done) {
          loc.iters += ws->status_host->k;
          break;
        }
        if (m_try >= prm.m_max) {
          loc.iters += ws->status_host->k;
          loc.status = MAGNUS_ENOCONV;
          if (info) *info = loc;
          set_error("Leja interpolation did not reach tol=%g within m_max=%d (theta=%g)", prm.tol, prm.m_max, theta);
          return MAGNUS_ENOCONV;
        }
        m_try = prm.m_max;   // the input vector is untouched (nothing is written without convergence): redo in full
      }
    }
    CU_TRY(cudaGetLastError());
    if (info) *info = loc;
    return MAGNUS_OK;
  }
  CU_TRY(cudaMemsetAsync(ws->status, 0, sizeof(LejaStatus), st));
  for (int sub = 0; sub < s; ++sub) {
    const cplx* src = sub == 0 ? v_in : v_out;
    if (ws->time_leja) CU_TRY(cudaEventRecord(ws->ev[0], st));
    launch_leja_init(src, ws->w[0], ws->p, n, make_double2(d[0].real(), d[0].imag()), std::abs(d[0]), ws, st);
    int k = 0;
    bool done = false;
    int chunk_end = first_chunk;
    while (!done && k < prm.m_max) {
      for (; k < chunk_end;) {
        ++k;
        need(k);
        const double shift = c_over_gamma + l[k - 1];
        if (launch_iter(op, ws->w[(k - 1) & 1], ws->w[k & 1], ws->p, inv_gamma, shift,
                        make_double2(d[k].real(), d[k].imag()), std::abs(d[k]), prm.tol, ws, st) < 0) {
          // nothing was launched (a csr_kernel tuning code outside the launch tables): without this the host would
          // poll an unchanged status up to m_max and report a misleading ENOCONV
          set_error("csr_kernel = %d selects no kernel for this operator (valid: 0 auto, 1 generic, 2 row-block, 3, 4, "
                    "5, 6 offset-slot, 7 sweep, or a tuning code listed in the kernel sources)", ws->csr_kernel);
          return MAGNUS_EINVAL;
        }
      }
      CU_TRY(cudaGetLastError());   // a failed launch must surface as ECUDA, not as ENOCONV at m_max
      if (ws->time_leja) CU_TRY(cudaEventRecord(ws->ev[1], st));
      CU_TRY(cudaMemcpyAsync(ws->status_host, ws->status, sizeof(LejaStatus), cudaMemcpyDeviceToHost, st));
      CU_TRY(cudaStreamSynchronize(st));
      if (ws->time_leja) {
        CU_TRY(cudaEventElapsedTime(&ms, ws->ev[0], ws->ev[1]));
        ws->leja_ms += ms;
        CU_TRY(cudaEventRecord(ws->ev[0], st));
      }
      done = ws->status_host->done != 0;
      chunk_end = std::min(prm.m_max, k + 4);
    }
    loc.iters = ws->status_host->iters;
    loc.err_est = ws->status_host->err_est;
    if (!done) {
      loc.status = MAGNUS_ENOCONV;
      if (info) *info = loc;
      set_error("Leja interpolation did not reach tol=%g within m_max=%d (theta=%g)", prm.tol, prm.m_max, theta);
      return MAGNUS_ENOCONV;
    }
    launch_leja_finish(ws->p, v_out, n, phase, st, ws);   // c7
  }
  CU_TRY(cudaGetLastError());
  if (info) *info = loc;
  return MAGNUS_OK;
}

static void default_params(const magnus_options* opt, LejaParams* prm, cudaStream_t* st, int* csr_kernel,
                           int* shortcuts) {
  *shortcuts = opt ? opt->shortcuts : 0;
  prm->tol = (opt && opt->tol > 0.0) ? opt->tol : 1e-12;
  prm->theta_max = (opt && opt->theta_max > 0.0) ? opt->theta_max : 16.0;
  prm->m_max = (opt && opt->m_max > 0 && opt->m_max <= kMaxDegree) ? opt->m_max : kMaxDegree;
  *st = opt ? (cudaStream_t)opt->stream : (cudaStream_t)0;
  *csr_kernel = opt ? opt->csr_kernel : 0;
}

}  // namespace magnus

using namespace magnus;

struct magnus_context {
  int scheme = 0;
  int format = 0;
  int shortcuts = 0;
  bool cached_p0 = false;      // dense M4 shortcut: h->P holds P0 = H0 H1
  ZgemmScratch zs;             // dense M4 / M6: workspace of the split-tail GEMM
  int lanczos_steps = 8;       // tight-interval shortcut
  cplx* lz[2] = {nullptr, nullptr};   // ... its Lanczos vectors q_j, q_{j-1}
  double* lz_scal = nullptr;          // ... and device scalars (norm, beta_prev, alpha[], beta[])
  int64_t lanczos_matvecs = 0;
  bool is_xxz = false;         // matrix-free XXZ shortcut: no matrices, format is MAGNUS_CSR only nominally
  magnus_xxz_model xxz_model;
  int64_t n = 0;
  magnus_matrix H0, H1;
  magnus_drive_fn f = nullptr;
  void* user = nullptr;
  LejaParams prm;
  cudaStream_t stream = 0;
  Workspace ws;
  // dense: assembled matrix (commutator-free schemes) or A1 (M4; Omega_H overwrites it), A2, P; M6: two more
  cplx* M = nullptr;
  cplx* A2 = nullptr;
  cplx* P = nullptr;
  cplx* X4 = nullptr;
  cplx* X5 = nullptr;
  // M6 on CSR input (n <= kM6DenseMaxN): handle-owned dense copies of H0, H1
  cplx* d0 = nullptr;
  cplx* d1 = nullptr;
  // CSR M4: cached C = [H0, H1] (row S0)
  int32_t* c_rp = nullptr;
  int32_t* c_ci = nullptr;
  cplx* c_v = nullptr;
  int64_t c_nnz = 0;
  // CSR: cached per-term row statistics for the Gershgorin bounds (valid while the terms' patterns are disjoint)
  double* gs_r[3] = {nullptr, nullptr, nullptr};
  cplx* gs_diag[3] = {nullptr, nullptr, nullptr};
  SliceLayout slice;           // CSR: slice-major copy of (H0, H1[, C]) for the slice kernel (csr_kernel 5)
  bool gs_disjoint2 = false;   // H0, H1 share no (row, column)
  bool gs_disjoint3 = false;   // H0, H1, C share none either
  int unit_cap2 = 0, unit_cap3 = 0;   // stream kernel: largest 32-row unit of (H0, H1) and of (H0, H1, C)
  cudaEvent_t ev_comm[2] = {nullptr, nullptr};
  double comm_ms = 0.0;
  bool time_comm = false;
};

// Row statistics r^t, diag^t of every CSR term and the overlap flags (see csr_gershgorin_cached_kernel).
static int csr_cache_rowstats(magnus_context* h) {
  const int64_t n = h->n;
  CsrTerm T[3];
  T[0] = csr_term(&h->H0, 1.0, 0.0);
  T[1] = csr_term(&h->H1, 1.0, 0.0);
  int nterms = 2;
  if (h->scheme == MAGNUS_M4 && h->c_nnz > 0) {
    T[2].rp = h->c_rp;
    T[2].ci = h->c_ci;
    T[2].v = h->c_v;
    T[2].coef = make_double2(1.0, 0.0);
    T[2].nnz = h->c_nnz;
    nterms = 3;
  }
  int* flags = nullptr;
  if (cudaMalloc(&flags, 2 * sizeof(int)) != cudaSuccess) { cudaGetLastError(); return MAGNUS_ENOMEM; }
  cudaMemsetAsync(flags, 0, 2 * sizeof(int), h->stream);
  for (int t = 0; t < nterms; ++t) {
    if (cudaMalloc(&h->gs_r[t], sizeof(double) * (size_t)n) != cudaSuccess ||
        cudaMalloc(&h->gs_diag[t], sizeof(cplx) * (size_t)n) != cudaSuccess) {
      cudaGetLastError();
      cudaFree(flags);
      set_error("row-statistics allocation failed (n=%lld)", (long long)n);
      return MAGNUS_ENOMEM;
    }
    launch_csr_rowstats(T[t], n, h->gs_r[t], h->gs_diag[t], h->stream);
  }
  CsrOp op;
  op.n = n;
  op.unit_cap = 0;
  for (int t = 0; t < 3; ++t) op.t[t] = T[t < nterms ? t : 0];
  op.nterms = 2;
  launch_csr_overlap(op, flags, h->stream);
  if (nterms == 3) {
    op.nterms = 3;
    launch_csr_overlap(op, flags + 1, h->stream);
  }
  int hf[2] = {1, 1};
  cudaMemcpyAsync(hf, flags, 2 * sizeof(int), cudaMemcpyDeviceToHost, h->stream);
  const cudaError_t e = cudaStreamSynchronize(h->stream);
  cudaFree(flags);
  if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) { set_error("row-statistics kernels failed"); return MAGNUS_ECUDA; }
  h->gs_disjoint2 = hf[0] == 0;
  h->gs_disjoint3 = nterms == 3 && hf[1] == 0;
  {
    op.nterms = 2;
    if (csr_unit_cap(op, h->stream, &h->unit_cap2) != MAGNUS_OK) h->unit_cap2 = 0;
    op.nterms = 3;
    if (nterms == 3 && csr_unit_cap(op, h->stream, &h->unit_cap3) != MAGNUS_OK) h->unit_cap3 = 0;
  }
  return MAGNUS_OK;
}

// ---------------------------------------------------------------------------
// Planned batches (small and medium problems, where a step is a handful of microseconds of kernel time
// and every host round trip shows).  The Gershgorin interval of an exponential depends on t only, not
// on psi, so a run of steps is planned ahead: every interval of the batch first (one host sync), the
// tables d_k on the host, one SweepJob per exponential, then the whole-sweep kernel runs the jobs back
// to back with no host in between and the host reads all the stop-test records at the end (second
// sync).  A job that does not meet tol within its table stops the batch with psi untouched by it; the
// host redoes that exponential on the stepwise path and resumes the batch behind it.
// ---------------------------------------------------------------------------
struct ExpSpec {
  double g;       // coefficient of H1
  double kappa;   // CSR M4: the coefficient of C = [H0, H1] is -i kappa
  int nterms;     // CSR terms in use
  double h;       // the exponential is exp(-i h M)
};

static void csr_op_from_spec(const magnus_context* h, const ExpSpec& sp, CsrOp* op) {
  op->n = h->n;
  op->nterms = sp.nterms;
  op->t[0] = csr_term(&h->H0, 1.0, 0.0);
  op->t[1] = csr_term(&h->H1, sp.g, 0.0);
  op->t[2] = op->t[1];
  if (h->c_v) {   // Omega_H = H0 + fbar H1 - i kappa [H0, H1]   (c1; [H(t2),H(t1)] = (f1 - f2)[H0,H1])
    CsrTerm c;
    c.rp = h->c_rp;
    c.ci = h->c_ci;
    c.v = h->c_v;
    c.coef = make_double2(0.0, -sp.kappa);
    c.nnz = h->c_nnz;
    op->t[2] = c;
  }
  op->unit_cap = sp.nterms == 3 ? h->unit_cap3 : h->unit_cap2;
  op->slice = h->slice.meta ? &h->slice : nullptr;
}

// the exponentials of one step (S1) for the operators that are a plain combination of stored terms:
// commutator-free schemes on either format, and M4 on CSR with its cached commutator
static void specs_from_coefficients(const magnus_context* h, int n_exp, const double* coef, const double* hscale, double kappa,
                                    double tau, ExpSpec* out) {
  for (int e = 0; e < n_exp; ++e) {
    out[e].g = coef[e];
    out[e].kappa = 0.0;
    out[e].nterms = 2;
    out[e].h = hscale[e] * tau;
  }
  if (h->scheme == MAGNUS_M4 && h->format == MAGNUS_CSR) {
    out[0].g = 0.5 * (coef[0] + coef[1]);
    out[0].kappa = kappa;
    out[0].nterms = (h->c_nnz > 0 && kappa != 0.0) ? 3 : 2;
  }
}

static int step_specs(magnus_context* h, double t, double tau, ExpSpec* out) {
  double coef[MAGNUS_MAX_EXP_PER_STEP], hscale[MAGNUS_MAX_EXP_PER_STEP], kappa = 0.0;
  const int n_exp = step_coefficients(h->scheme, h->f, h->user, t, tau, coef, hscale, &kappa);
  specs_from_coefficients(h, n_exp, coef, hscale, kappa, tau, out);
  return n_exp;
}

static bool plan_supported(const magnus_context* h) {
  if (h->is_xxz || (h->shortcuts & MAGNUS_SHORTCUT_TIGHT_INTERVAL)) return false;   // the interval depends on psi
  if (h->format == MAGNUS_CSR)
    return (h->n <= kSmallSweepMaxN && h->ws.csr_kernel == 0) || csr_mid_sweep_supported(h->n, h->ws.csr_kernel);
  // dense: the commutator-free schemes (M = H0 + g H1 per exponential); M4 / M6 build Omega_H per step
  return h->scheme != MAGNUS_M4 && h->scheme != MAGNUS_M6 && dense_sweep_supported(h->n) && h->ws.csr_kernel == 0;
}

const int kPlanDeclined = 1;   // internal: not a planned-path handle after all

// Steps s0 .. s0 + ns - 1 of the grid t0 + s tau (at most kPlanCap exponentials); infos (nullable) gets one entry
// per step.  Host planning (tables, jobs) of launch i + 1 overlaps the device's work on launch i: jobs go
// through a ring of kJobRing slots of kJobsPerLaunch jobs, each guarded by the event of its last launch.
static int run_planned(magnus_context* h, double t0, double tau, int64_t s0, int ns, cplx* psi, magnus_step_info* infos) {
  Workspace* ws = &h->ws;
  cudaStream_t st = h->stream;
  if (ensure_sweep_jobs(ws, st) != MAGNUS_OK) { set_error("planned batch: buffer allocation failed"); return MAGNUS_ENOMEM; }
  std::vector<ExpSpec> specs;
  std::vector<int> first_of_step((size_t)ns + 1, 0);
  for (int s = 0; s < ns; ++s) {
    ExpSpec sp[MAGNUS_MAX_EXP_PER_STEP];
    const int n_exp = step_specs(h, t0 + (double)(s0 + s) * tau, tau, sp);   // S1
    first_of_step[s] = (int)specs.size();
    for (int e = 0; e < n_exp; ++e) specs.push_back(sp[e]);
  }
  const int E = (int)specs.size();
  first_of_step[ns] = E;
  if (E > kPlanCap) { set_error("planned batch too long"); return MAGNUS_EINVAL; }

  const bool dense = h->format == MAGNUS_DENSE;
  const cplx* H0v = (const cplx*)h->H0.values;
  const cplx* H1v = (const cplx*)h->H1.values;
  std::vector<double> ab((size_t)2 * E);   // raw Gershgorin bounds of every exponential
  // S3 for the whole batch: one launch when the cached row statistics apply to every exponential
  bool all_cached = !dense;
  for (int e = 0; e < E; ++e)
    all_cached = all_cached && ((specs[e].nterms == 2 && h->gs_disjoint2) || (specs[e].nterms == 3 && h->gs_disjoint3));
  if (all_cached || dense) {
    for (int e = 0; e < E; ++e) {
      ws->coef_arr_host[4 * e] = specs[e].g;
      ws->coef_arr_host[4 * e + 1] = specs[e].kappa;
      ws->coef_arr_host[4 * e + 2] = (double)specs[e].nterms;
      ws->coef_arr_host[4 * e + 3] = 0.0;
    }
    CU_TRY(cudaMemcpyAsync(ws->coef_arr, ws->coef_arr_host, sizeof(double) * 4 * (size_t)E, cudaMemcpyHostToDevice, st));
    if (dense) {
      if (launch_dense_gershgorin_batch(h->n, H0v, dense_ld(&h->H0), H1v, dense_ld(&h->H1), ws->coef_arr, E, ws->ab_arr, ws,
                                        st) != MAGNUS_OK) {
        set_error("batched Gershgorin launch failed");
        return MAGNUS_ECUDA;
      }
    } else {
      launch_csr_gershgorin_cached_batch(h->n, h->gs_r, h->gs_diag, h->gs_r[2] ? 3 : 2, ws->coef_arr, E, ws->ab_arr, ws, st);
    }
  } else {
    for (int e = 0; e < E; ++e) {
      CsrOp op;
      csr_op_from_spec(h, specs[e], &op);
      ws->ab_out = ws->ab_arr + 2 * e;
      if ((op.nterms == 2 && h->gs_disjoint2) || (op.nterms == 3 && h->gs_disjoint3))
        launch_csr_gershgorin_cached(op, h->gs_r, h->gs_diag, ws, st);
      else
        launch_csr_gershgorin(op, ws, st);
    }
    ws->ab_out = nullptr;
  }
  CU_TRY(cudaMemcpyAsync(ws->ab_arr_host, ws->ab_arr, sizeof(double) * 2 * (size_t)E, cudaMemcpyDeviceToHost, st));
  CU_TRY(cudaMemsetAsync(ws->status_arr, 0, sizeof(LejaStatus) * (size_t)E, st));
  CU_TRY(cudaStreamSynchronize(st));
  if (dense) dense_gershgorin_batch_decode(ws->ab_arr_host, E, ab.data());
  else std::memcpy(ab.data(), ws->ab_arr_host, sizeof(double) * 2 * (size_t)E);

  // S4, cheap part: interval -> (c, gamma, theta); an exponential the sweep kernel does not take (gamma = 0,
  // sub-steps, non-finite bounds) is done on the stepwise path when the plan reaches it
  std::vector<magnus_expmv_info> plan((size_t)E);
  std::vector<double> cc((size_t)E), gg((size_t)E);
  std::vector<char> plannable((size_t)E);
  for (int e = 0; e < E; ++e) {
    double a = ab[2 * e], b = ab[2 * e + 1];
    std::memset(&plan[e], 0, sizeof plan[e]);
    plannable[e] = 0;
    if (!std::isfinite(a) || !std::isfinite(b)) continue;
    snap_interval(&a, &b);
    cc[e] = 0.5 * (a + b);
    gg[e] = 0.25 * (b - a);
    if (!(gg[e] > 0.0) || std::fabs(specs[e].h * gg[e]) > h->prm.theta_max) continue;
    plannable[e] = 1;
    plan[e].a = a;
    plan[e].b = b;
    plan[e].theta = specs[e].h * gg[e];
    plan[e].substeps = 1;
  }

  CsrOp op_all;   // every term the handle has; a job says how many it uses and with which coefficients
  if (!dense) {
    ExpSpec widest = specs[0];
    widest.nterms = h->c_v && h->c_nnz > 0 ? 3 : 2;
    csr_op_from_spec(h, widest, &op_all);
  }
  auto stepwise = [&](int e) {
    OpRef ref;
    if (dense) {   // S2 (+S3, unused: the bounds are known) into the handle's matrix, then the per-iteration kernels
      launch_dense_assemble(h->n, H0v, dense_ld(&h->H0), H1v, dense_ld(&h->H1), specs[e].g, h->M, ws, st);
      ref.dense = true;
      ref.dns.n = h->n;
      ref.dns.ld = h->n;
      ref.dns.M = h->M;
    } else {
      ref.dense = false;
      csr_op_from_spec(h, specs[e], &ref.csr);
    }
    return expmv_on_interval(ref, ab[2 * e], ab[2 * e + 1], psi, psi, specs[e].h, h->prm, ws, st, &plan[e]);
  };
  bool slot_used[kJobRing];
  auto drain_slot = [&](int slot) {   // the launch that used the slot is over: its time, and the slot is free
    if (!slot_used[slot]) return;
    cudaEventSynchronize(ws->ring_ev[2 * slot + 1]);
    if (ws->time_leja) {
      float ms = 0.f;
      if (cudaEventElapsedTime(&ms, ws->ring_ev[2 * slot], ws->ring_ev[2 * slot + 1]) == cudaSuccess) ws->leja_ms += ms;
    }
    slot_used[slot] = false;
  };

  int rc = MAGNUS_OK, seg = 0;   // exponentials before seg are done
  while (seg < E && rc == MAGNUS_OK) {
    int seg_end = seg;
    while (seg_end < E && plannable[seg_end]) ++seg_end;
    // S4 (tables) and S5-S8 of [seg, seg_end): launches of a few jobs each, planned while the device works
    for (int i = 0; i < kJobRing; ++i) slot_used[i] = false;
    int e_next = seg, li = 0;
    while (e_next < seg_end) {
      const int slot = li % kJobRing;
      drain_slot(slot);
      const int nj = std::min(li == 0 ? 4 : kJobsPerLaunch, seg_end - e_next);   // a short first launch starts the device early
      SweepJob* jh = ws->jobs_host + (size_t)slot * kJobsPerLaunch;
      SweepJob* jd = ws->jobs + (size_t)slot * kJobsPerLaunch;
      for (int i = 0; i < nj; ++i) {
        const int e = e_next + i;
        const double hh = specs[e].h, c = cc[e], gamma = gg[e];
        LejaTable T(plan[e].theta, h->prm);
        const int m_try = std::min(h->prm.m_max, std::max(T.have - 1, T.first_chunk()));
        T.need(m_try);
        SweepJob& J = jh[i];
        J.coef[0] = make_double2(1.0, 0.0);
        J.coef[1] = make_double2(specs[e].g, 0.0);
        J.coef[2] = make_double2(0.0, -specs[e].kappa);
        J.phase = make_double2(std::cos(hh * c), -std::sin(hh * c));
        J.inv_gamma = 1.0 / gamma;
        J.c_over_gamma = c / gamma;
        J.m_max = m_try;
        J.nterms = specs[e].nterms;
        J.flags = 0;
        J.pad = 0;
        for (int k = 0; k <= m_try; ++k) J.d[k] = make_double2(T.d[k].real(), T.d[k].imag());
      }
      CU_TRY(cudaMemcpyAsync(jd, jh, sizeof(SweepJob) * (size_t)nj, cudaMemcpyHostToDevice, st));
      CU_TRY(cudaEventRecord(ws->ring_ev[2 * slot], st));
      const LejaStatus* gate = e_next > seg ? ws->status_arr + e_next - 1 : nullptr;
      const int lrc = dense ? launch_dense_leja_sweep_jobs(h->n, H0v, dense_ld(&h->H0), H1v, dense_ld(&h->H1), h->M, psi, jd,
                                                           nj, h->prm.tol, ws->status_arr + e_next, gate, ws, st)
                      : !csr_mid_sweep_supported(h->n, ws->csr_kernel)
                          ? launch_csr_leja_sweep_small_jobs(op_all, psi, jd, nj, ws->leja_l, h->prm.tol,
                                                             ws->status_arr + e_next, gate, ws, st)
                          : launch_csr_leja_sweep_mid_jobs(op_all, psi, jd, nj, h->prm.tol, ws->status_arr + e_next, gate,
                                                           ws, st);
      if (lrc != MAGNUS_OK) {
        set_error("whole-sweep launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        return MAGNUS_ECUDA;
      }
      CU_TRY(cudaEventRecord(ws->ring_ev[2 * slot + 1], st));
      slot_used[slot] = true;
      e_next += nj;
      ++li;
    }
    int e = seg;
    if (seg_end > seg) {
      CU_TRY(cudaMemcpyAsync(ws->status_arr_host + seg, ws->status_arr + seg, sizeof(LejaStatus) * (size_t)(seg_end - seg),
                             cudaMemcpyDeviceToHost, st));
      CU_TRY(cudaStreamSynchronize(st));
      for (int i = 0; i < kJobRing; ++i) drain_slot(i);
      for (; e < seg_end && ws->status_arr_host[e].done; ++e) {
        plan[e].iters = ws->status_arr_host[e].iters;
        plan[e].err_est = ws->status_arr_host[e].err_est;
      }
      if (e < seg_end)   // the launches behind a failed job did nothing: forget their records
        CU_TRY(cudaMemsetAsync(ws->status_arr + e, 0, sizeof(LejaStatus) * (size_t)(seg_end - e), st));
    }
    // e == seg_end: the segment is through and exponential seg_end (if any) is not for the sweep kernel;
    // e <  seg_end: job e did not converge within its table and psi is the state before it.  Stepwise either way.
    if (e < E) {
      rc = stepwise(e);
      ++e;
    }
    seg = e;
  }
  if (infos)
    for (int s = 0; s < ns; ++s) {
      std::memset(&infos[s], 0, sizeof infos[s]);
      infos[s].n_exp = first_of_step[s + 1] - first_of_step[s];
      for (int e = first_of_step[s]; e < first_of_step[s + 1]; ++e) infos[s].exp[e - first_of_step[s]] = plan[e];
    }
  return rc;
}

// Shortcut MAGNUS_SHORTCUT_TIGHT_INTERVAL: raw interval of op from Lanczos started at v (kernels_lanczos.cu).
// Returns kPlanDeclined when v = 0 (the caller keeps the Gershgorin interval).
static int lanczos_interval(magnus_context* h, const OpRef& op, const cplx* v, double* a, double* b) {
  Workspace* ws = &h->ws;
  cudaStream_t st = h->stream;
  const int64_t n = h->n;
  const int m = h->lanczos_steps;
  if (!h->lz[0]) {
    if (cudaMalloc(&h->lz[0], sizeof(cplx) * (size_t)n) != cudaSuccess || cudaMalloc(&h->lz[1], sizeof(cplx) * (size_t)n) != cudaSuccess ||
        cudaMalloc(&h->lz_scal, sizeof(double) * (2 + 2 * 64)) != cudaSuccess) {
      cudaGetLastError();
      set_error("tight interval: allocation of the Lanczos vectors failed");
      return MAGNUS_ENOMEM;
    }
  }
  CU_TRY(cudaMemsetAsync(ws->status, 0, sizeof(LejaStatus), st));
  CU_TRY(cudaMemsetAsync(ws->p, 0, sizeof(cplx) * (size_t)n, st));   // the mat-vec kernel's Newton sum: d_k = 0 keeps it 0
  CU_TRY(cudaMemsetAsync(h->lz_scal, 0, sizeof(double) * (2 + 2 * 64), st));
  cplx* q = h->lz[0];
  cplx* qp = h->lz[1];
  launch_lanczos_start(v, q, qp, n, h->lz_scal, ws, st);
  for (int j = 0; j < m; ++j) {
    // u = M q_j: the fused Leja iteration as a plain mat-vec (1/gamma = 1, shift = 0, d_k = 0; |d_k| = 1, tol = 0: no stop)
    launch_iter(op, q, ws->w[0], ws->p, 1.0, 0.0, make_double2(0.0, 0.0), 1.0, 0.0, ws, st);
    launch_lanczos_step(ws->w[0], q, qp, n, h->lz_scal, j, m, ws, st);
    std::swap(q, qp);
  }
  h->lanczos_matvecs += m;
  double sc[2 + 2 * 64];
  CU_TRY(cudaGetLastError());
  CU_TRY(cudaMemcpyAsync(sc, h->lz_scal, sizeof(double) * (size_t)(2 + 2 * m), cudaMemcpyDeviceToHost, st));
  CU_TRY(cudaStreamSynchronize(st));
  if (!(sc[0] > 0.0)) return kPlanDeclined;
  const double* alpha = sc + 2;
  const double* beta = sc + 2 + m;
  int k = m;
  double scale = 0.0;
  for (int j = 0; j < m; ++j) {
    if (!std::isfinite(alpha[j]) || !std::isfinite(beta[j])) { set_error("tight interval: Lanczos produced a non-finite value"); return MAGNUS_EINVAL; }
    scale = std::max(scale, std::max(std::fabs(alpha[j]), beta[j]));
    if (beta[j] <= 1e-12 * scale) { k = j + 1; break; }      // invariant subspace: T is exact, later steps are noise
  }
  double lo = 0.0, hi = 0.0;
  tridiag_extreme_eigenvalues(alpha, beta, k, &lo, &hi);
  *a = lo - beta[k - 1];
  *b = hi + beta[k - 1];
  return MAGNUS_OK;
}

// One step on the stepwise path: interval, table and stop polling per exponential (rows S1-S8, D3, D4).
static int magnus_step_unplanned(magnus_context* h, double t, double tau, cplx* psi, magnus_step_info* info) {
  double coef[MAGNUS_MAX_EXP_PER_STEP], hscale[MAGNUS_MAX_EXP_PER_STEP], kappa = 0.0;
  const int n_exp = step_coefficients(h->scheme, h->f, h->user, t, tau, coef, hscale, &kappa);   // S1
  if (info) {
    std::memset(info, 0, sizeof *info);
    info->n_exp = n_exp;
  }
  cudaStream_t st = h->stream;
  Workspace* ws = &h->ws;
  int rc = MAGNUS_OK;
  ExpSpec specs[MAGNUS_MAX_EXP_PER_STEP];      // the same scalars in the form the CSR operator takes them
  specs_from_coefficients(h, n_exp, coef, hscale, kappa, tau, specs);
  for (int e = 0; e < n_exp && rc == MAGNUS_OK; ++e) {
    OpRef op;
    double a = 0.0, b = 0.0;
    if (h->is_xxz) {   // S2, S3 without a matrix: entries from the row bits, bounds from their closed form
      op.dense = false;
      op.xxz = true;
      op.xx.nspins = h->xxz_model.nspins;
      op.xx.jz = h->xxz_model.jz;
      op.xx.apair = 2.0 * h->xxz_model.jxy;
      op.xx.asingle = coef[e] * h->xxz_model.hx;
      xxz_gershgorin(op.xx, &a, &b);
    } else if (h->format == MAGNUS_CSR) {
      op.dense = false;
      csr_op_from_spec(h, specs[e], &op.csr);     // S2: the terms with this exponential's coefficients (M4: c1, g12)
      if ((op.csr.nterms == 2 && h->gs_disjoint2) || (op.csr.nterms == 3 && h->gs_disjoint3)) {     // S3
        const int nblk = launch_csr_gershgorin_cached(op.csr, h->gs_r, h->gs_diag, ws, st);
        rc = read_interval(nblk, ws, st, &a, &b);
      } else {
        rc = op_interval(op, ws, st, &a, &b);
      }
    } else {
      op.dense = true;
      const cplx* H0v = (const cplx*)h->H0.values;
      const cplx* H1v = (const cplx*)h->H1.values;
      int nblk = 0;
      if (h->scheme == MAGNUS_M6) {
        // P:103-114 with A = -iH (reading m6); X1 = h->M, X2 = h->A2, X3 = h->P, X4, X5; see magnus.h at magnus_step
        const int64_t n = h->n;
        const double f1 = coef[0], f2 = coef[1], f3 = coef[2];
        const double b2 = (std::sqrt(15.0) / 3.0) * tau * (f3 - f1), b3 = (10.0 / 3.0) * tau * (f3 - 2.0 * f2 + f1);
        LinComb lc;
        auto term = [&](int k, const cplx* x, double re, double im) {
          lc.x[k] = x;
          lc.c[k] = make_double2(re, im);
        };
        term(0, H0v, 1.0, 0.0); term(1, H1v, f2, 0.0); term(2, nullptr, 0.0, 0.0); term(3, nullptr, 0.0, 0.0);
        if (dense_ld(&h->H0) != n || dense_ld(&h->H1) != n) { set_error("MAGNUS_M6 needs ld == n"); rc = MAGNUS_EINVAL; break; }
        if (tau == 0.0) {   // Omega_H carries b3 / (12 tau) and 1 / (240 tau); a zero step is the identity anyway
          set_error("MAGNUS_M6: tau must be non-zero");
          rc = MAGNUS_EINVAL;
          break;
        }
        auto gemm_failed = [&](const char* which) {
          set_error("MAGNUS_M6: zgemm launch of %s failed: %s", which, cudaGetErrorString(cudaGetLastError()));
        };
        launch_dense_lincomb(n, h->M, lc, ws, st);                                   // X1 = H2 = H0 + f2 H1
        if (h->time_comm) cudaEventRecord(h->ev_comm[0], st);
        rc = launch_zgemm(n, h->M, n, H1v, n, h->A2, n, st, &h->zs);                          // X2 = P1 = H2 H1
        if (rc) { gemm_failed("P1 = H2 H1"); break; }
        launch_dense_antiherm(n, h->A2, h->P, -1.0, st);                              // X3 = G = P1 - P1^H = [H2, H1]
        rc = launch_zgemm(n, h->M, n, h->P, n, h->A2, n, st, &h->zs);                         // X2 = P2 = H2 G
        if (rc) { gemm_failed("P2 = H2 G"); break; }
        launch_dense_antiherm(n, h->A2, h->X4, 1.0, st);                              // X4 = S = P2 + P2^H = [H2, G]
        term(0, h->M, 0.0, 20.0 * tau); term(1, H1v, 0.0, b3); term(2, h->P, -tau * b2, 0.0); term(3, nullptr, 0.0, 0.0);
        launch_dense_lincomb(n, h->A2, lc, ws, st);                                  // X2 = L
        term(0, H1v, 0.0, -b2); term(1, h->P, tau * b3 / 30.0, 0.0); term(2, h->X4, 0.0, -tau * tau * b2 / 60.0);
        term(3, nullptr, 0.0, 0.0);
        launch_dense_lincomb(n, h->X5, lc, ws, st);                                  // X5 = R
        rc = launch_zgemm(n, h->A2, n, h->X5, n, h->X4, n, st, &h->zs);                       // X4 = P3 = L R
        ws->launches += 5;      // 3 GEMMs + 2 antiherm (the 3 lincomb launches count themselves, the omega launch below too)
        if (h->time_comm) cudaEventRecord(h->ev_comm[1], st);
        if (rc) { gemm_failed("P3 = L R"); break; }
        // Omega_H = H2 + (b3/(12 tau)) H1 + (i/(240 tau)) (P3 - P3^H), over X1, with its Gershgorin bounds
        nblk = launch_dense_omega(n, h->M, H1v, h->X4, 1.0, b3 / (12.0 * tau), -1.0 / (240.0 * tau), ws, st);
      } else if (h->scheme == MAGNUS_M4 && h->cached_p0) {
        // shortcut: Omega_H = H0 + fbar H1 - i kappa (P0 - P0^H), kappa = (sqrt(3) tau/12)(f1 - f2), no GEMM
        LinComb lc;
        lc.x[0] = H0v; lc.c[0] = make_double2(1.0, 0.0);
        lc.x[1] = H1v; lc.c[1] = make_double2(0.5 * (coef[0] + coef[1]), 0.0);
        lc.x[2] = lc.x[3] = nullptr; lc.c[2] = lc.c[3] = make_double2(0.0, 0.0);
        launch_dense_lincomb(h->n, h->M, lc, ws, st);
        nblk = launch_dense_omega(h->n, h->M, H1v, h->P, 1.0, 0.0, kappa, ws, st);
      } else if (h->scheme == MAGNUS_M4) {
        launch_dense_assemble2(h->n, H0v, dense_ld(&h->H0), H1v, dense_ld(&h->H1), coef[0], coef[1], h->M, h->A2, ws,
                               st);                                                                // S2: A1, A2
        if (h->time_comm) cudaEventRecord(h->ev_comm[0], st);
        rc = launch_zgemm(h->n, h->A2, h->n, h->M, h->n, h->P, h->n, st, &h->zs);                          // D3: P = A2 A1
        ws->launches += 1;
        if (h->time_comm) cudaEventRecord(h->ev_comm[1], st);
        if (rc) { set_error("zgemm launch failed: %s", cudaGetErrorString(cudaGetLastError())); break; }
        nblk = launch_dense_omega(h->n, h->M, h->A2, h->P, 0.5, 0.5, std::sqrt(3.0) * tau / 12.0, ws, st);   // D4 (+S3)
      } else {
        nblk = launch_dense_assemble(h->n, H0v, dense_ld(&h->H0), H1v, dense_ld(&h->H1), coef[e], h->M, ws, st);
      }
      op.dns.n = h->n;
      op.dns.ld = h->n;
      op.dns.M = h->M;
      rc = read_interval(nblk, ws, st, &a, &b);
      if (rc == MAGNUS_OK && h->time_comm) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, h->ev_comm[0], h->ev_comm[1]) == cudaSuccess) h->comm_ms += ms;
      }
    }
    if (rc) break;
    if (h->shortcuts & MAGNUS_SHORTCUT_TIGHT_INTERVAL) {
      double ta = 0.0, tb = 0.0;
      rc = lanczos_interval(h, op, psi, &ta, &tb);
      if (rc == MAGNUS_OK) {
        // the Lanczos interval is an estimate, not an enclosure: never let it reach beyond the Gershgorin
        // enclosure [a, b] on either side (reading ti); disjoint (cannot happen in exact arithmetic): keep [a, b]
        const double ia = std::max(a, ta), ib = std::min(b, tb);
        if (ia <= ib) {
          a = ia;
          b = ib;
        }
      } else if (rc == kPlanDeclined) {
        rc = MAGNUS_OK;       // psi = 0: nothing to estimate from, the Gershgorin interval stays
      } else {
        break;
      }
    }
    rc = expmv_on_interval(op, a, b, psi, psi, hscale[e] * tau, h->prm, ws, st, info ? &info->exp[e] : nullptr);
  }
  return rc;
}


extern "C" {

const char* magnus_strerror(int code) {
  switch (code) {
    case MAGNUS_OK: return "ok";
    case MAGNUS_EINVAL: return "invalid argument";
    case MAGNUS_ENOMEM: return "out of memory";
    case MAGNUS_ECUDA: return "CUDA error";
    case MAGNUS_ENOCONV: return "Leja interpolation did not converge within m_max";
    case MAGNUS_ENOTHERMITIAN: return "matrix is not Hermitian";
    default: return "unknown error";
  }
}

const char* magnus_last_error(void) { return g_err; }

const char* magnus_version(void) { return "magnus-b200 0.1 (sm_100a)"; }

int magnus_host_leja_points(int m, double* out_host) {
  if (!out_host || m < 0 || m > kMaxDegree + 1) { set_error("magnus_host_leja_points: bad m"); return MAGNUS_EINVAL; }
  std::memcpy(out_host, leja_points(), sizeof(double) * (size_t)m);
  return MAGNUS_OK;
}

int magnus_host_divided_differences(double theta, int m, double* out_host) {
  if (!out_host || m < 1 || m > kMaxDegree + 1) { set_error("magnus_host_divided_differences: bad m"); return MAGNUS_EINVAL; }
  divided_differences(theta, m, reinterpret_cast<std::complex<double>*>(out_host));
  return MAGNUS_OK;
}

int magnus_host_snap_interval(double* a, double* b) {
  if (!a || !b) return MAGNUS_EINVAL;
  snap_interval(a, b);
  return MAGNUS_OK;
}

int magnus_host_tridiag_extremes(const double* alpha_host, const double* beta_host, int k, double* lo, double* hi) {
  if (!alpha_host || (k > 1 && !beta_host) || k < 1 || !lo || !hi) { set_error("magnus_host_tridiag_extremes: bad arguments"); return MAGNUS_EINVAL; }
  tridiag_extreme_eigenvalues(alpha_host, beta_host, k, lo, hi);
  return MAGNUS_OK;
}

int magnus_host_step_coefficients(int scheme, magnus_drive_fn f, void* user, double t, double tau, double* coef_h1,
                                  double* h_scale, double* kappa_out) {
  if (!f || !coef_h1 || !h_scale) return MAGNUS_EINVAL;
  const int n = step_coefficients(scheme, f, user, t, tau, coef_h1, h_scale, kappa_out);
  if (n < 0) { set_error("unknown scheme %d", scheme); return MAGNUS_EINVAL; }
  return n;
}

int magnus_destroy(magnus_handle h) {
  if (!h) return MAGNUS_OK;
  workspace_free(&h->ws);
  slice_layout_free(&h->slice);
  cudaFree(h->M);
  cudaFree(h->A2);
  cudaFree(h->P);
  cudaFree(h->X4);
  cudaFree(h->X5);
  cudaFree(h->d0);
  cudaFree(h->d1);
  zgemm_scratch_free(&h->zs);
  cudaFree(h->lz[0]);
  cudaFree(h->lz[1]);
  cudaFree(h->lz_scal);
  cudaFree(h->c_rp);
  cudaFree(h->c_ci);
  cudaFree(h->c_v);
  for (int t = 0; t < 3; ++t) {
    cudaFree(h->gs_r[t]);
    cudaFree(h->gs_diag[t]);
  }
  for (int i = 0; i < 2; ++i)
    if (h->ev_comm[i]) cudaEventDestroy(h->ev_comm[i]);
  delete h;
  return MAGNUS_OK;
}

int magnus_describe(magnus_handle h, magnus_path_info* out) {
  if (!h || !out) { set_error("magnus_describe: NULL argument"); return MAGNUS_EINVAL; }
  std::memset(out, 0, sizeof *out);
  const int64_t n = h->n;
  const char* name = "dense_leja_iter_kernel";
  if (h->is_xxz) {
    name = "xxz_leja_iter_kernel";
    out->bytes_per_iteration = 64 * n;          // w gather (16 n ideal), w+ write, p read + write: no matrix bytes
    const int64_t N = h->xxz_model.nspins;
    out->csr_bytes_per_iteration = 20 * (n * (3 * N + 2) / 2) + 4 * (n + 1) * 2 + 64 * n;
  } else if (h->format == MAGNUS_DENSE) {
    out->bytes_per_iteration = 16 * n * n + 64 * n;
    if (dense_sweep_supported(n) && h->ws.csr_kernel == 0) name = "dense_leja_sweep_kernel";
  } else {
    int64_t nnz = h->H0.nnz + h->H1.nnz, terms = 2;
    if (h->scheme == MAGNUS_M4 && h->c_nnz > 0) {
      nnz += h->c_nnz;
      terms = 3;
    }
    out->csr_bytes_per_iteration = 20 * nnz + 4 * (n + 1) * terms + 64 * n;
    out->bytes_per_iteration = out->csr_bytes_per_iteration;
    const int k = h->ws.csr_kernel;
    if (csr_mid_sweep_supported(n, k)) {
      name = "csr_leja_sweep_mid_kernel";
    } else if (n <= kSmallSweepMaxN && k == 0) {
      name = "csr_leja_sweep_small_kernel";
    } else if (h->slice.meta && (k == 0 || slice_layout_kind(k) != 0)) {
      out->slices = h->slice.nslices;
      out->slots = h->slice.nslots;
      out->entries = h->slice.nent;
      if (h->slice.offsets) {
        name = "csr_leja_iter_sliceoff_kernel";
        out->bytes_per_iteration = (h->slice.real_values ? 8 : 16) * h->slice.nent + 8 * h->slice.nslots +
                                   24 * h->slice.nslices + 64 * n;
        if (h->slice.real_values) name = "csr_leja_iter_sliceoff_kernel (real values)";
      } else {
        name = "csr_leja_iter_slice_kernel";
        out->bytes_per_iteration = 20 * h->slice.nent + 4 * h->slice.nslots + 24 * h->slice.nslices + 64 * n;
      }
    } else if (k == 3 || (k >= 20000 && k < 30000)) {
      name = "csr_leja_iter_stream_kernel";
    } else if (k == 4) {
      name = "csr_leja_iter_rowtma_kernel";
    } else if (k == 2 || k >= 1000 || (k == 0 && n >= 32768)) {
      name = "csr_leja_iter_rowblock_kernel";
    } else {
      name = "csr_leja_iter_generic";
    }
  }
  std::snprintf(out->leja_kernel, sizeof out->leja_kernel, "%s", name);
  return MAGNUS_OK;
}

int magnus_create(magnus_handle* out, const magnus_matrix* H0, const magnus_matrix* H1, magnus_drive_fn f, void* user,
                  int scheme, const magnus_options* opt) {
  if (!out) { set_error("out is NULL"); return MAGNUS_EINVAL; }
  *out = nullptr;
  int rc = check_matrix(H0, "H0");
  if (rc) return rc;
  rc = check_matrix(H1, "H1");
  if (rc) return rc;
  if (H0->format != H1->format || H0->n != H1->n) { set_error("H0 and H1 differ in format or n"); return MAGNUS_EINVAL; }
  if (!f) { set_error("f is NULL"); return MAGNUS_EINVAL; }
  if (scheme < MAGNUS_CF4 || scheme > MAGNUS_M6) { set_error("unknown scheme %d", scheme); return MAGNUS_EINVAL; }
  rc = require_device();
  if (rc) return rc;

  magnus_context* h = new (std::nothrow) magnus_context();
  if (!h) return MAGNUS_ENOMEM;
  h->scheme = scheme;
  h->format = H0->format;
  h->n = H0->n;
  h->H0 = *H0;
  h->H1 = *H1;
  h->f = f;
  h->user = user;
  default_params(opt, &h->prm, &h->stream, &h->ws.csr_kernel, &h->shortcuts);
  h->lanczos_steps = (opt && opt->lanczos_steps > 0) ? std::min(64, opt->lanczos_steps) : 8;
  const int csr_kernel = h->ws.csr_kernel;
  rc = workspace_alloc(&h->ws, h->n, h->stream);
  h->ws.csr_kernel = csr_kernel;
  h->ws.time_leja = true;
  if (rc) { set_error("workspace allocation failed (n=%lld)", (long long)h->n); magnus_destroy(h); return rc; }

  if (opt && opt->check_hermitian) {
    double bad0 = 0.0, bad1 = 0.0;
    if (h->format == MAGNUS_CSR) {
      rc = csr_hermitian_check(H0, h->stream, &bad0);
      if (!rc) rc = csr_hermitian_check(H1, h->stream, &bad1);
    } else {
      DenseOp d0{H0->n, dense_ld(H0), (const cplx*)H0->values}, d1{H1->n, dense_ld(H1), (const cplx*)H1->values};
      rc = dense_hermitian_check(d0, h->stream, &bad0);
      if (!rc) rc = dense_hermitian_check(d1, h->stream, &bad1);
    }
    if (rc) { magnus_destroy(h); return rc; }
    if (bad0 > 1e-12 || bad1 > 1e-12) {
      set_error("sampled Hermitian check failed: max |M_ij - conj(M_ji)| = %g (H0), %g (H1)", bad0, bad1);
      magnus_destroy(h);
      return MAGNUS_ENOTHERMITIAN;
    }
  }

  if (scheme == MAGNUS_M6 && h->format == MAGNUS_CSR) {
    // the nested commutators of M6 fill in: CSR input of the sizes the paper runs (n <= 2^14) is
    // expanded into dense copies and takes the dense path; larger CSR input is refused
    if (h->n > kM6DenseMaxN) {
      set_error("MAGNUS_M6 on CSR input needs n <= %d (the nested commutators fill in; got n=%lld)", kM6DenseMaxN,
                (long long)h->n);
      magnus_destroy(h);
      return MAGNUS_EINVAL;
    }
    const size_t bytes = sizeof(cplx) * (size_t)h->n * (size_t)h->n;
    if (cudaMalloc(&h->d0, bytes) != cudaSuccess || cudaMalloc(&h->d1, bytes) != cudaSuccess) {
      cudaGetLastError();
      set_error("dense copies for M6 on CSR input: allocation failed (%zu bytes each)", bytes);
      magnus_destroy(h);
      return MAGNUS_ENOMEM;
    }
    launch_csr_to_dense(h->n, H0->row_ptr, H0->col_idx, (const cplx*)H0->values, h->d0, h->stream);
    launch_csr_to_dense(h->n, H1->row_ptr, H1->col_idx, (const cplx*)H1->values, h->d1, h->stream);
    std::memset(&h->H0, 0, sizeof h->H0);
    std::memset(&h->H1, 0, sizeof h->H1);
    h->H0.format = h->H1.format = MAGNUS_DENSE;
    h->H0.n = h->H1.n = h->n;
    h->H0.ld = h->H1.ld = h->n;
    h->H0.values = h->d0;
    h->H1.values = h->d1;
    h->format = MAGNUS_DENSE;
  }
  if (h->format == MAGNUS_DENSE) {
    const size_t bytes = sizeof(cplx) * (size_t)h->n * (size_t)h->n;
    bool ok = cudaMalloc(&h->M, bytes) == cudaSuccess;
    if (ok && (scheme == MAGNUS_M4 || scheme == MAGNUS_M6))
      ok = cudaMalloc(&h->A2, bytes) == cudaSuccess && cudaMalloc(&h->P, bytes) == cudaSuccess;
    if (ok && scheme == MAGNUS_M6)
      ok = cudaMalloc(&h->X4, bytes) == cudaSuccess && cudaMalloc(&h->X5, bytes) == cudaSuccess;
    if (!ok) {
      cudaGetLastError();
      set_error("dense workspace allocation failed (%zu bytes per matrix)", bytes);
      magnus_destroy(h);
      return MAGNUS_ENOMEM;
    }
    if (scheme == MAGNUS_M4 || scheme == MAGNUS_M6) {
      zgemm_scratch_alloc(&h->zs);     // on failure the plain one-CTA-per-tile form runs
      cudaEventCreate(&h->ev_comm[0]);
      cudaEventCreate(&h->ev_comm[1]);
      h->time_comm = true;
    }
    if (scheme == MAGNUS_M6 && (dense_ld(&h->H0) != h->n || dense_ld(&h->H1) != h->n)) {
      set_error("MAGNUS_M6 needs dense H0, H1 with ld == n (the products read them as n x n blocks)");
      magnus_destroy(h);
      return MAGNUS_EINVAL;
    }
    if (scheme == MAGNUS_M4 && (h->shortcuts & MAGNUS_SHORTCUT_CACHED_COMMUTATOR)) {
      if (dense_ld(H0) != h->n || dense_ld(H1) != h->n) {
        set_error("MAGNUS_SHORTCUT_CACHED_COMMUTATOR needs ld == n");
        magnus_destroy(h);
        return MAGNUS_EINVAL;
      }
      rc = launch_zgemm(h->n, (const cplx*)H0->values, h->n, (const cplx*)H1->values, h->n, h->P, h->n, h->stream, &h->zs);
      if (rc) { set_error("zgemm launch failed: %s", cudaGetErrorString(cudaGetLastError())); magnus_destroy(h); return rc; }
      h->cached_p0 = true;
      h->time_comm = false;
    }
  } else if (scheme == MAGNUS_M4) {
    int64_t nnz = 0;
    rc = csr_commutator_owned(H0, H1, &h->c_rp, &h->c_ci, &h->c_v, &nnz, h->stream);   // S0
    if (rc) { magnus_destroy(h); return rc; }
    h->c_nnz = nnz;
  }
  if (h->format == MAGNUS_CSR) {
    rc = csr_cache_rowstats(h);
    if (rc) { magnus_destroy(h); return rc; }
    // slice-major copy of the operator: asked for explicitly, or by default for large n when its slots are
    // well filled (spin chains: about 20 entries per slot); otherwise the CSR kernels run
    const int kind = slice_layout_kind(csr_kernel);
    if (kind != 0 || (csr_kernel == 0 && h->n >= kSliceAutoMinN && !csr_mid_sweep_supported(h->n, csr_kernel))) {
      CsrOp op;
      op.n = h->n;
      op.unit_cap = 0;
      op.nterms = (scheme == MAGNUS_M4 && h->c_nnz > 0) ? 3 : 2;
      op.t[0] = csr_term(&h->H0, 1.0, 0.0);
      op.t[1] = csr_term(&h->H1, 1.0, 0.0);
      op.t[2] = op.t[1];
      if (op.nterms == 3) {
        op.t[2].rp = h->c_rp;
        op.t[2].ci = h->c_ci;
        op.t[2].v = h->c_v;
        op.t[2].nnz = h->c_nnz;
      }
      const bool allow_real = (h->shortcuts & MAGNUS_SHORTCUT_REAL_VALUES) != 0 || (csr_kernel >= 6500 && csr_kernel < 7000);
      if (slice_layout_build(op, &h->slice, h->stream, kind != 1, allow_real) == MAGNUS_OK && kind == 0 &&
          (double)h->slice.nent < kSliceAutoMinFill * (double)h->slice.nslots)
        slice_layout_free(&h->slice);                  // poorly filled slots: not worth it
      // on failure the CSR kernels run
    }
  }
  if (cudaStreamSynchronize(h->stream) != cudaSuccess) { magnus_destroy(h); return MAGNUS_ECUDA; }
  *out = h;
  return MAGNUS_OK;
}

int magnus_create_xxz(magnus_handle* out, const magnus_xxz_model* model, magnus_drive_fn f, void* user, int scheme,
                      const magnus_options* opt) {
  if (!out) { set_error("out is NULL"); return MAGNUS_EINVAL; }
  *out = nullptr;
  if (!model || !f) { set_error("magnus_create_xxz: NULL model or f"); return MAGNUS_EINVAL; }
  if (model->nspins < 3 || model->nspins > 30) { set_error("magnus_create_xxz: nspins must be in [3, 30]"); return MAGNUS_EINVAL; }
  if (scheme != MAGNUS_CF4 && scheme != MAGNUS_M2 && scheme != MAGNUS_CF4_3) {
    set_error("magnus_create_xxz: commutator-free schemes only (got %d)", scheme);
    return MAGNUS_EINVAL;
  }
  int rc = require_device();
  if (rc) return rc;
  magnus_context* h = new (std::nothrow) magnus_context();
  if (!h) return MAGNUS_ENOMEM;
  h->scheme = scheme;
  h->format = MAGNUS_CSR;
  h->is_xxz = true;
  h->xxz_model = *model;
  h->n = (int64_t)1 << model->nspins;
  std::memset(&h->H0, 0, sizeof h->H0);
  std::memset(&h->H1, 0, sizeof h->H1);
  h->f = f;
  h->user = user;
  default_params(opt, &h->prm, &h->stream, &h->ws.csr_kernel, &h->shortcuts);
  h->lanczos_steps = (opt && opt->lanczos_steps > 0) ? std::min(64, opt->lanczos_steps) : 8;
  rc = workspace_alloc(&h->ws, h->n, h->stream);
  h->ws.csr_kernel = 1;       // no whole-sweep kernels on this path
  h->ws.time_leja = true;
  if (rc) { set_error("workspace allocation failed (n=%lld)", (long long)h->n); magnus_destroy(h); return rc; }
  *out = h;
  return MAGNUS_OK;
}

int magnus_step(magnus_handle h, double t, double tau, void* psi_, magnus_step_info* info) {
  if (!h || !psi_) { set_error("magnus_step: NULL handle or psi"); return MAGNUS_EINVAL; }
  cplx* psi = (cplx*)psi_;
  if (plan_supported(h)) {   // a batch of one step: two host syncs instead of two per exponential
    const int rc = run_planned(h, t, tau, 0, 1, psi, info);
    if (rc != kPlanDeclined) return rc;
  }
  return magnus_step_unplanned(h, t, tau, psi, info);
}

int magnus_integrate(magnus_handle h, double t0, double t_end, int64_t nsteps, void* psi, magnus_stats* stats) {
  if (!h || !psi || nsteps <= 0) { set_error("magnus_integrate: bad arguments"); return MAGNUS_EINVAL; }
  const double tau = (t_end - t0) / (double)nsteps;
  cudaStream_t st = h->stream;
  Workspace* ws = &h->ws;
  const int64_t launches0 = ws->launches;
  ws->leja_ms = 0.0;
  h->comm_ms = 0.0;
  h->lanczos_matvecs = 0;
  CU_TRY(cudaEventRecord(ws->ev[2], st));
  int64_t total = 0, nexp = 0;
  int rc = MAGNUS_OK;
  auto account = [&](const magnus_step_info& si, int rc_step) {
    for (int e = 0; e < si.n_exp; ++e) {
      if (rc_step != MAGNUS_OK && si.exp[e].iters == 0 && si.exp[e].substeps == 0) break;
      if (stats && stats->iters && nexp < stats->iters_cap) stats->iters[nexp] = si.exp[e].iters;
      total += si.exp[e].iters;
      ++nexp;
    }
  };
  const int batch_steps = kPlanCap / MAGNUS_MAX_EXP_PER_STEP;
  std::vector<magnus_step_info> infos;
  for (int64_t s = 0; s < nsteps && rc == MAGNUS_OK;) {
    if (plan_supported(h)) {
      const int ns = (int)std::min<int64_t>(batch_steps, nsteps - s);
      infos.resize((size_t)ns);
      std::memset(infos.data(), 0, sizeof(magnus_step_info) * (size_t)ns);
      const int prc = run_planned(h, t0, tau, s, ns, (cplx*)psi, infos.data());
      if (prc != kPlanDeclined) {
        rc = prc;
        for (int i = 0; i < ns; ++i) account(infos[(size_t)i], rc);
        s += ns;
        continue;
      }
    }
    magnus_step_info si;
    rc = magnus_step_unplanned(h, t0 + (double)s * tau, tau, (cplx*)psi, &si);
    account(si, rc);
    ++s;
  }
  CU_TRY(cudaEventRecord(ws->ev[3], st));
  CU_TRY(cudaStreamSynchronize(st));
  if (stats) {
    float ms = 0.f;
    cudaEventElapsedTime(&ms, ws->ev[2], ws->ev[3]);
    stats->total_matvecs = total;
    stats->n_exp = nexp;
    stats->seconds_device = ms * 1e-3;
    stats->seconds_leja = ws->leja_ms * 1e-3;
    stats->seconds_commutator = h->comm_ms * 1e-3;
    stats->kernel_launches = ws->launches - launches0;
    stats->lanczos_matvecs = h->lanczos_matvecs;
  }
  return rc;
}

int leja_expmv(const magnus_matrix* H, const void* v_in, void* v_out, double h, double tol, void* stream,
               magnus_expmv_info* info) {
  int rc = check_matrix(H, "H");
  if (rc) return rc;
  if (!v_in || !v_out) { set_error("leja_expmv: NULL vector"); return MAGNUS_EINVAL; }
  rc = require_device();
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  LejaParams prm;
  prm.tol = tol > 0.0 ? tol : 1e-12;
  prm.theta_max = 16.0;
  prm.m_max = kMaxDegree;
  Workspace ws;
  rc = workspace_alloc(&ws, H->n, st);
  if (rc) { cudaGetLastError(); workspace_free(&ws); set_error("leja_expmv: workspace allocation failed"); return rc; }
  OpRef op;
  if (H->format == MAGNUS_CSR) {
    op.dense = false;
    op.csr.n = H->n;
    op.csr.nterms = 1;
    op.csr.t[0] = csr_term(H, 1.0, 0.0);
    op.csr.t[1] = op.csr.t[2] = op.csr.t[0];
    op.csr.unit_cap = 0;
    if (csr_unit_cap(op.csr, st, &op.csr.unit_cap) != MAGNUS_OK) op.csr.unit_cap = 0;
  } else {
    op.dense = true;
    op.dns.n = H->n;
    op.dns.ld = dense_ld(H);
    op.dns.M = (const cplx*)H->values;
  }
  double a = 0.0, b = 0.0;
  rc = op_interval(op, &ws, st, &a, &b);
  if (rc == MAGNUS_OK) rc = expmv_on_interval(op, a, b, (const cplx*)v_in, (cplx*)v_out, h, prm, &ws, st, info);
  if (cudaStreamSynchronize(st) != cudaSuccess && rc == MAGNUS_OK) rc = MAGNUS_ECUDA;
  workspace_free(&ws);
  return rc;
}

// ---- host-buffer end-to-end call -------------------------------------------------
static int upload_matrix(const magnus_matrix* Hh, magnus_matrix* Hd, cudaStream_t st) {
  *Hd = *Hh;
  Hd->values = nullptr;
  Hd->col_idx = nullptr;
  Hd->row_ptr = nullptr;
  void* p = nullptr;
  if (Hh->format == MAGNUS_CSR) {
    const size_t nnz = (size_t)(Hh->nnz > 0 ? Hh->nnz : 1);
    if (cudaMalloc(&p, sizeof(cplx) * nnz) != cudaSuccess) return MAGNUS_ENOMEM;
    Hd->values = p;
    if (cudaMalloc(&p, sizeof(int32_t) * nnz) != cudaSuccess) return MAGNUS_ENOMEM;
    Hd->col_idx = (const int32_t*)p;
    if (cudaMalloc(&p, sizeof(int32_t) * (size_t)(Hh->n + 1)) != cudaSuccess) return MAGNUS_ENOMEM;
    Hd->row_ptr = (const int32_t*)p;
    CU_TRY(cudaMemcpyAsync((void*)Hd->values, Hh->values, sizeof(cplx) * (size_t)Hh->nnz, cudaMemcpyHostToDevice, st));
    CU_TRY(cudaMemcpyAsync((void*)Hd->col_idx, Hh->col_idx, sizeof(int32_t) * (size_t)Hh->nnz, cudaMemcpyHostToDevice, st));
    CU_TRY(cudaMemcpyAsync((void*)Hd->row_ptr, Hh->row_ptr, sizeof(int32_t) * (size_t)(Hh->n + 1), cudaMemcpyHostToDevice, st));
  } else {
    const int64_t ld = dense_ld(Hh);
    if (cudaMalloc(&p, sizeof(cplx) * (size_t)Hh->n * (size_t)Hh->n) != cudaSuccess) return MAGNUS_ENOMEM;
    Hd->values = p;
    Hd->ld = Hh->n;
    CU_TRY(cudaMemcpy2DAsync(p, sizeof(cplx) * (size_t)Hh->n, Hh->values, sizeof(cplx) * (size_t)ld,
                             sizeof(cplx) * (size_t)Hh->n, (size_t)Hh->n, cudaMemcpyHostToDevice, st));
  }
  return MAGNUS_OK;
}

static void free_uploaded(magnus_matrix* Hd) {
  cudaFree((void*)Hd->values);
  cudaFree((void*)Hd->col_idx);
  cudaFree((void*)Hd->row_ptr);
}

int magnus_integrate_host(const magnus_matrix* H0_host, const magnus_matrix* H1_host, magnus_drive_fn f, void* user,
                          int scheme, const magnus_options* opt, double t0, double t_end, int64_t nsteps,
                          void* psi_host, magnus_stats* stats) {
  int rc = check_matrix(H0_host, "H0");
  if (rc) return rc;
  rc = check_matrix(H1_host, "H1");
  if (rc) return rc;
  if (!psi_host) { set_error("psi_host is NULL"); return MAGNUS_EINVAL; }
  rc = require_device();
  if (rc) return rc;
  cudaStream_t st = opt ? (cudaStream_t)opt->stream : (cudaStream_t)0;
  magnus_matrix d0, d1;
  std::memset(&d0, 0, sizeof d0);
  std::memset(&d1, 0, sizeof d1);
  cplx* psi = nullptr;
  magnus_handle h = nullptr;
  const size_t vb = sizeof(cplx) * (size_t)H0_host->n;
  rc = upload_matrix(H0_host, &d0, st);
  if (rc == MAGNUS_OK) rc = upload_matrix(H1_host, &d1, st);
  if (rc == MAGNUS_OK && cudaMalloc(&psi, vb) != cudaSuccess) rc = MAGNUS_ENOMEM;
  if (rc == MAGNUS_OK && cudaMemcpyAsync(psi, psi_host, vb, cudaMemcpyHostToDevice, st) != cudaSuccess) rc = MAGNUS_ECUDA;
  if (rc == MAGNUS_OK) rc = magnus_create(&h, &d0, &d1, f, user, scheme, opt);
  if (rc == MAGNUS_OK) rc = magnus_integrate(h, t0, t_end, nsteps, psi, stats);
  if (rc == MAGNUS_OK && cudaMemcpyAsync(psi_host, psi, vb, cudaMemcpyDeviceToHost, st) != cudaSuccess) rc = MAGNUS_ECUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess && rc == MAGNUS_OK) rc = MAGNUS_ECUDA;
  if (rc == MAGNUS_ENOMEM) { cudaGetLastError(); set_error("magnus_integrate_host: device allocation failed"); }
  magnus_destroy(h);
  cudaFree(psi);
  free_uploaded(&d0);
  free_uploaded(&d1);
  return rc;
}

// ---- single kernels -----------------------------------------------------------------
static int build_op(const magnus_matrix* H0, const magnus_matrix* H1, double g, OpRef* op, cplx** tmpM, Workspace* ws,
                    cudaStream_t st, int* assemble_blocks, SliceLayout* tmpS = nullptr) {
  *tmpM = nullptr;
  *assemble_blocks = -1;
  if (H0->format == MAGNUS_CSR) {
    op->dense = false;
    op->csr.n = H0->n;
    op->csr.nterms = H1 ? 2 : 1;
    op->csr.t[0] = csr_term(H0, 1.0, 0.0);
    op->csr.t[1] = H1 ? csr_term(H1, g, 0.0) : op->csr.t[0];
    op->csr.t[2] = op->csr.t[0];
    op->csr.unit_cap = 0;
    if (csr_unit_cap(op->csr, st, &op->csr.unit_cap) != MAGNUS_OK) op->csr.unit_cap = 0;
    if (tmpS && slice_layout_kind(ws->csr_kernel) != 0 &&
        slice_layout_build(op->csr, tmpS, st, slice_layout_kind(ws->csr_kernel) == 2,
                           ws->csr_kernel >= 6500 && ws->csr_kernel < 7000) == MAGNUS_OK)
      op->csr.slice = tmpS;
  } else {
    op->dense = true;
    op->dns.n = H0->n;
    if (H1) {
      if (cudaMalloc(tmpM, sizeof(cplx) * (size_t)H0->n * (size_t)H0->n) != cudaSuccess) {
        cudaGetLastError();
        set_error("assembled matrix allocation failed");
        return MAGNUS_ENOMEM;
      }
      *assemble_blocks = launch_dense_assemble(H0->n, (const cplx*)H0->values, dense_ld(H0), (const cplx*)H1->values,
                                               dense_ld(H1), g, *tmpM, ws, st);
      op->dns.ld = H0->n;
      op->dns.M = *tmpM;
    } else {
      op->dns.ld = dense_ld(H0);
      op->dns.M = (const cplx*)H0->values;
    }
  }
  return MAGNUS_OK;
}

int magnus_gershgorin(const magnus_matrix* H0, const magnus_matrix* H1, double g, void* stream, double* ab_host) {
  int rc = check_matrix(H0, "H0");
  if (rc) return rc;
  if (H1 && (rc = check_matrix(H1, "H1"))) return rc;
  if (H1 && (H1->format != H0->format || H1->n != H0->n)) { set_error("H0 and H1 differ"); return MAGNUS_EINVAL; }
  if (!ab_host) return MAGNUS_EINVAL;
  rc = require_device();
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  Workspace ws;
  rc = workspace_alloc(&ws, 1, st);
  if (rc) { workspace_free(&ws); return rc; }
  OpRef op;
  cplx* tmp = nullptr;
  int ab = -1;
  rc = build_op(H0, H1, g, &op, &tmp, &ws, st, &ab);
  if (rc == MAGNUS_OK)
    rc = ab >= 0 ? read_interval(ab, &ws, st, &ab_host[0], &ab_host[1]) : op_interval(op, &ws, st, &ab_host[0], &ab_host[1]);
  cudaFree(tmp);
  workspace_free(&ws);
  return rc;
}

int magnus_leja_iteration(const magnus_matrix* H0, const magnus_matrix* H1, double g, const void* w_in, void* w_out,
                          void* p, double inv_gamma, double shift, double d_re, double d_im, void* stream,
                          int csr_kernel, int reps, double* sums_host, float* ms_per_launch) {
  int rc = check_matrix(H0, "H0");
  if (rc) return rc;
  if (H1 && (rc = check_matrix(H1, "H1"))) return rc;
  if (H1 && (H1->format != H0->format || H1->n != H0->n)) { set_error("H0 and H1 differ"); return MAGNUS_EINVAL; }
  if (!w_in || !w_out || !p || w_in == w_out) { set_error("magnus_leja_iteration: bad vectors"); return MAGNUS_EINVAL; }
  if (reps < 1) reps = 1;
  rc = require_device();
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  Workspace ws;
  rc = workspace_alloc(&ws, 1, st);
  if (rc) { workspace_free(&ws); return rc; }
  ws.csr_kernel = csr_kernel;
  OpRef op;
  cplx* tmp = nullptr;
  SliceLayout tmp_slice;
  int ab = -1;
  rc = build_op(H0, H1, g, &op, &tmp, &ws, st, &ab, &tmp_slice);
  if (rc == MAGNUS_OK) {
    cudaMemsetAsync(ws.status, 0, sizeof(LejaStatus), st);
    cudaEventRecord(ws.ev[0], st);
    bool launched = true;
    for (int r = 0; r < reps; ++r)   // |d_k| = 1, tol = 0: the fused stop test only records the norms
      launched = launched && launch_iter(op, (const cplx*)w_in, (cplx*)w_out, (cplx*)p, inv_gamma, shift,
                                         make_double2(d_re, d_im), 1.0, 0.0, &ws, st) >= 0;
    cudaEventRecord(ws.ev[1], st);
    cudaMemcpyAsync(ws.status_host, ws.status, sizeof(LejaStatus), cudaMemcpyDeviceToHost, st);
    cudaError_t ke = cudaStreamSynchronize(st);
    if (ke == cudaSuccess) ke = cudaGetLastError();
    if (ke != cudaSuccess) {
      set_error("magnus_leja_iteration: kernel failed: %s", cudaGetErrorString(ke));
      cudaGetLastError();
      rc = MAGNUS_ECUDA;
    } else if (!launched) {
      set_error("magnus_leja_iteration: csr_kernel = %d selects no kernel for this operator", csr_kernel);
      rc = MAGNUS_EINVAL;
    } else {
      float ms = 0.f;
      cudaEventElapsedTime(&ms, ws.ev[0], ws.ev[1]);
      if (ms_per_launch) *ms_per_launch = ms / (float)reps;
      if (sums_host) {
        sums_host[0] = ws.status_host->norm_w2;
        sums_host[1] = ws.status_host->norm_p2;
      }
    }
  }
  cudaFree(tmp);
  slice_layout_free(&tmp_slice);
  workspace_free(&ws);
  return rc;
}

int magnus_zgemm(int64_t n, const void* A, int64_t lda, const void* B, int64_t ldb, void* C, int64_t ldc, void* stream,
                 float* ms) {
  if (n <= 0 || !A || !B || !C || C == A || C == B) { set_error("magnus_zgemm: bad arguments"); return MAGNUS_EINVAL; }
  if (lda == 0) lda = n;
  if (ldb == 0) ldb = n;
  if (ldc == 0) ldc = n;
  int rc = require_device();
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  cudaEvent_t e0, e1;
  CU_TRY(cudaEventCreate(&e0));
  CU_TRY(cudaEventCreate(&e1));
  ZgemmScratch zs;
  zgemm_scratch_alloc(&zs);
  cudaEventRecord(e0, st);
  rc = launch_zgemm(n, (const cplx*)A, lda, (const cplx*)B, ldb, (cplx*)C, ldc, st, &zs);
  cudaEventRecord(e1, st);
  if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) {
    set_error("magnus_zgemm: kernel failed");
    rc = MAGNUS_ECUDA;
  } else if (ms) {
    cudaEventElapsedTime(ms, e0, e1);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  zgemm_scratch_free(&zs);
  return rc;
}

int magnus_commutator_dense(int64_t n, const void* A, const void* B, void* K, void* work, void* stream) {
  if (n <= 0 || !A || !B || !K || !work || work == A || work == B || work == K) {
    set_error("magnus_commutator_dense: bad arguments");
    return MAGNUS_EINVAL;
  }
  int rc = require_device();
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  rc = launch_zgemm(n, (const cplx*)A, n, (const cplx*)B, n, (cplx*)work, n, st);   // P = A B
  if (rc) return rc;
  launch_dense_antiherm(n, (const cplx*)work, (cplx*)K, -1.0, st);                  // K = P - P^H
  CU_TRY(cudaStreamSynchronize(st));
  CU_TRY(cudaGetLastError());
  return MAGNUS_OK;
}

int magnus_omega_dense(int64_t n, const void* H0, int64_t ld0, const void* H1, int64_t ld1, double f1, double f2,
                       double tau, void* Omega, void* work_a2, void* work_p, void* stream, double* ab_host) {
  if (n <= 0 || !H0 || !H1 || !Omega || !work_a2 || !work_p || Omega == work_a2 || Omega == work_p ||
      work_a2 == work_p || Omega == H0 || Omega == H1) {
    set_error("magnus_omega_dense: bad arguments");
    return MAGNUS_EINVAL;
  }
  if (ld0 == 0) ld0 = n;
  if (ld1 == 0) ld1 = n;
  int rc = require_device();
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  Workspace ws;
  rc = workspace_alloc(&ws, 1, st);
  if (rc) { workspace_free(&ws); return rc; }
  // the same three launches magnus_step makes for M4 on dense H: S2 (A1, A2), D3 (P = A2 A1), D4 + S3
  launch_dense_assemble2(n, (const cplx*)H0, ld0, (const cplx*)H1, ld1, f1, f2, (cplx*)Omega, (cplx*)work_a2, &ws, st);
  rc = launch_zgemm(n, (const cplx*)work_a2, n, (const cplx*)Omega, n, (cplx*)work_p, n, st);
  if (rc == MAGNUS_OK) {
    const int nblk = launch_dense_omega(n, (cplx*)Omega, (const cplx*)work_a2, (const cplx*)work_p, 0.5, 0.5,
                                        std::sqrt(3.0) * tau / 12.0, &ws, st);
    double a = 0.0, b = 0.0;
    rc = read_interval(nblk, &ws, st, &a, &b);
    if (rc == MAGNUS_OK && ab_host) {
      ab_host[0] = a;
      ab_host[1] = b;
    }
    if (rc == MAGNUS_OK && cudaGetLastError() != cudaSuccess) rc = MAGNUS_ECUDA;
  } else {
    set_error("magnus_omega_dense: zgemm launch failed: %s", cudaGetErrorString(cudaGetLastError()));
  }
  workspace_free(&ws);
  return rc;
}

int magnus_commutator_csr(const magnus_matrix* A, const magnus_matrix* B, int64_t cap_nnz, int64_t* nnz_out,
                          int32_t* row_ptr_out, int32_t* col_idx_out, void* values_out, void* stream) {
  int rc = check_matrix(A, "A");
  if (rc) return rc;
  rc = check_matrix(B, "B");
  if (rc) return rc;
  if (A->format != MAGNUS_CSR || B->format != MAGNUS_CSR || A->n != B->n || !nnz_out) {
    set_error("magnus_commutator_csr: needs two CSR matrices of equal n");
    return MAGNUS_EINVAL;
  }
  if (cap_nnz > 0 && (!row_ptr_out || !col_idx_out || !values_out)) return MAGNUS_EINVAL;
  rc = require_device();
  if (rc) return rc;
  return csr_commutator(A, B, cap_nnz, nnz_out, row_ptr_out, col_idx_out, (cplx*)values_out, (cudaStream_t)stream);
}

int magnus_fp64_peaks(double* dmma_tflops, double* dfma_tflops, void* stream) {
  if (!dmma_tflops || !dfma_tflops) return MAGNUS_EINVAL;
  int rc = require_device();
  if (rc) return rc;
  return fp64_peaks(dmma_tflops, dfma_tflops, (cudaStream_t)stream);
}

}  // extern "C"
