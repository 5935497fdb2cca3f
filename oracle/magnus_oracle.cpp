// ORACLE -- TEST INFRASTRUCTURE ONLY.  NOT PART OF THE PRODUCT PATH.
//
// A plain, slow, obviously-correct CPU implementation of the hot path of
// arXiv 1709.06483 ("Magnus integrators on multicore CPUs and GPUs"): one time
// step of the 4th-order Magnus integrators Cf4 and M4 for i dpsi/dt = H(t) psi,
// H(t) = H0 + f(t) H1, with exp(-i h M) v computed by Newton interpolation at
// Leja points on a Gershgorin interval.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no
// code, header, table or constant with paper_1709_06483_b200/ (the CUDA path)
// and neither imports the other.
//
// Citations: "P:n" = /root/reference/PAPER.md line n; "c1..c7, g1..g16" = the
// readings of SURVEY.md section 8(c), restated in DESIGN.md section 3.
//
//   Scheme M4   P:97-101 (Method 2), P:260-264 (pseudocode)        -> step_m4
//   Scheme Cf4  P:130-134 (Method 4)                                -> step_cf4
//   Scheme M6   P:103-114 (Method 3; reading m6: the coefficient of B3)  -> m6_omega_dense / m6_omega_csr
//   Leja/Newton P:169-186 (formula and code fragment)               -> leja_expmv
//   early stop  P:188, P:229-231 (reading c6)                       -> leja_expmv
//   spectrum    P:190 (estimate "from the matrix"; Gershgorin, c4)  -> gershgorin_*
//               shortcut beside it (reading ti): Lanczos interval     -> lanczos_interval
//   Leja points P:169 ("see [11]"; reading c2)                      -> leja_points
//   d_i         P:171 (definition; reading c3: __float128 table)    -> divided_differences
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): every function below is pinned to
// closed forms / numpy.linalg.eigh / mpmath / invariants, EXCEPT the Leja
// iteration COUNT, which the paper never prints: "parity unpinned" for counts
// (only sanity: monotone in tol and |h|).
//
// Floating point: double for all vector work (the paper's precision, complex
// double P:194-203); __float128 only inside the divided-difference table.
// Parallelism: OpenMP "parallel for" over rows, nothing else; every sum is in
// stored order, norms are sequential, so results do not depend on the thread
// count.

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>

#include <quadmath.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;
typedef double (*drive_fn)(double t, void* user);

namespace {

const int kMaxDegree = 128;      // m_max (reading c6)
const double kThetaMax = 16.0;   // theta_max (reading c6)

// ---------------------------------------------------------------------------
// Leja points on [-2, 2]  ("chosen to be Leja points (see [11])"; c2)
//   l0 = 2, l1 = -2, l2 = 0, l3 = +2/sqrt(3) (exact tie, positive root taken),
//   l_k = argmax_{x in [-2,2]} prod_{j<k} |x - l_j|.
// In each gap between two neighbouring nodes the log-product is concave, so its
// maximum is the unique zero of g(x) = sum_j 1/(x - l_j), found by bisection;
// the gap with the largest product wins.
// ---------------------------------------------------------------------------
std::vector<double> leja_points(int m) {
  std::vector<double> pts;
  const double first[4] = {2.0, -2.0, 0.0, 2.0 / std::sqrt(3.0)};
  for (int k = 0; k < m && k < 4; ++k) pts.push_back(first[k]);
  while ((int)pts.size() < m) {
    std::vector<long double> s(pts.begin(), pts.end());
    std::sort(s.begin(), s.end());
    long double best_val = -1e300L, best_x = 0.0L;
    for (size_t gidx = 0; gidx + 1 < s.size(); ++gidx) {
      long double lo = s[gidx], hi = s[gidx + 1];
      for (int it = 0; it < 200; ++it) {
        long double mid = 0.5L * (lo + hi);
        if (mid == lo || mid == hi) break;
        long double g = 0.0L;
        for (size_t j = 0; j < s.size(); ++j) g += 1.0L / (mid - s[j]);
        if (g > 0.0L) lo = mid; else hi = mid;   // g decreases from +inf to -inf
      }
      long double x = 0.5L * (lo + hi);
      long double val = 0.0L;
      for (size_t j = 0; j < s.size(); ++j) val += logl(fabsl(x - s[j]));
      if (val > best_val) { best_val = val; best_x = x; }
    }
    pts.push_back((double)best_x);
  }
  return pts;
}

const std::vector<double>& leja_table() {
  static const std::vector<double> t = leja_points(kMaxDegree + 1);
  return t;
}

// ---------------------------------------------------------------------------
// Divided differences d_i = F[l_0, ..., l_i], F(x) = exp(-i theta x)
// ("d_i := exp[xi_0, ..., xi_i]"; reading c3: nodes are the FIXED Leja
// points of [-2,2] because the recurrence runs on B = (M - cI)/gamma, and the
// function carries theta = h*gamma).  Textbook recurrence, in __float128 so that
// tiny d_i (1e-14) still have ~1e-18 relative error after rounding to double.
// ---------------------------------------------------------------------------
void divided_differences(double theta, int m, cplx* out) {
  const std::vector<double>& l = leja_table();
  std::vector<__float128> re(m), im(m);
  for (int j = 0; j < m; ++j) {
    __float128 arg = (__float128)theta * (__float128)l[j];
    re[j] = cosq(arg);
    im[j] = -sinq(arg);
  }
  for (int k = 1; k < m; ++k) {
    for (int j = m - 1; j >= k; --j) {
      __float128 den = (__float128)l[j] - (__float128)l[j - k];
      re[j] = (re[j] - re[j - 1]) / den;
      im[j] = (im[j] - im[j - 1]) / den;
    }
  }
  for (int j = 0; j < m; ++j) out[j] = cplx((double)re[j], (double)im[j]);
}

// ---------------------------------------------------------------------------
// Matrices.  Dense: row-major n x n.  CSR: 0-based, columns ascending in a row.
// ---------------------------------------------------------------------------
struct Matrix {
  int64_t n;
  virtual void matvec(const cplx* w, cplx* y) const = 0;   // y = M w
  // raw Gershgorin bounds: a = min_i(Re M_ii - R_i), b = max_i(Re M_ii + R_i),
  // R_i = sum_{j != i} |M_ij|  (reading c4)
  virtual void gershgorin(double* a, double* b) const = 0;
  virtual ~Matrix() {}
};

struct DenseView : Matrix {
  const cplx* a;
  DenseView(int64_t n_, const cplx* a_) { n = n_; a = a_; }
  void matvec(const cplx* w, cplx* y) const override {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
      cplx s = 0.0;
      const cplx* row = a + i * n;
      for (int64_t j = 0; j < n; ++j) s += row[j] * w[j];
      y[i] = s;
    }
  }
  void gershgorin(double* lo, double* hi) const override {
    std::vector<double> dl(n), dh(n);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
      double R = 0.0;
      const cplx* row = a + i * n;
      for (int64_t j = 0; j < n; ++j) if (j != i) R += std::abs(row[j]);
      dl[i] = row[i].real() - R;
      dh[i] = row[i].real() + R;
    }
    *lo = *std::min_element(dl.begin(), dl.end());
    *hi = *std::max_element(dh.begin(), dh.end());
  }
};

struct CsrView : Matrix {
  const int32_t* rp; const int32_t* ci; const cplx* v;
  CsrView(int64_t n_, const int32_t* rp_, const int32_t* ci_, const cplx* v_) { n = n_; rp = rp_; ci = ci_; v = v_; }
  void matvec(const cplx* w, cplx* y) const override {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
      cplx s = 0.0;
      for (int32_t q = rp[i]; q < rp[i + 1]; ++q) s += v[q] * w[ci[q]];
      y[i] = s;
    }
  }
  void gershgorin(double* lo, double* hi) const override {
    std::vector<double> dl(n), dh(n);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
      double R = 0.0, d = 0.0;                      // an absent diagonal is 0
      for (int32_t q = rp[i]; q < rp[i + 1]; ++q) {
        if (ci[q] == i) d = v[q].real(); else R += std::abs(v[q]);
      }
      dl[i] = d - R;
      dh[i] = d + R;
    }
    *lo = *std::min_element(dl.begin(), dl.end());
    *hi = *std::max_element(dh.begin(), dh.end());
  }
};

// Owned sparse matrix with the two plain operations M4 needs on CSR input.
struct SpMat {
  int64_t n = 0;
  std::vector<int32_t> rp, ci;
  std::vector<cplx> v;
  CsrView view() const { return CsrView(n, rp.data(), ci.data(), v.data()); }
};

// C = alpha*A + beta*B on the union pattern (two-pointer merge of sorted rows).
SpMat sp_axpby(cplx alpha, const CsrView& A, cplx beta, const CsrView& B) {
  SpMat C; C.n = A.n; C.rp.assign(A.n + 1, 0);
  for (int64_t i = 0; i < A.n; ++i) {
    int32_t p = A.rp[i], q = B.rp[i];
    while (p < A.rp[i + 1] || q < B.rp[i + 1]) {
      int32_t ca = p < A.rp[i + 1] ? A.ci[p] : INT32_MAX;
      int32_t cb = q < B.rp[i + 1] ? B.ci[q] : INT32_MAX;
      if (ca == cb)      { C.ci.push_back(ca); C.v.push_back(alpha * A.v[p] + beta * B.v[q]); ++p; ++q; }
      else if (ca < cb)  { C.ci.push_back(ca); C.v.push_back(alpha * A.v[p]); ++p; }
      else               { C.ci.push_back(cb); C.v.push_back(beta * B.v[q]); ++q; }
    }
    C.rp[i + 1] = (int32_t)C.ci.size();
  }
  return C;
}

// C = A*B by the definition C_ij = sum_k A_ik B_kj, one dense accumulator row
// at a time; every structurally reachable (i,j) is stored, also if it sums to 0.
SpMat sp_mul(const CsrView& A, const CsrView& B) {
  int64_t n = A.n;
  std::vector<std::vector<int32_t>> cols(n);
  std::vector<std::vector<cplx>> vals(n);
#pragma omp parallel
  {
    std::vector<cplx> acc(n, cplx(0.0));
    std::vector<char> hit(n, 0);
    std::vector<int32_t> touched;
#pragma omp for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
      touched.clear();
      for (int32_t p = A.rp[i]; p < A.rp[i + 1]; ++p) {
        int32_t k = A.ci[p];
        for (int32_t q = B.rp[k]; q < B.rp[k + 1]; ++q) {
          int32_t j = B.ci[q];
          if (!hit[j]) { hit[j] = 1; touched.push_back(j); }
          acc[j] += A.v[p] * B.v[q];
        }
      }
      std::sort(touched.begin(), touched.end());
      for (int32_t j : touched) { cols[i].push_back(j); vals[i].push_back(acc[j]); acc[j] = 0.0; hit[j] = 0; }
    }
  }
  SpMat C; C.n = n; C.rp.assign(n + 1, 0);
  for (int64_t i = 0; i < n; ++i) C.rp[i + 1] = C.rp[i] + (int32_t)cols[i].size();
  C.ci.resize(C.rp[n]); C.v.resize(C.rp[n]);
  for (int64_t i = 0; i < n; ++i) {
    std::copy(cols[i].begin(), cols[i].end(), C.ci.begin() + C.rp[i]);
    std::copy(vals[i].begin(), vals[i].end(), C.v.begin() + C.rp[i]);
  }
  return C;
}

// Dense C = A*B, C_ij = sum_k A_ik B_kj with k ascending (i-k-j loop nest).
void dense_mul(int64_t n, const cplx* A, const cplx* B, cplx* C) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    cplx* crow = C + i * n;
    for (int64_t j = 0; j < n; ++j) crow[j] = 0.0;
    for (int64_t k = 0; k < n; ++k) {
      cplx aik = A[i * n + k];
      const cplx* brow = B + k * n;
      for (int64_t j = 0; j < n; ++j) crow[j] += aik * brow[j];
    }
  }
}

double norm2(const cplx* x, int64_t n) {
  double s = 0.0;
  for (int64_t i = 0; i < n; ++i) s += x[i].real() * x[i].real() + x[i].imag() * x[i].imag();
  return std::sqrt(s);
}

// Reading c4: widen [a,b] outward to a grid of spacing 2^(E-12),
// E = ceil(log2(b-a)), so that two implementations that sum the row radii in a
// different order still obtain bit-identical c, gamma, theta.
void snap_interval(double* a, double* b) {
  double width = *b - *a;
  if (!(width > 0.0)) return;
  int e;
  double f = std::frexp(width, &e);      // width = f * 2^e, f in [0.5, 1)
  int E = (f == 0.5) ? e - 1 : e;        // ceil(log2(width))
  double delta = std::ldexp(1.0, E - 12);
  *a = std::floor(*a / delta) * delta;
  *b = std::ceil(*b / delta) * delta;
}

}  // namespace

extern "C" {

struct oracle_expmv_info {
  int32_t iters;       // mat-vecs used (summed over sub-steps)
  int32_t substeps;    // s
  int32_t status;      // 0 ok, -4 = m_max reached without meeting tol
  int32_t _pad;
  double a, b;         // snapped Gershgorin interval
  double theta;        // (h/s) * gamma
  double err_est;      // e_k + e_{k-1} at the stop
};

}  // extern "C"

namespace {

// ---------------------------------------------------------------------------
// Shortcut "tight spectral interval" (P:190 leaves the estimate of the spectrum open, NS fixes
// Gershgorin for the mandated path; this is the option beside it, reading ti in DESIGN.md section 3).
// m steps of the Lanczos process on the Hermitian M, started at the vector v that is about to be propagated:
//   q_1 = v / ||v||;   for j = 1..m:   u = M q_j - beta_{j-1} q_{j-1};   alpha_j = Re(q_j^H u);
//                                      r = u - alpha_j q_j;   beta_j = ||r||;   q_{j+1} = r / beta_j
// (stopped early -- an invariant subspace -- when beta_j <= 1e-12 * max_i max(|alpha_i|, beta_i)).
// T = tridiag(alpha_1..alpha_m; beta_1..beta_{m-1}); its extreme eigenvalues theta_min, theta_max (Ritz values: inside
// the spectrum of M) are widened by the norm of the last residual:  [theta_min - beta_m, theta_max + beta_m].
// The eigenvalues of the small T come from cyclic Jacobi rotations on the dense m x m matrix.
// ---------------------------------------------------------------------------
int g_lanczos_steps = 0;   // 0: Gershgorin (the mandated path); m > 0: the interval of every leja_expmv call from m Lanczos steps

void jacobi_eigenvalues(std::vector<double>& A, int m, std::vector<double>& ev) {   // A: m x m symmetric, row-major
  for (int sweep = 0; sweep < 60; ++sweep) {
    double off = 0.0;
    for (int p = 0; p < m; ++p)
      for (int q = p + 1; q < m; ++q) off += A[p * m + q] * A[p * m + q];
    if (off == 0.0) break;
    for (int p = 0; p < m; ++p)
      for (int q = p + 1; q < m; ++q) {
        const double apq = A[p * m + q];
        if (apq == 0.0) continue;
        const double tau = (A[q * m + q] - A[p * m + p]) / (2.0 * apq);
        const double t = (tau >= 0.0 ? 1.0 : -1.0) / (std::fabs(tau) + std::sqrt(1.0 + tau * tau));
        const double c = 1.0 / std::sqrt(1.0 + t * t), sn = t * c;
        for (int k = 0; k < m; ++k) {   // columns p, q
          const double akp = A[k * m + p], akq = A[k * m + q];
          A[k * m + p] = c * akp - sn * akq;
          A[k * m + q] = sn * akp + c * akq;
        }
        for (int k = 0; k < m; ++k) {   // rows p, q
          const double apk = A[p * m + k], aqk = A[q * m + k];
          A[p * m + k] = c * apk - sn * aqk;
          A[q * m + k] = sn * apk + c * aqk;
        }
      }
  }
  ev.resize(m);
  for (int i = 0; i < m; ++i) ev[i] = A[i * m + i];
}

// returns the number of Lanczos steps actually taken (0: v = 0, interval left untouched); alpha, beta (nullable): m entries
int lanczos_interval(const Matrix& M, const cplx* v, int m, double* a, double* b, double* alpha_out, double* beta_out) {
  const int64_t n = M.n;
  const double nv = norm2(v, n);
  if (!(nv > 0.0) || m < 1) return 0;
  std::vector<cplx> qp(n, cplx(0.0)), q(n), u(n);
  for (int64_t i = 0; i < n; ++i) q[i] = v[i] / nv;
  std::vector<double> alpha, beta;
  double beta_prev = 0.0, scale = 0.0;
  for (int j = 0; j < m; ++j) {
    M.matvec(q.data(), u.data());
    for (int64_t i = 0; i < n; ++i) u[i] -= beta_prev * qp[i];
    double al = 0.0;
    for (int64_t i = 0; i < n; ++i) al += (std::conj(q[i]) * u[i]).real();
    for (int64_t i = 0; i < n; ++i) u[i] -= al * q[i];
    const double be = norm2(u.data(), n);
    alpha.push_back(al);
    beta.push_back(be);
    scale = std::max(scale, std::max(std::fabs(al), be));
    if (be <= 1e-12 * scale) break;              // invariant subspace reached: T is exact
    for (int64_t i = 0; i < n; ++i) { qp[i] = q[i]; q[i] = u[i] / be; }
    beta_prev = be;
  }
  const int k = (int)alpha.size();
  std::vector<double> T((size_t)k * k, 0.0), ev;
  for (int i = 0; i < k; ++i) {
    T[i * k + i] = alpha[i];
    if (i + 1 < k) T[i * k + i + 1] = T[(i + 1) * k + i] = beta[i];
  }
  jacobi_eigenvalues(T, k, ev);
  const double lo = *std::min_element(ev.begin(), ev.end()), hi = *std::max_element(ev.begin(), ev.end());
  *a = lo - beta[k - 1];
  *b = hi + beta[k - 1];
  for (int i = 0; i < k; ++i) {
    if (alpha_out) alpha_out[i] = alpha[i];
    if (beta_out) beta_out[i] = beta[i];
  }
  return k;
}

// ---------------------------------------------------------------------------
// exp(-i h M) v by Newton interpolation at Leja points (c3-c7).
//   B = (M - cI)/gamma has its spectrum in [-2,2]; exp(-ihM) = e^{-ihc} exp(-i theta B).
//   w_0 = v, p_0 = d_0 v;
//   w_k = (1/gamma) M w_{k-1} - (c/gamma + l_{k-1}) w_{k-1};  p_k = p_{k-1} + d_k w_k
//   e_k = |d_k| ||w_k||_2;  stop at the first k >= 1 with e_k + e_{k-1} <= tol ||p_k||_2 (c6)
//   s = max(1, ceil(|h gamma| / theta_max)) sub-steps of h/s share interval and table (c6)
// ---------------------------------------------------------------------------
int leja_expmv(const Matrix& M, const cplx* v_in, cplx* v_out, double h, double tol,
               oracle_expmv_info* info) {
  const int64_t n = M.n;
  const std::vector<double>& l = leja_table();
  double a, b;
  M.gershgorin(&a, &b);
  if (g_lanczos_steps > 0) {
    // reading ti: the Lanczos interval is an ESTIMATE (P:190 asks for no more), not an enclosure, and its widening by
    // beta_m can stick out of the Gershgorin enclosure; the spectrum lies in both only where they overlap, so the
    // interval used is their intersection (Gershgorin alone when Lanczos declines or the two do not overlap).
    double la, lb;
    if (lanczos_interval(M, v_in, g_lanczos_steps, &la, &lb, nullptr, nullptr) != 0) {
      const double ia = std::max(a, la), ib = std::min(b, lb);
      if (ia <= ib) { a = ia; b = ib; }
    }
  }
  snap_interval(&a, &b);
  const double c = 0.5 * (a + b);
  const double gamma = 0.25 * (b - a);
  oracle_expmv_info loc;
  std::memset(&loc, 0, sizeof loc);
  loc.a = a; loc.b = b;
  std::vector<cplx> v(v_in, v_in + n);
  if (gamma == 0.0) {                       // M = c I: exact, no iterations
    const cplx ph(std::cos(h * c), -std::sin(h * c));
    for (int64_t i = 0; i < n; ++i) v_out[i] = ph * v[i];
    loc.substeps = 1;
    if (info) *info = loc;
    return 0;
  }
  const int s = std::max(1, (int)std::ceil(std::fabs(h * gamma) / kThetaMax));
  const double hs = h / s;
  const double theta = hs * gamma;
  loc.substeps = s; loc.theta = theta;
  std::vector<cplx> d(kMaxDegree + 1);
  divided_differences(theta, kMaxDegree + 1, d.data());
  std::vector<cplx> w(n), wn(n), p(n), y(n);
  const cplx phase(std::cos(hs * c), -std::sin(hs * c));
  for (int sub = 0; sub < s; ++sub) {
    for (int64_t i = 0; i < n; ++i) { w[i] = v[i]; p[i] = d[0] * v[i]; }
    double e_prev = std::abs(d[0]) * norm2(w.data(), n);
    bool done = false;
    for (int k = 1; k <= kMaxDegree; ++k) {
      M.matvec(w.data(), y.data());
      const double shift = c / gamma + l[k - 1];
      const double inv_gamma = 1.0 / gamma;
      for (int64_t i = 0; i < n; ++i) {
        wn[i] = inv_gamma * y[i] - shift * w[i];
        p[i] += d[k] * wn[i];
      }
      w.swap(wn);
      loc.iters += 1;
      const double e_k = std::abs(d[k]) * norm2(w.data(), n);
      loc.err_est = e_k + e_prev;
      if (e_k + e_prev <= tol * norm2(p.data(), n)) { done = true; break; }
      e_prev = e_k;
    }
    if (!done) { loc.status = -4; if (info) *info = loc; return -4; }
    for (int64_t i = 0; i < n; ++i) v[i] = phase * p[i];     // c7
  }
  for (int64_t i = 0; i < n; ++i) v_out[i] = v[i];
  if (info) *info = loc;
  return 0;
}

// Gauss nodes and Cf4 coefficients.
const double kC1 = 0.5 - std::sqrt(3.0) / 6.0;
const double kC2 = 0.5 + std::sqrt(3.0) / 6.0;
const double kAlpha1 = (3.0 - 2.0 * std::sqrt(3.0)) / 12.0;
const double kAlpha2 = (3.0 + 2.0 * std::sqrt(3.0)) / 12.0;

// Scheme codes: 0 = Cf4, 1 = M4, 2 = M2, 3 = Cf4:3, 4 = M6, 101 = M4 with the commutator sign flipped
// (a NEGATIVE CONTROL for the order test only: it must drop to order 2), 104 = M6 with the coefficient of B3
// exactly as PAPER.md prints it (1/2; NEGATIVE CONTROL: see m6_c3).
double m4_kappa(int scheme, double tau) {
  double kappa = std::sqrt(3.0) * tau / 12.0;
  return scheme == 101 ? -kappa : kappa;
}

// Commutator-free schemes as a list of exponentials exp(-i h_e (H0 + g_e H1)), in the order
// they ACT on psi (the right-most factor of the printed product first).  With A_j = -i H(t_j),
// H = H0 + f H1:  exp(tau sum_j a_ij A_j) = exp(-i tau s_i (H0 + (sum_j a_ij f_j / s_i) H1)),
// s_i = sum_j a_ij.
//   scheme 0, Cf4: rows (a1, a2) and (a2, a1); the row (a2, a1) acts first.
//   scheme 2, M2:   one exponential, h = tau, g = f(t + tau/2).
//   scheme 3, Cf4:3: nodes c = 1/2 -+ sqrt(15)/10 and 1/2, the printed 3x3 alpha;
//                                row 3 acts first.
// Returns the number of exponentials, 0 if the scheme is not commutator-free.
int cf_exponentials(int scheme, drive_fn f, void* user, double t, double tau, double* h, double* g) {
  if (scheme == 0) {
    const double f1 = f(t + kC1 * tau, user), f2 = f(t + kC2 * tau, user);
    // alpha1 + alpha2 = 1/2 exactly (reading c1): h = tau/2, g_a = 2(a2 f1 + a1 f2), g_b = 2(a1 f1 + a2 f2)
    h[0] = h[1] = 0.5 * tau;
    g[0] = 2.0 * (kAlpha2 * f1 + kAlpha1 * f2);
    g[1] = 2.0 * (kAlpha1 * f1 + kAlpha2 * f2);
    return 2;
  }
  if (scheme == 2) {
    h[0] = tau;
    g[0] = f(t + 0.5 * tau, user);
    return 1;
  }
  if (scheme == 3) {
    const double r15 = std::sqrt(15.0);
    const double fn[3] = {f(t + (0.5 - r15 / 10.0) * tau, user), f(t + 0.5 * tau, user),
                          f(t + (0.5 + r15 / 10.0) * tau, user)};
    const double am = 37.0 / 240.0 - 10.0 * r15 / 261.0, ap = 37.0 / 240.0 + 10.0 * r15 / 261.0;
    const double alpha[3][3] = {{am, -1.0 / 30.0, ap}, {-11.0 / 360.0, 23.0 / 45.0, -11.0 / 360.0}, {ap, -1.0 / 30.0, am}};
    for (int e = 0; e < 3; ++e) {
      const double* row = alpha[2 - e];                                    // row 3 acts first
      const double s = row[0] + row[1] + row[2];
      h[e] = tau * s;
      g[e] = (row[0] * fn[0] + row[1] * fn[1] + row[2] * fn[2]) / s;
    }
    return 3;
  }
  return 0;
}

int exponentials_per_step(int scheme) { return scheme == 0 ? 2 : scheme == 3 ? 3 : 1; }

// ---------------------------------------------------------------------------
// M6 (Method 3).  With A_j = A(t + c_j tau) = -i H(t_j), c = 1/2 - sqrt(15)/10, 1/2, 1/2 + sqrt(15)/10:
//   B1 = tau A2,  B2 = (sqrt(15)/3) tau (A3 - A1),  B3 = (10/3) tau (A3 - 2 A2 + A1),
//   Omega = B1 + c3 B3 + (1/240) [ -20 B1 - B3 + [B1, B2],  B2 - (1/60) [B1, 2 B3 + [B1, B2]] ],
//   psi <- exp(Omega) psi = exp(-i tau Omega_H) psi,  Omega_H = (i / tau) Omega  (Hermitian).
// Reading m6: PAPER.md l.105 prints the coefficient of B3 as 1/2.  For A(t) = a0 + a1 s + a2 s^2 (s measured from
// the midpoint) B1 = tau a0 and B3 = tau^3 a2 exactly, while the first Magnus term is int A = tau a0 + tau^3 a2 / 12:
// the coefficient must be c3 = 1/12 for the scheme to be consistent beyond order 2 (the extracted formula lost a
// digit).  tests/test_oracle_magnus.py shows order 6 with 1/12 and order 2 with the printed 1/2 (scheme 104).
// Every commutator is formed by its plain definition X Y - Y X (two products).
// ---------------------------------------------------------------------------
double m6_c3(int scheme) { return scheme == 104 ? 0.5 : 1.0 / 12.0; }

void m6_nodes(drive_fn f, void* user, double t, double tau, double* fn) {
  const double r15 = std::sqrt(15.0);
  fn[0] = f(t + (0.5 - r15 / 10.0) * tau, user);
  fn[1] = f(t + 0.5 * tau, user);
  fn[2] = f(t + (0.5 + r15 / 10.0) * tau, user);
}

void dense_comm(int64_t n, const cplx* X, const cplx* Y, cplx* K) {
  std::vector<cplx> xy(n * n), yx(n * n);
  dense_mul(n, X, Y, xy.data());
  dense_mul(n, Y, X, yx.data());
#pragma omp parallel for schedule(static)
  for (int64_t q = 0; q < n * n; ++q) K[q] = xy[q] - yx[q];
}

// Omega_H of one M6 step, dense.
void m6_omega_dense(int64_t n, const cplx* H0, const cplx* H1, const double* fn, double tau, double c3, cplx* OmH) {
  const int64_t nn = n * n;
  const cplx mi(0.0, -1.0);
  const double r15 = std::sqrt(15.0);
  std::vector<cplx> B1(nn), B2(nn), B3(nn), C1(nn), T(nn), C2(nn), L(nn), R(nn), K(nn);
#pragma omp parallel for schedule(static)
  for (int64_t q = 0; q < nn; ++q) {
    const cplx A1 = mi * (H0[q] + fn[0] * H1[q]), A2 = mi * (H0[q] + fn[1] * H1[q]), A3 = mi * (H0[q] + fn[2] * H1[q]);
    B1[q] = tau * A2;
    B2[q] = (r15 / 3.0) * tau * (A3 - A1);
    B3[q] = (10.0 / 3.0) * tau * (A3 - 2.0 * A2 + A1);
  }
  dense_comm(n, B1.data(), B2.data(), C1.data());                    // [B1, B2]
#pragma omp parallel for schedule(static)
  for (int64_t q = 0; q < nn; ++q) T[q] = 2.0 * B3[q] + C1[q];
  dense_comm(n, B1.data(), T.data(), C2.data());                     // [B1, 2 B3 + [B1, B2]]
#pragma omp parallel for schedule(static)
  for (int64_t q = 0; q < nn; ++q) {
    L[q] = -20.0 * B1[q] - B3[q] + C1[q];
    R[q] = B2[q] - C2[q] / 60.0;
  }
  dense_comm(n, L.data(), R.data(), K.data());
  const cplx i_over_tau(0.0, 1.0 / tau);
#pragma omp parallel for schedule(static)
  for (int64_t q = 0; q < nn; ++q) OmH[q] = i_over_tau * (B1[q] + c3 * B3[q] + K[q] / 240.0);
}

SpMat sp_comm(const CsrView& X, const CsrView& Y) {
  SpMat xy = sp_mul(X, Y), yx = sp_mul(Y, X);
  return sp_axpby(1.0, xy.view(), -1.0, yx.view());
}

// Omega_H of one M6 step, CSR (same formulas on sparse matrices).
SpMat m6_omega_csr(const CsrView& H0, const CsrView& H1, const double* fn, double tau, double c3) {
  const cplx mi(0.0, -1.0);
  const double r15 = std::sqrt(15.0);
  SpMat A1 = sp_axpby(mi, H0, mi * fn[0], H1), A2 = sp_axpby(mi, H0, mi * fn[1], H1), A3 = sp_axpby(mi, H0, mi * fn[2], H1);
  SpMat B1 = sp_axpby(tau, A2.view(), 0.0, A2.view());
  SpMat B2 = sp_axpby((r15 / 3.0) * tau, A3.view(), -(r15 / 3.0) * tau, A1.view());
  SpMat S13 = sp_axpby(1.0, A3.view(), 1.0, A1.view());
  SpMat B3 = sp_axpby((10.0 / 3.0) * tau, S13.view(), -(20.0 / 3.0) * tau, A2.view());
  SpMat C1 = sp_comm(B1.view(), B2.view());
  SpMat T = sp_axpby(2.0, B3.view(), 1.0, C1.view());
  SpMat C2 = sp_comm(B1.view(), T.view());
  SpMat L0 = sp_axpby(-20.0, B1.view(), -1.0, B3.view());
  SpMat L = sp_axpby(1.0, L0.view(), 1.0, C1.view());
  SpMat R = sp_axpby(1.0, B2.view(), -1.0 / 60.0, C2.view());
  SpMat K = sp_comm(L.view(), R.view());
  SpMat O1 = sp_axpby(1.0, B1.view(), c3, B3.view());
  const cplx i_over_tau(0.0, 1.0 / tau);
  return sp_axpby(i_over_tau, O1.view(), i_over_tau / 240.0, K.view());
}

// One step on dense H0, H1.  Cf4: P:132-134 with A = -iH (c1): first
// exp(-i tau/2 (H0 + g_a H1)), g_a = 2(alpha2 f1 + alpha1 f2), then
// exp(-i tau/2 (H0 + g_b H1)), g_b = 2(alpha1 f1 + alpha2 f2).
// M4: P:262 lines 1-10: A1, A2, K = A2 A1 - A1 A2 by the plain definition,
// Omega_H = (A1 + A2)/2 - i (sqrt(3) tau / 12) K, psi <- exp(-i tau Omega_H) psi.
int step_dense(int64_t n, const cplx* H0, const cplx* H1, drive_fn f, void* user, int scheme,
               double t, double tau, cplx* psi, double tol, oracle_expmv_info* infos) {
  const int64_t nn = n * n;
  double hh[3], gg[3];
  const int ncf = cf_exponentials(scheme, f, user, t, tau, hh, gg);
  if (ncf > 0) {
    std::vector<cplx> M(nn);
    for (int e = 0; e < ncf; ++e) {
#pragma omp parallel for schedule(static)
      for (int64_t q = 0; q < nn; ++q) M[q] = H0[q] + gg[e] * H1[q];
      int rc = leja_expmv(DenseView(n, M.data()), psi, psi, hh[e], tol, infos ? infos + e : nullptr);
      if (rc) return rc;
    }
    return 0;
  }
  if (scheme == 4 || scheme == 104) {
    double fn[3];
    m6_nodes(f, user, t, tau, fn);
    std::vector<cplx> OmH(nn);
    m6_omega_dense(n, H0, H1, fn, tau, m6_c3(scheme), OmH.data());
    return leja_expmv(DenseView(n, OmH.data()), psi, psi, tau, tol, infos);
  }
  const double f1 = f(t + kC1 * tau, user), f2 = f(t + kC2 * tau, user);
  std::vector<cplx> A1(nn), A2(nn), P21(nn), P12(nn), Om(nn);
#pragma omp parallel for schedule(static)
  for (int64_t q = 0; q < nn; ++q) { A1[q] = H0[q] + f1 * H1[q]; A2[q] = H0[q] + f2 * H1[q]; }
  dense_mul(n, A2.data(), A1.data(), P21.data());
  dense_mul(n, A1.data(), A2.data(), P12.data());
  const cplx mi_kappa(0.0, -m4_kappa(scheme, tau));
#pragma omp parallel for schedule(static)
  for (int64_t q = 0; q < nn; ++q) Om[q] = 0.5 * (A1[q] + A2[q]) + mi_kappa * (P21[q] - P12[q]);
  return leja_expmv(DenseView(n, Om.data()), psi, psi, tau, tol, infos);
}

int step_csr(const CsrView& H0, const CsrView& H1, drive_fn f, void* user, int scheme,
             double t, double tau, cplx* psi, double tol, oracle_expmv_info* infos) {
  double hh[3], gg[3];
  const int ncf = cf_exponentials(scheme, f, user, t, tau, hh, gg);
  if (ncf > 0) {
    for (int e = 0; e < ncf; ++e) {
      SpMat M = sp_axpby(1.0, H0, gg[e], H1);
      int rc = leja_expmv(M.view(), psi, psi, hh[e], tol, infos ? infos + e : nullptr);
      if (rc) return rc;
    }
    return 0;
  }
  if (scheme == 4 || scheme == 104) {
    double fn[3];
    m6_nodes(f, user, t, tau, fn);
    SpMat OmH = m6_omega_csr(H0, H1, fn, tau, m6_c3(scheme));
    return leja_expmv(OmH.view(), psi, psi, tau, tol, infos);
  }
  const double f1 = f(t + kC1 * tau, user), f2 = f(t + kC2 * tau, user);
  SpMat A1 = sp_axpby(1.0, H0, f1, H1), A2 = sp_axpby(1.0, H0, f2, H1);
  SpMat P21 = sp_mul(A2.view(), A1.view()), P12 = sp_mul(A1.view(), A2.view());
  SpMat K = sp_axpby(1.0, P21.view(), -1.0, P12.view());
  SpMat S = sp_axpby(0.5, A1.view(), 0.5, A2.view());
  SpMat Om = sp_axpby(1.0, S.view(), cplx(0.0, -m4_kappa(scheme, tau)), K.view());
  return leja_expmv(Om.view(), psi, psi, tau, tol, infos);
}

}  // namespace

extern "C" {

int oracle_max_degree() { return kMaxDegree; }

// 0 = Gershgorin interval (mandated path); m > 0 = shortcut "tight interval": m Lanczos steps per exponential
void oracle_set_lanczos_steps(int m) { g_lanczos_steps = m; }
int oracle_get_lanczos_steps() { return g_lanczos_steps; }

// raw (unsnapped) interval; returns the steps taken; alpha, beta: capacity m
int oracle_lanczos_interval_dense(int64_t n, const double* M, const double* v, int m, double* ab, double* alpha, double* beta) {
  return lanczos_interval(DenseView(n, reinterpret_cast<const cplx*>(M)), reinterpret_cast<const cplx*>(v), m, &ab[0], &ab[1],
                          alpha, beta);
}
int oracle_lanczos_interval_csr(int64_t n, const int32_t* rp, const int32_t* ci, const double* val, const double* v, int m,
                                double* ab, double* alpha, double* beta) {
  return lanczos_interval(CsrView(n, rp, ci, reinterpret_cast<const cplx*>(val)), reinterpret_cast<const cplx*>(v), m, &ab[0],
                          &ab[1], alpha, beta);
}

int oracle_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void oracle_set_num_threads(int t) {
#ifdef _OPENMP
  omp_set_num_threads(t);
#else
  (void)t;
#endif
}

void oracle_leja_points(int m, double* out) {
  std::vector<double> p = leja_points(m);
  std::copy(p.begin(), p.end(), out);
}

// out: m complex numbers (interleaved re, im)
void oracle_divided_differences(double theta, int m, double* out) {
  divided_differences(theta, m, reinterpret_cast<cplx*>(out));
}

void oracle_snap_interval(double* a, double* b) { snap_interval(a, b); }

// raw[0..1] = unsnapped (a, b); snapped[0..1] = after reading c4's grid.
void oracle_gershgorin_dense(int64_t n, const double* M, double* raw, double* snapped) {
  DenseView V(n, reinterpret_cast<const cplx*>(M));
  V.gershgorin(&raw[0], &raw[1]);
  snapped[0] = raw[0]; snapped[1] = raw[1];
  snap_interval(&snapped[0], &snapped[1]);
}

void oracle_gershgorin_csr(int64_t n, const int32_t* rp, const int32_t* ci, const double* v,
                           double* raw, double* snapped) {
  CsrView V(n, rp, ci, reinterpret_cast<const cplx*>(v));
  V.gershgorin(&raw[0], &raw[1]);
  snapped[0] = raw[0]; snapped[1] = raw[1];
  snap_interval(&snapped[0], &snapped[1]);
}

void oracle_matvec_dense(int64_t n, const double* M, const double* w, double* y) {
  DenseView(n, reinterpret_cast<const cplx*>(M)).matvec(reinterpret_cast<const cplx*>(w), reinterpret_cast<cplx*>(y));
}

void oracle_matvec_csr(int64_t n, const int32_t* rp, const int32_t* ci, const double* v,
                       const double* w, double* y) {
  CsrView(n, rp, ci, reinterpret_cast<const cplx*>(v)).matvec(reinterpret_cast<const cplx*>(w), reinterpret_cast<cplx*>(y));
}

int oracle_leja_expmv_dense(int64_t n, const double* M, const double* v_in, double* v_out,
                            double h, double tol, oracle_expmv_info* info) {
  return leja_expmv(DenseView(n, reinterpret_cast<const cplx*>(M)), reinterpret_cast<const cplx*>(v_in),
                    reinterpret_cast<cplx*>(v_out), h, tol, info);
}

int oracle_leja_expmv_csr(int64_t n, const int32_t* rp, const int32_t* ci, const double* v,
                          const double* v_in, double* v_out, double h, double tol, oracle_expmv_info* info) {
  return leja_expmv(CsrView(n, rp, ci, reinterpret_cast<const cplx*>(v)), reinterpret_cast<const cplx*>(v_in),
                    reinterpret_cast<cplx*>(v_out), h, tol, info);
}

// C = A B by the definition (P:262 line 6 "A_4 = A_2 A_1"): the product the commutator is made of.
void oracle_matmul_dense(int64_t n, const double* A, const double* B, double* Cout) {
  dense_mul(n, reinterpret_cast<const cplx*>(A), reinterpret_cast<const cplx*>(B), reinterpret_cast<cplx*>(Cout));
}

// K = A B - B A by the plain definition (P:262 lines 6-8 with A = A2, B = A1).
void oracle_commutator_dense(int64_t n, const double* A, const double* B, double* K) {
  const cplx* a = reinterpret_cast<const cplx*>(A);
  const cplx* b = reinterpret_cast<const cplx*>(B);
  cplx* k = reinterpret_cast<cplx*>(K);
  std::vector<cplx> ab(n * n), ba(n * n);
  dense_mul(n, a, b, ab.data());
  dense_mul(n, b, a, ba.data());
  for (int64_t q = 0; q < n * n; ++q) k[q] = ab[q] - ba[q];
}

// Sparse K = A B - B A.  Two calls: with cap = 0 only *nnz_out is written; with
// cap >= nnz the three arrays are filled.
int oracle_commutator_csr(int64_t n, const int32_t* arp, const int32_t* aci, const double* av,
                          const int32_t* brp, const int32_t* bci, const double* bv,
                          int64_t cap, int64_t* nnz_out, int32_t* rp_out, int32_t* ci_out, double* v_out) {
  CsrView A(n, arp, aci, reinterpret_cast<const cplx*>(av)), B(n, brp, bci, reinterpret_cast<const cplx*>(bv));
  SpMat AB = sp_mul(A, B), BA = sp_mul(B, A);
  SpMat K = sp_axpby(1.0, AB.view(), -1.0, BA.view());
  *nnz_out = (int64_t)K.ci.size();
  if (cap < *nnz_out) return 1;
  std::copy(K.rp.begin(), K.rp.end(), rp_out);
  std::copy(K.ci.begin(), K.ci.end(), ci_out);
  std::memcpy(v_out, K.v.data(), K.v.size() * sizeof(cplx));
  return 0;
}

// One step t -> t + tau.  infos: room for 3 entries (Cf4:3 uses all, Cf4 two, M4 and M2 the first).
// Omega_H of one M6 step (dense) at the three node values fn[0..2] of f: exposed so that its structure can be pinned.
void oracle_m6_omega_dense(int64_t n, const double* H0, const double* H1, const double* fn, double tau, double* out) {
  m6_omega_dense(n, reinterpret_cast<const cplx*>(H0), reinterpret_cast<const cplx*>(H1), fn, tau, m6_c3(4),
                 reinterpret_cast<cplx*>(out));
}

int oracle_magnus_step_dense(int64_t n, const double* H0, const double* H1, drive_fn f, void* user,
                             int scheme, double t, double tau, double* psi, double tol,
                             oracle_expmv_info* infos) {
  return step_dense(n, reinterpret_cast<const cplx*>(H0), reinterpret_cast<const cplx*>(H1), f, user, scheme,
                    t, tau, reinterpret_cast<cplx*>(psi), tol, infos);
}

int oracle_magnus_step_csr(int64_t n, const int32_t* rp0, const int32_t* ci0, const double* v0,
                           const int32_t* rp1, const int32_t* ci1, const double* v1, drive_fn f, void* user,
                           int scheme, double t, double tau, double* psi, double tol,
                           oracle_expmv_info* infos) {
  CsrView H0(n, rp0, ci0, reinterpret_cast<const cplx*>(v0)), H1(n, rp1, ci1, reinterpret_cast<const cplx*>(v1));
  return step_csr(H0, H1, f, user, scheme, t, tau, reinterpret_cast<cplx*>(psi), tol, infos);
}

// nsteps steps of size tau = (t_end - t0)/nsteps from t_n = t0 + n tau (g16).
// iters_out (nullable): one entry per exponential, in call order (2 per Cf4
// step, 1 per M4 step), capacity iters_cap.
int oracle_magnus_integrate_dense(int64_t n, const double* H0, const double* H1, drive_fn f, void* user,
                                  int scheme, double t0, double t_end, int64_t nsteps, double* psi,
                                  double tol, int32_t* iters_out, int64_t iters_cap) {
  const double tau = (t_end - t0) / (double)nsteps;
  const int per = exponentials_per_step(scheme);
  for (int64_t s = 0; s < nsteps; ++s) {
    oracle_expmv_info infos[3];
    int rc = oracle_magnus_step_dense(n, H0, H1, f, user, scheme, t0 + (double)s * tau, tau, psi, tol, infos);
    if (rc) return rc;
    for (int e = 0; e < per; ++e)
      if (iters_out && s * per + e < iters_cap) iters_out[s * per + e] = infos[e].iters;
  }
  return 0;
}

int oracle_magnus_integrate_csr(int64_t n, const int32_t* rp0, const int32_t* ci0, const double* v0,
                                const int32_t* rp1, const int32_t* ci1, const double* v1, drive_fn f, void* user,
                                int scheme, double t0, double t_end, int64_t nsteps, double* psi,
                                double tol, int32_t* iters_out, int64_t iters_cap) {
  const double tau = (t_end - t0) / (double)nsteps;
  const int per = exponentials_per_step(scheme);
  for (int64_t s = 0; s < nsteps; ++s) {
    oracle_expmv_info infos[3];
    int rc = oracle_magnus_step_csr(n, rp0, ci0, v0, rp1, ci1, v1, f, user, scheme, t0 + (double)s * tau, tau,
                                    psi, tol, infos);
    if (rc) return rc;
    for (int e = 0; e < per; ++e)
      if (iters_out && s * per + e < iters_cap) iters_out[s * per + e] = infos[e].iters;
  }
  return 0;
}

}  // extern "C"
