// Host-side pieces of the Leja/Magnus path (row S1 and S4 of the scope table):
// Leja points, divided differences, interval snapping, scheme scalars.
// Plain C++; no CUDA in this file.  Nothing here is shared with oracle/.
//
// P:n = PAPER.md line n; c1..c7 = readings in DESIGN.md section 3.
#include "magnus_internal.h"

#include <algorithm>
#include <cmath>
#include <complex>
#include <mutex>
#include <vector>

namespace magnus {

// ---------------------------------------------------------------------------
// Leja points of [-2, 2] ("Leja points (see [11])"; reading c2):
//   l0 = 2, l1 = -2, l2 = 0, l3 = +2/sqrt(3); l_k maximises prod_{j<k} |x - l_j|.
// Between two neighbouring nodes log prod |x - l_j| is strictly concave, so the
// maximiser of that gap is the only root of g(x) = sum_j 1/(x - l_j) there.  The
// root is bracketed by the gap and found by Newton steps that fall back to
// bisection whenever they would leave the bracket (long double throughout).
// ---------------------------------------------------------------------------
static long double gap_stationary_point(const std::vector<long double>& nodes, long double lo, long double hi) {
  long double a = lo, b = hi;            // g(a+) = +inf, g(b-) = -inf, g decreasing
  long double x = 0.5L * (a + b);
  for (int it = 0; it < 200; ++it) {
    long double g = 0.0L, dg = 0.0L;
    for (long double t : nodes) {
      const long double r = 1.0L / (x - t);
      g += r;
      dg -= r * r;
    }
    if (g > 0.0L) a = x; else b = x;
    long double xn = x - g / dg;
    if (!(xn > a && xn < b)) xn = 0.5L * (a + b);
    if (xn == x || b - a <= 0.0L) break;
    if (fabsl(xn - x) <= 1e-20L * (1.0L + fabsl(x))) { x = xn; break; }
    x = xn;
  }
  return x;
}

static std::vector<double> compute_leja_points(int m) {
  std::vector<double> pts;
  const double head[4] = {2.0, -2.0, 0.0, 2.0 / std::sqrt(3.0)};
  for (int k = 0; k < m && k < 4; ++k) pts.push_back(head[k]);
  std::vector<long double> sorted;
  while ((int)pts.size() < m) {
    sorted.assign(pts.begin(), pts.end());
    std::sort(sorted.begin(), sorted.end());
    long double best_log = -INFINITY, best_x = 0.0L;
    for (size_t g = 0; g + 1 < sorted.size(); ++g) {
      const long double x = gap_stationary_point(sorted, sorted[g], sorted[g + 1]);
      long double lg = 0.0L;
      for (long double t : sorted) lg += logl(fabsl(x - t));
      if (lg > best_log) { best_log = lg; best_x = x; }
    }
    pts.push_back((double)best_x);
  }
  return pts;
}

const double* leja_points() {
  static std::vector<double> table;
  static std::once_flag once;
  std::call_once(once, [] { table = compute_leja_points(kMaxDegree + 1); });
  return table.data();
}

// ---------------------------------------------------------------------------
// Divided differences d_k = F[l_0..l_k], F(x) = exp(-i theta x)  (c3).
// Route: by Opitz' theorem the d_k are the first column of F(Z) for the lower
// bidiagonal Z = diag(l_0..l_m) + subdiag(1), i.e. d = exp(-i theta Z) e_1.  The
// exponential is applied as s = ceil(|theta|/0.25) Taylor sweeps of step
// theta/s; component k of (Z^j e_1) is zero for j < k, so m + 24 terms reach
// every component with full relative accuracy.  long double arithmetic.
// ---------------------------------------------------------------------------
void divided_differences(double theta, int m, std::complex<double>* out) {
  const double* l = leja_points();
  // real and imaginary parts in separate arrays (plain x87 multiplies and adds; no complex-multiply helper calls)
  std::vector<long double> vr(m, 0.0L), vi(m, 0.0L), tr(m), ti(m), ar(m), ai(m), ll(m);
  for (int k = 0; k < m; ++k) ll[k] = (long double)l[k];
  vr[0] = 1.0L;
  const int s = std::max(1, (int)std::ceil(std::fabs(theta) / 0.25));
  const long double tp = (long double)theta / (long double)s;
  const int nterms = m + 24;
  int top = 0;   // largest index with a nonzero entry in v: Z is lower bidiagonal, so a sweep's j-th term reaches top + j
  for (int sweep = 0; sweep < s; ++sweep) {
    tr = vr; ti = vi;
    ar = vr; ai = vi;
    for (int j = 1; j <= nterms; ++j) {
      // term <- (-i tp / j) Z term, with (Z x)_k = l_k x_k + x_{k-1}; entries above top + j are exactly zero
      const long double f = tp / (long double)j;
      const int kend = std::min(m - 1, top + j);
      long double pr = 0.0L, pi = 0.0L;
      for (int k = 0; k <= kend; ++k) {
        const long double cr = tr[k], ci = ti[k];
        const long double zr = ll[k] * cr + pr, zi = ll[k] * ci + pi;
        tr[k] = f * zi;            // (-i f) z
        ti[k] = -(f * zr);
        pr = cr;
        pi = ci;
        ar[k] += tr[k];
        ai[k] += ti[k];
      }
    }
    vr = ar; vi = ai;
    top = m - 1;   // after one sweep v is full
  }
  for (int k = 0; k < m; ++k) out[k] = std::complex<double>((double)vr[k], (double)vi[k]);
}

// Extreme eigenvalues of the symmetric tridiagonal T = tridiag(alpha_0..alpha_{k-1}; beta_0..beta_{k-2}) by bisection on
// the Sturm count (number of eigenvalues below x = number of negative pivots of T - xI); used by the tight-interval
// shortcut (kernels_lanczos.cu).  Accurate to a few ulps of ||T||.
static int sturm_count(const double* alpha, const double* beta, int k, double x) {
  int cnt = 0;
  double d = 1.0;
  for (int i = 0; i < k; ++i) {
    const double b2 = i > 0 ? beta[i - 1] * beta[i - 1] : 0.0;
    d = (alpha[i] - x) - (i > 0 ? b2 / d : 0.0);
    if (d == 0.0) d = -1e-300;          // a pivot of exactly 0 counts as negative (eigenvalue <= x)
    if (d < 0.0) ++cnt;
  }
  return cnt;
}

void tridiag_extreme_eigenvalues(const double* alpha, const double* beta, int k, double* lo_out, double* hi_out) {
  double lo = alpha[0], hi = alpha[0];
  for (int i = 0; i < k; ++i) {         // Gershgorin bounds of T bracket its spectrum
    const double r = (i > 0 ? std::fabs(beta[i - 1]) : 0.0) + (i + 1 < k ? std::fabs(beta[i]) : 0.0);
    lo = std::min(lo, alpha[i] - r);
    hi = std::max(hi, alpha[i] + r);
  }
  auto kth = [&](int want) {            // smallest x with count(x) >= want, i.e. the want-th eigenvalue
    double a = lo, b = hi;
    for (int it = 0; it < 200; ++it) {
      const double mid = 0.5 * (a + b);
      if (mid <= a || mid >= b) break;
      if (sturm_count(alpha, beta, k, mid) >= want) b = mid; else a = mid;
    }
    return 0.5 * (a + b);
  };
  *lo_out = kth(1);
  *hi_out = kth(k);
}

// Reading c4: widen [a,b] outward to the grid of spacing 2^(E-12), E = ceil(log2(b-a)).
void snap_interval(double* a, double* b) {
  const double width = *b - *a;
  if (!(width > 0.0) || !std::isfinite(width)) return;
  const int E = (int)std::ceil(std::log2(width));
  // log2 may be off by one ulp near exact powers of two: fix with exact comparisons
  int e = E;
  while (std::ldexp(1.0, e) < width) ++e;
  while (std::ldexp(1.0, e - 1) >= width) --e;
  const double delta = std::ldexp(1.0, e - 12);
  *a = std::floor(*a / delta) * delta;
  *b = std::ceil(*b / delta) * delta;
}

// ---------------------------------------------------------------------------
// Scheme scalars (row S1; reading c1).  With A = -iH and H(t) = H0 + f(t) H1 every
// exponential of a step is exp(-i h_e (H0 + g_e H1)), h_e = h_scale[e] * tau.
// ---------------------------------------------------------------------------
int step_coefficients(int scheme, magnus_drive_fn f, void* user, double t, double tau,
                      double* coef_h1, double* h_scale, double* kappa) {
  if (kappa) *kappa = 0.0;
  const double s3 = std::sqrt(3.0), s15 = std::sqrt(15.0);
  switch (scheme) {
    case MAGNUS_CF4: {   // exp(tau(a1 A1 + a2 A2)) exp(tau(a2 A1 + a1 A2)) Y; right factor first
      const double f1 = f(t + (0.5 - s3 / 6.0) * tau, user), f2 = f(t + (0.5 + s3 / 6.0) * tau, user);
      const double a1 = (3.0 - 2.0 * s3) / 12.0, a2 = (3.0 + 2.0 * s3) / 12.0;
      coef_h1[0] = 2.0 * (a2 * f1 + a1 * f2);
      coef_h1[1] = 2.0 * (a1 * f1 + a2 * f2);
      h_scale[0] = h_scale[1] = 0.5;
      return 2;
    }
    case MAGNUS_M4: {    // Omega_H = H0 + fbar H1 - i kappa [H0,H1], kappa = sqrt(3) tau/12 (f1-f2)
      const double f1 = f(t + (0.5 - s3 / 6.0) * tau, user), f2 = f(t + (0.5 + s3 / 6.0) * tau, user);
      coef_h1[0] = f1;   // the two node values; the step driver forms fbar and kappa
      coef_h1[1] = f2;
      h_scale[0] = 1.0;
      if (kappa) *kappa = (s3 * tau / 12.0) * (f1 - f2);
      return 1;
    }
    case MAGNUS_M2: {
      coef_h1[0] = f(t + 0.5 * tau, user);
      h_scale[0] = 1.0;
      return 1;
    }
    case MAGNUS_CF4_3: { // rows of alpha; Y <- E1 E2 E3 Y, so row 3 acts first
      const double fn[3] = {f(t + (0.5 - s15 / 10.0) * tau, user), f(t + 0.5 * tau, user),
                            f(t + (0.5 + s15 / 10.0) * tau, user)};
      const double p = 37.0 / 240.0, q = 10.0 * s15 / 261.0;
      const double al[3][3] = {{p - q, -1.0 / 30.0, p + q},
                               {-11.0 / 360.0, 23.0 / 45.0, -11.0 / 360.0},
                               {p + q, -1.0 / 30.0, p - q}};
      for (int e = 0; e < 3; ++e) {
        const double* row = al[2 - e];
        const double S = row[0] + row[1] + row[2];
        h_scale[e] = S;
        coef_h1[e] = (row[0] * fn[0] + row[1] * fn[1] + row[2] * fn[2]) / S;
      }
      return 3;
    }
    case MAGNUS_M6: {    // the three Gauss nodes; the step driver forms b2, b3 and the nested commutators
      coef_h1[0] = f(t + (0.5 - s15 / 10.0) * tau, user);
      coef_h1[1] = f(t + 0.5 * tau, user);
      coef_h1[2] = f(t + (0.5 + s15 / 10.0) * tau, user);
      h_scale[0] = 1.0;
      return 1;
    }
    default:
      return -1;
  }
}

}  // namespace magnus
