// S5-S8 in ONE launch for small CSR problems (n <= kSmallSweepMaxN, e.g. CFG1: n = 1024,
// 0.33 MB of matrix, resident in L1/L2): one CTA of 1024 threads runs a whole Leja sweep of a
// sub-step -- init, the fused iterations with the stop test after each, finish -- separated
// by __syncthreads() instead of kernel boundaries.  At this size a launch (a few microseconds)
// costs more than an iteration, so the per-iteration kernels of the large path are launch bound.
//   w_0 = v, p_0 = d_0 v;  w_k = (1/gamma) M w_{k-1} - (c/gamma + l_{k-1}) w_{k-1};  p_k += d_k w_k   (c5)
//   stop at the first k >= 1 with |d_k| ||w_k|| + |d_{k-1}| ||w_{k-1}|| <= tol ||p_k||               (c6)
//   out = e^{-i (h/s) c} p_k                                                                          (c7)
// The divided differences and Leja points arrive as a kernel argument (3 KB, __grid_constant__).
// Thread t owns rows t, t + 1024, ...; its p entries stay in registers, w ping-pongs through
// global memory (L1/L2) because every row gathers other rows' previous w.  Deterministic: sequential
// sum along a row, fixed block-reduction tree.
#include "magnus_internal.h"
#include "device_utils.cuh"

namespace magnus {

namespace {

constexpr int SS_THREADS = 1024;
constexpr int SS_ROWS = kSmallSweepMaxN / SS_THREADS;   // rows per thread
constexpr int SS_U = 6;                                 // entries in flight per thread

// Sum of (a, b) over the block, result in EVERY thread.  Fixed tree.
__device__ __forceinline__ void block_allreduce_sum2(double& a, double& b, double* sa, double* sb) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += shfl_xor_d(a, o);
    b += shfl_xor_d(b, o);
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  __syncthreads();            // previous use of sa/sb is over
  if (lane == 0) {
    sa[warp] = a;
    sb[warp] = b;
  }
  __syncthreads();
  a = sa[lane];               // SS_THREADS / 32 == 32 warps: one value per lane
  b = sb[lane];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += shfl_xor_d(a, o);
    b += shfl_xor_d(b, o);
  }
}

__global__ void __launch_bounds__(SS_THREADS, 1)
    csr_leja_sweep_small_kernel(CsrOp op, const cplx* v, cplx* w0, cplx* w1, cplx* out, double inv_gamma,
                                double c_over_gamma, double tol, int m_max, cplx phase,
                                const __grid_constant__ SweepTable tab, LejaStatus* status) {
  static_assert(SS_THREADS == 1024, "the all-reduce assumes 32 warps");
  __shared__ double sa[32], sb[32];
  if (status->pad) return;                 // an earlier sub-step did not converge
  const int tid = threadIdx.x;
  const int n = (int)op.n;
  cplx pr[SS_ROWS];
  double s0 = 0.0, s1 = 0.0;
#pragma unroll
  for (int j = 0; j < SS_ROWS; ++j) {      // S5
    const int row = tid + j * SS_THREADS;
    pr[j] = make_double2(0.0, 0.0);
    if (row < n) {
      const cplx x = v[row];
      w0[row] = x;
      pr[j] = cmul(tab.d[0], x);
      s0 += x.x * x.x + x.y * x.y;
    }
  }
  block_allreduce_sum2(s0, s1, sa, sb);
  double e_prev = hypot(tab.d[0].x, tab.d[0].y) * sqrt(s0);
  double err = 0.0, sw = 0.0, sp = 0.0;
  cplx* w_in = w0;
  cplx* w_out = w1;
  int k = 0;
  bool done = false;
  while (!done && k < m_max) {
    ++k;
    __syncthreads();                       // w_in complete (block-wide visibility of the global stores)
    const cplx dk = tab.d[k];
    const double shift = c_over_gamma + tab.l[k - 1];
    sw = 0.0;
    sp = 0.0;
#pragma unroll
    for (int j = 0; j < SS_ROWS; ++j) {    // S6
      const int row = tid + j * SS_THREADS;
      if (row < n) {
        cplx y = make_double2(0.0, 0.0);
        for (int t = 0; t < op.nterms; ++t) {
          const CsrTerm& T = op.t[t];
          cplx a = make_double2(0.0, 0.0);
          const int qs = T.rp[row], qe = T.rp[row + 1];
          // batches of SS_U entries: all column loads, then all value / w loads, then the FMAs in stored
          // order -- two dependent memory latencies per batch instead of per entry
          for (int q0 = qs; q0 < qe; q0 += SS_U) {
            int c[SS_U];
            cplx mv[SS_U], xv[SS_U];
#pragma unroll
            for (int u = 0; u < SS_U; ++u) c[u] = q0 + u < qe ? T.ci[q0 + u] : row;
#pragma unroll
            for (int u = 0; u < SS_U; ++u) {
              mv[u] = q0 + u < qe ? T.v[q0 + u] : make_double2(0.0, 0.0);
              xv[u] = w_in[c[u]];
            }
#pragma unroll
            for (int u = 0; u < SS_U; ++u) cfma(a, mv[u], xv[u]);
          }
          const cplx ca = cmul(T.coef, a);
          y.x += ca.x;
          y.y += ca.y;
        }
        const cplx wi = w_in[row];
        cplx wn;
        wn.x = inv_gamma * y.x - shift * wi.x;
        wn.y = inv_gamma * y.y - shift * wi.y;
        w_out[row] = wn;
        cfma(pr[j], dk, wn);
        sw += wn.x * wn.x + wn.y * wn.y;
        sp += pr[j].x * pr[j].x + pr[j].y * pr[j].y;
      }
    }
    block_allreduce_sum2(sw, sp, sa, sb);
    const double e_k = hypot(dk.x, dk.y) * sqrt(sw);   // S7
    err = e_k + e_prev;
    e_prev = e_k;
    done = err <= tol * sqrt(sp);
    cplx* tmp = w_in;
    w_in = w_out;
    w_out = tmp;
  }
  if (done) {
#pragma unroll
    for (int j = 0; j < SS_ROWS; ++j) {    // S8
      const int row = tid + j * SS_THREADS;
      if (row < n) out[row] = cmul(phase, pr[j]);
    }
  }
  if (tid == 0) {
    status->done = done ? 1 : 0;
    status->pad = done ? 0 : 1;
    status->k = k;
    status->iters += k;
    status->err_est = err;
    status->e_prev = e_prev;
    status->norm_w2 = sw;
    status->norm_p2 = sp;
  }
}

}  // namespace

void launch_csr_leja_sweep_small(const CsrOp& op, const cplx* v, cplx* out, double inv_gamma, double c_over_gamma,
                                 double tol, int m_max, cplx phase, const SweepTable& tab, Workspace* ws,
                                 cudaStream_t st) {
  csr_leja_sweep_small_kernel<<<1, SS_THREADS, 0, st>>>(op, v, ws->w[0], ws->w[1], out, inv_gamma, c_over_gamma, tol,
                                                        m_max, phase, tab, ws->status);
  ws->launches += 1;
}

}  // namespace magnus
