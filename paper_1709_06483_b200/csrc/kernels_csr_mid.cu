// S5-S8 for MEDIUM CSR problems (kSmallSweepMaxN < n <= kMidSweepMaxN, e.g. the paper's Example 2 at 2^13, 2^14 and
// spin chains of 13 to 17 sites): one persistent cooperative launch runs the exponentials of a planned batch
// (SweepJob list) back to back -- init, the fused Leja iterations with the stop test after each, finish -- separated
// by grid barriers instead of kernel boundaries.  At these sizes the matrix (a few MB to tens of MB) lives in L2 and an
// iteration is a few microseconds, so one launch per iteration plus a host poll every few iterations (the large
// path) is bound by launch latency.
//   w_0 = v, p_0 = d_0 v;  w_k = (1/gamma) M w_{k-1} - (c/gamma + l_{k-1}) w_{k-1};  p_k += d_k w_k   (c5)
//   stop at the first k >= 1 with |d_k| ||w_k|| + |d_{k-1}| ||w_{k-1}|| <= tol ||p_k||               (c6)
//   out = e^{-i h c} p_k                                                                              (c7)
// Layout: one CTA per SM; CTA b owns the contiguous rows [b per, (b+1) per).  M = sum_t coef_t A_t is formed on the
// fly from the CSR terms (coefficients from the job).  w lives in a global ping-pong buffer: a CTA writes its rows of
// the new w (L2), passes ONE grid barrier and gathers from the whole w with L2 loads (other CTAs wrote it, so L1 is
// bypassed); p of the CTA's rows stays in global memory too (only its owner touches it).  MS_G lanes share a row.
// The per-CTA partial norms go through global memory; every CTA adds all of them in the same order and takes the
// same stop decision.  Deterministic: fixed lane -> entry map, fixed trees, no floating-point atomics.
#include "magnus_internal.h"
#include "device_utils.cuh"

namespace magnus {

namespace {

constexpr int MS_THREADS = 512;
constexpr int MS_WARPS = MS_THREADS / 32;
constexpr int MS_G = 8;                          // lanes per row
constexpr int MS_GROUPS = MS_THREADS / MS_G;

__device__ __forceinline__ cplx ldcg_c(const cplx* p) { return __ldcg(reinterpret_cast<const double2*>(p)); }

__global__ void __launch_bounds__(MS_THREADS, 1)
    csr_leja_sweep_mid_kernel(CsrOp op, cplx* psi, const SweepJob* __restrict__ jobs, int njobs,
                              const double* __restrict__ leja_l, double tol, LejaStatus* status, const LejaStatus* gate,
                              cplx* wg0, cplx* wg1, cplx* pbuf, double* partials, unsigned* bar) {
  __shared__ double s_l[kMaxDegree + 1];           // Leja points (c2)
  __shared__ double s_absd[kMaxDegree + 1];        // |d_k| of the current job
  __shared__ double s_red[2][MS_WARPS];
  __shared__ double s_sum[2];
  if (gate && !gate->done) return;                 // an earlier job of the plan failed (grid-uniform)
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, grp = tid / MS_G, sub = tid % MS_G;
  const int n = (int)op.n;
  const int per = (n + (int)gridDim.x - 1) / (int)gridDim.x;
  const int r0 = min(n, (int)blockIdx.x * per), r1 = min(n, r0 + per);
  cplx* wg[2] = {wg0, wg1};
  unsigned generation = 0;
  for (int k = tid; k <= kMaxDegree; k += MS_THREADS) s_l[k] = leja_l[k];

  // this CTA's (a, b) -> the grid's sum, the same value in every thread of every CTA (fixed order).
  // The two partials buffers alternate on a counter that runs over ALL calls of the launch (not on the iteration
  // number): a CTA writes its slot for call c+1 into the buffer call c did not use, and reaches call c+2's write
  // into call c's buffer only behind barrier c+1, which no CTA passes before it has finished reading for call c.
  // Keyed on k & 1 instead, a job that stopped at an even k and the next job's init (call "0") shared a buffer with
  // no barrier in between: a fast CTA could overwrite its slot while a slow one was still summing the stop test.
  unsigned nsum = 0;
  auto grid_sum2 = [&](double a, double b, double& ta, double& tb) {
    const int parity = (int)(nsum++ & 1u);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      a += shfl_xor_d(a, o);
      b += shfl_xor_d(b, o);
    }
    if (lane == 0) {
      s_red[0][warp] = a;
      s_red[1][warp] = b;
    }
    __syncthreads();
    if (tid == 0) {
      double x = 0.0, y = 0.0;
#pragma unroll
      for (int w = 0; w < MS_WARPS; ++w) {
        x += s_red[0][w];
        y += s_red[1][w];
      }
      double* q = partials + (size_t)parity * 2 * gridDim.x + 2 * blockIdx.x;
      __stcg(q, x);
      __stcg(q + 1, y);
    }
    grid_barrier(bar, generation);                 // also publishes what the CTAs wrote to w before the call
    if (warp == 0) {
      double x = 0.0, y = 0.0;
      const double* q = partials + (size_t)parity * 2 * gridDim.x;
      for (int c = lane; c < (int)gridDim.x; c += 32) {
        x += __ldcg(q + 2 * c);
        y += __ldcg(q + 2 * c + 1);
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        x += shfl_xor_d(x, o);
        y += shfl_xor_d(y, o);
      }
      if (lane == 0) {
        s_sum[0] = x;
        s_sum[1] = y;
      }
    }
    __syncthreads();
    ta = s_sum[0];
    tb = s_sum[1];
  };

#pragma unroll 1
  for (int e = 0; e < njobs; ++e) {
    const SweepJob& J = jobs[e];
    const int m_max = J.m_max, nterms = min(J.nterms, op.nterms);
    const double inv_gamma = J.inv_gamma, c_over_gamma = J.c_over_gamma;
    cplx coef[3];
#pragma unroll
    for (int t = 0; t < 3; ++t) coef[t] = J.coef[t];
    __syncthreads();                               // the previous job's reads of s_absd are over
    for (int k = tid; k <= m_max; k += MS_THREADS) s_absd[k] = hypot(J.d[k].x, J.d[k].y);
    // S5: w_0 = psi, p_0 = d_0 psi on the CTA's rows; ||psi||^2 over the grid
    const cplx d0 = J.d[0];
    double a0 = 0.0;
    for (int r = r0 + tid; r < r1; r += MS_THREADS) {
      const cplx x = ldcg_c(psi + r);
      __stcg(reinterpret_cast<double2*>(wg[0] + r), x);
      pbuf[r] = cmul(d0, x);
      a0 += x.x * x.x + x.y * x.y;
    }
    double s0, dummy;
    grid_sum2(a0, 0.0, s0, dummy);
    double e_prev = s_absd[0] * sqrt(s0);
    double err = 0.0, sw = 0.0, sp = 0.0;
    int k = 0, cur = 0;
    bool done = false;

    while (!done && k < m_max) {
      ++k;
      const cplx dk = J.d[k];
      const double shift = c_over_gamma + s_l[k - 1];
      const cplx* w_in = wg[cur];
      cplx* w_out = wg[cur ^ 1];
      double bw = 0.0, bp = 0.0;
#pragma unroll 1
      for (int rb = r0; rb < r1; rb += MS_GROUPS) {          // S6 on the CTA's rows
        const int row = rb + grp;
        const bool valid = row < r1;
        cplx y = make_double2(0.0, 0.0);
        for (int t = 0; t < nterms; ++t) {
          const CsrTerm& T = op.t[t];
          cplx a = make_double2(0.0, 0.0);
          if (valid) {
            const int qe = T.rp[row + 1];
            for (int q = T.rp[row] + sub; q < qe; q += MS_G) cfma(a, T.v[q], ldcg_c(w_in + T.ci[q]));
          }
          const cplx ca = cmul(coef[t], a);
          y.x += ca.x;
          y.y += ca.y;
        }
#pragma unroll
        for (int o = MS_G / 2; o > 0; o >>= 1) {
          y.x += shfl_xor_d(y.x, o);
          y.y += shfl_xor_d(y.y, o);
        }
        if (valid && sub == 0) {
          const cplx wi = ldcg_c(w_in + row);
          cplx wn;
          wn.x = inv_gamma * y.x - shift * wi.x;
          wn.y = inv_gamma * y.y - shift * wi.y;
          cplx pi = pbuf[row];
          cfma(pi, dk, wn);
          pbuf[row] = pi;
          bw += wn.x * wn.x + wn.y * wn.y;
          bp += pi.x * pi.x + pi.y * pi.y;
          __stcg(reinterpret_cast<double2*>(w_out + row), wn);
        }
      }
      grid_sum2(bw, bp, sw, sp);                   // S7: one barrier per iteration
      const double e_k = s_absd[k] * sqrt(sw);
      err = e_k + e_prev;
      e_prev = e_k;
      done = err <= tol * sqrt(sp);
      cur ^= 1;
    }
    if (blockIdx.x == 0 && tid == 0) {
      LejaStatus* S = status + e;
      S->done = done ? 1 : 0;
      S->pad = done ? 0 : 1;
      S->k = k;
      S->iters += k;
      S->err_est = err;
      S->e_prev = e_prev;
      S->norm_w2 = sw;
      S->norm_p2 = sp;
    }
    if (!done) break;                              // grid-uniform: psi is the state before this job
    const cplx phase = J.phase;                    // S8 (the next job reads only this CTA's rows of psi: no barrier)
    for (int r = r0 + tid; r < r1; r += MS_THREADS) __stcg(reinterpret_cast<double2*>(psi + r), cmul(phase, pbuf[r]));
    __syncthreads();
  }
}

}  // namespace

bool csr_mid_sweep_supported(int64_t n, int csr_kernel) {
  if (csr_kernel == 7) return n <= kMidSweepMaxN;
  return csr_kernel == 0 && n > kMidSweepMinN && n <= kMidSweepMaxN;
}

// jobs[0..njobs) applied to psi in order, one cooperative launch; protocol of launch_csr_leja_sweep_small_jobs
int launch_csr_leja_sweep_mid_jobs(const CsrOp& op, cplx* psi, const SweepJob* jobs, int njobs, double tol,
                                   LejaStatus* status, const LejaStatus* gate, Workspace* ws, cudaStream_t st) {
  if (ensure_sweep_jobs(ws, st) != MAGNUS_OK) return MAGNUS_ENOMEM;
  if (cudaMemsetAsync(ws->grid_bar, 0, sizeof(unsigned), st) != cudaSuccess) return MAGNUS_ECUDA;
  CsrOp opv = op;
  const double* leja_l = ws->leja_l;
  cplx* wg0 = ws->w[0];
  cplx* wg1 = ws->w[1];
  cplx* pbuf = ws->p;
  double* partials = ws->sweep_partials;
  unsigned* bar = ws->grid_bar;
  void* args[] = {&opv, &psi, &jobs, &njobs, &leja_l, &tol, &status, &gate, &wg0, &wg1, &pbuf, &partials, &bar};
  if (cudaLaunchCooperativeKernel((const void*)csr_leja_sweep_mid_kernel, dim3(device_sm_count()), dim3(MS_THREADS), args, 0,
                                  st) != cudaSuccess)
    return MAGNUS_ECUDA;
  ws->launches += 1;
  return MAGNUS_OK;
}

// one sweep (leja_expmv, sub-steps, the fall-back after a failed batch): a one-job batch through job slot 0
int launch_csr_leja_sweep_mid(const CsrOp& op, const cplx* v, cplx* out, double inv_gamma, double c_over_gamma, double tol,
                              int m_max, cplx phase, const SweepTable& tab, Workspace* ws, cudaStream_t st) {
  if (ensure_sweep_jobs(ws, st) != MAGNUS_OK) return MAGNUS_ENOMEM;
  SweepJob& J = ws->jobs_host[0];
  for (int t = 0; t < 3; ++t) J.coef[t] = op.t[t].coef;
  J.phase = phase;
  J.inv_gamma = inv_gamma;
  J.c_over_gamma = c_over_gamma;
  J.m_max = m_max;
  J.nterms = op.nterms;
  J.flags = 0;
  J.pad = 0;
  for (int k = 0; k <= m_max; ++k) J.d[k] = tab.d[k];
  if (cudaMemcpyAsync(ws->jobs, &J, sizeof(SweepJob), cudaMemcpyHostToDevice, st) != cudaSuccess) return MAGNUS_ECUDA;
  if (out != v && cudaMemcpyAsync(out, v, sizeof(cplx) * (size_t)op.n, cudaMemcpyDeviceToDevice, st) != cudaSuccess)
    return MAGNUS_ECUDA;
  return launch_csr_leja_sweep_mid_jobs(op, out, ws->jobs, 1, tol, ws->status, nullptr, ws, st);
}

}  // namespace magnus
