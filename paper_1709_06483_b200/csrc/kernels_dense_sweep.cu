// S2, S5-S8 for MEDIUM dense problems (n <= kDenseSweepMaxN, e.g. CFG2: n = 2048, 67 MB per matrix):
// one persistent cooperative launch runs the exponentials of a planned batch (SweepJob list) back to
// back -- assembly of M = H0 + g H1, init, the fused Leja iterations with the stop test after each,
// finish -- separated by grid barriers instead of kernel boundaries.  At this size the assembled matrix
// stays in the 126 MB L2 and an iteration is a few microseconds of L2 traffic, so the per-iteration
// kernels of the large path are bound by launch latency and by their one-warp-per-row tail.
//   w_0 = v, p_0 = d_0 v;  w_k = (1/gamma) M w_{k-1} - (c/gamma + l_{k-1}) w_{k-1};  p_k += d_k w_k   (c5)
//   stop at the first k >= 1 with |d_k| ||w_k|| + |d_{k-1}| ||w_{k-1}|| <= tol ||p_k||               (c6)
//   out = e^{-i h c} p_k                                                                              (c7)
// Layout: one CTA per SM; CTA b owns the contiguous rows [b per, (b+1) per), per = ceil(n / grid) <= 32.
// The rows of M a CTA reads are the rows it assembled itself, so the assembly needs no barrier; only w
// crosses CTAs: every CTA writes its rows of the new w to a global ping-pong buffer, passes ONE grid
// barrier and reads the whole w (16 n bytes, from L2) into shared memory.  Inside a CTA thread t owns the
// columns t, t + 512, ...: the row loop streams M with coalesced 128-bit loads, many rows in flight, and
// the per-row sums are reduced by shuffles and one shared-memory pass.  The per-CTA partial norms go the
// same way; every CTA adds all of them in the same order and takes the same stop decision.
// Deterministic: fixed thread -> entry map, fixed trees, no floating-point atomics.
#include "magnus_internal.h"
#include "device_utils.cuh"

namespace magnus {

namespace {

constexpr int DS_THREADS = 512;
constexpr int DS_WARPS = DS_THREADS / 32;
constexpr int DS_MAX_ROWS = 32;                 // rows per CTA
constexpr int DS_RG = 7;                        // rows in flight together
constexpr int DS_SMEM = kDenseSweepMaxN * (int)sizeof(cplx);   // the vector w

__device__ __forceinline__ cplx ldcg_cplx(const cplx* p) {
  const double2 v = __ldcg(reinterpret_cast<const double2*>(p));
  return v;
}

__global__ void __launch_bounds__(DS_THREADS, 1)
    dense_leja_sweep_kernel(int n, const cplx* __restrict__ H0, int64_t ld0, const cplx* __restrict__ H1, int64_t ld1,
                            cplx* M, cplx* psi, const SweepJob* __restrict__ jobs, int njobs,
                            const double* __restrict__ leja_l, double tol, LejaStatus* status, const LejaStatus* gate,
                            cplx* wg0, cplx* wg1, double* partials, unsigned* bar) {
  extern __shared__ __align__(16) unsigned char ds_smem[];
  __shared__ cplx red[DS_WARPS][DS_MAX_ROWS];      // per-warp partial row sums
  __shared__ cplx prow[DS_MAX_ROWS];               // p of the CTA's rows
  __shared__ double s_l[kMaxDegree + 1];           // Leja points (c2)
  __shared__ double s_red[2][DS_WARPS];
  __shared__ double s_sum[2];
  if (gate && !gate->done) return;                 // an earlier job of the plan failed (grid-uniform)
  cplx* wsm = reinterpret_cast<cplx*>(ds_smem);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int per = (n + (int)gridDim.x - 1) / (int)gridDim.x;
  const int r0 = min(n, (int)blockIdx.x * per), r1 = min(n, r0 + per), nrows = r1 - r0;
  cplx* wg[2] = {wg0, wg1};
  unsigned generation = 0;
  for (int k = tid; k <= kMaxDegree; k += DS_THREADS) s_l[k] = leja_l[k];

  // sum over the block of (a, b), the same value in every thread; fixed tree
  auto block_sum2 = [&](double& a, double& b) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      a += shfl_xor_d(a, o);
      b += shfl_xor_d(b, o);
    }
    __syncthreads();
    if (lane == 0) {
      s_red[0][warp] = a;
      s_red[1][warp] = b;
    }
    __syncthreads();
    a = 0.0;
    b = 0.0;
#pragma unroll
    for (int w = 0; w < DS_WARPS; ++w) {
      a += s_red[0][w];
      b += s_red[1][w];
    }
  };

#pragma unroll 1
  for (int e = 0; e < njobs; ++e) {
    const SweepJob& J = jobs[e];
    const int m_max = J.m_max;
    const double inv_gamma = J.inv_gamma, c_over_gamma = J.c_over_gamma;
    // S2: the CTA's rows of M = H0 + g H1; they are read by this CTA only
    if (!(J.flags & kSweepJobAssembled)) {
      const double g = J.coef[1].x;
      for (int r = r0; r < r1; ++r) {
        const cplx* a = H0 + (int64_t)r * ld0;
        const cplx* b = H1 + (int64_t)r * ld1;
        cplx* m = M + (int64_t)r * n;
        for (int j = tid; j < n; j += DS_THREADS) {
          const cplx x = ld_gather_na(a + j), y = ld_gather_na(b + j);
          __stcg(reinterpret_cast<double2*>(m + j), make_double2(fma(g, y.x, x.x), fma(g, y.y, x.y)));
        }
      }
    }
    // S5: every CTA reads the whole psi (fixed-order norm, identical in all CTAs); p_0 for its own rows
    double s0 = 0.0, s1 = 0.0;
    for (int j = tid; j < n; j += DS_THREADS) {
      const cplx x = ldcg_cplx(psi + j);
      wsm[j] = x;
      s0 += x.x * x.x + x.y * x.y;
    }
    block_sum2(s0, s1);                              // also orders the wsm writes before the reads below
    const cplx d0 = J.d[0];
    if (tid < nrows) prow[tid] = cmul(d0, wsm[r0 + tid]);
    double e_prev = hypot(d0.x, d0.y) * sqrt(s0);
    double err = 0.0, sw = 0.0, sp = 0.0;
    int k = 0;
    bool done = false;
    __syncthreads();                                 // M rows written above are visible to the whole CTA

    while (!done && k < m_max) {
      ++k;
      const cplx dk = J.d[k];
      const double shift = c_over_gamma + s_l[k - 1];
      // S6 on the CTA's rows: thread t owns columns t, t + 512, ...
#pragma unroll 1
      for (int rg = 0; rg < nrows; rg += DS_RG) {
        cplx acc[DS_RG];
#pragma unroll
        for (int r = 0; r < DS_RG; ++r) acc[r] = make_double2(0.0, 0.0);
        const cplx* mrow = M + (int64_t)(r0 + rg) * n;
#pragma unroll 2
        for (int j = tid; j < n; j += DS_THREADS) {
          const cplx x = wsm[j];
          cplx mv[DS_RG];
#pragma unroll
          for (int r = 0; r < DS_RG; ++r)
            mv[r] = rg + r < nrows ? ldcg_cplx(mrow + (int64_t)r * n + j) : make_double2(0.0, 0.0);
#pragma unroll
          for (int r = 0; r < DS_RG; ++r) cfma(acc[r], mv[r], x);
        }
#pragma unroll
        for (int r = 0; r < DS_RG; ++r) {
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) {
            acc[r].x += shfl_xor_d(acc[r].x, o);
            acc[r].y += shfl_xor_d(acc[r].y, o);
          }
          if (lane == 0 && rg + r < nrows) red[warp][rg + r] = acc[r];
        }
      }
      __syncthreads();
      double bw = 0.0, bp = 0.0;
      if (tid < nrows) {                             // warp 0 (nrows <= 32): finish the rows
        cplx y = make_double2(0.0, 0.0);
#pragma unroll
        for (int w = 0; w < DS_WARPS; ++w) {
          y.x += red[w][tid].x;
          y.y += red[w][tid].y;
        }
        const cplx wi = wsm[r0 + tid];
        cplx wn;
        wn.x = inv_gamma * y.x - shift * wi.x;
        wn.y = inv_gamma * y.y - shift * wi.y;
        cplx pi = prow[tid];
        cfma(pi, dk, wn);
        prow[tid] = pi;
        bw = wn.x * wn.x + wn.y * wn.y;
        bp = pi.x * pi.x + pi.y * pi.y;
        __stcg(reinterpret_cast<double2*>(wg[k & 1] + r0 + tid), wn);
      }
      if (warp == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          bw += shfl_down_d(bw, o);
          bp += shfl_down_d(bp, o);
        }
        if (lane == 0) {
          double* q = partials + (size_t)(k & 1) * 2 * gridDim.x + 2 * blockIdx.x;
          __stcg(q, bw);
          __stcg(q + 1, bp);
        }
      }
      grid_barrier(bar, generation);                 // every CTA's rows of the new w and its partials are written
      for (int j = tid; j < n; j += DS_THREADS) wsm[j] = ldcg_cplx(wg[k & 1] + j);
      if (warp == 0) {                               // S7: all partials in a fixed order, the same in every CTA
        double a = 0.0, b = 0.0;
        const double* q = partials + (size_t)(k & 1) * 2 * gridDim.x;
        for (int c = lane; c < (int)gridDim.x; c += 32) {
          a += __ldcg(q + 2 * c);
          b += __ldcg(q + 2 * c + 1);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          a += shfl_xor_d(a, o);
          b += shfl_xor_d(b, o);
        }
        if (lane == 0) {
          s_sum[0] = a;
          s_sum[1] = b;
        }
      }
      __syncthreads();
      sw = s_sum[0];
      sp = s_sum[1];
      const double e_k = hypot(dk.x, dk.y) * sqrt(sw);
      err = e_k + e_prev;
      e_prev = e_k;
      done = err <= tol * sqrt(sp);
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
    if (!done) break;                                // grid-uniform: psi is the state before this job
    const cplx phase = J.phase;                      // S8
    if (tid < nrows) __stcg(reinterpret_cast<double2*>(psi + r0 + tid), cmul(phase, prow[tid]));
    if (e + 1 < njobs) grid_barrier(bar, generation);   // the next job reads the whole psi
  }
}

}  // namespace

bool dense_sweep_supported(int64_t n) {
  return n <= kDenseSweepMaxN && (n + device_sm_count() - 1) / device_sm_count() <= DS_MAX_ROWS;
}

// jobs[0..njobs) applied to psi in order, one cooperative launch; see launch_csr_leja_sweep_small_jobs for the protocol.
// H0, H1 may be null when every job carries kSweepJobAssembled (M is then the operator itself).
int launch_dense_leja_sweep_jobs(int64_t n, const cplx* H0, int64_t ld0, const cplx* H1, int64_t ld1, cplx* M, cplx* psi,
                                 const SweepJob* jobs, int njobs, double tol, LejaStatus* status, const LejaStatus* gate,
                                 Workspace* ws, cudaStream_t st) {
  if (ensure_sweep_jobs(ws, st) != MAGNUS_OK) return MAGNUS_ENOMEM;
  if (cudaFuncSetAttribute(dense_leja_sweep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, DS_SMEM) != cudaSuccess)
    return MAGNUS_ECUDA;
  if (cudaMemsetAsync(ws->grid_bar, 0, sizeof(unsigned), st) != cudaSuccess) return MAGNUS_ECUDA;
  int ni = (int)n;
  const double* leja_l = ws->leja_l;
  cplx* wg0 = ws->w[0];
  cplx* wg1 = ws->w[1];
  double* partials = ws->sweep_partials;
  unsigned* bar = ws->grid_bar;
  void* args[] = {&ni, &H0, &ld0, &H1, &ld1, &M, &psi, &jobs, &njobs, &leja_l, &tol, &status, &gate,
                  &wg0, &wg1, &partials, &bar};
  const int grid = device_sm_count();
  if (cudaLaunchCooperativeKernel((const void*)dense_leja_sweep_kernel, dim3(grid), dim3(DS_THREADS), args, DS_SMEM, st) !=
      cudaSuccess)
    return MAGNUS_ECUDA;
  ws->launches += 1;
  return MAGNUS_OK;
}

// one sweep on an assembled matrix (leja_expmv, M4 / M6 steps, sub-steps, the fall-back after a failed batch): a
// one-job batch through job slot 0.  out != v: v is copied first (the kernel works in place); a sweep that does
// not converge leaves out as that copy.
int launch_dense_leja_sweep(const DenseOp& op, const cplx* v, cplx* out, double inv_gamma, double c_over_gamma,
                            double tol, int m_max, cplx phase, const SweepTable& tab, Workspace* ws, cudaStream_t st) {
  if (ensure_sweep_jobs(ws, st) != MAGNUS_OK) return MAGNUS_ENOMEM;
  SweepJob& J = ws->jobs_host[0];
  J.coef[0] = J.coef[1] = J.coef[2] = make_double2(0.0, 0.0);
  J.phase = phase;
  J.inv_gamma = inv_gamma;
  J.c_over_gamma = c_over_gamma;
  J.m_max = m_max;
  J.nterms = 1;
  J.flags = kSweepJobAssembled;
  J.pad = 0;
  for (int k = 0; k <= m_max; ++k) J.d[k] = tab.d[k];
  if (cudaMemcpyAsync(ws->jobs, &J, sizeof(SweepJob), cudaMemcpyHostToDevice, st) != cudaSuccess) return MAGNUS_ECUDA;
  if (out != v &&
      cudaMemcpyAsync(out, v, sizeof(cplx) * (size_t)op.n, cudaMemcpyDeviceToDevice, st) != cudaSuccess)
    return MAGNUS_ECUDA;
  return launch_dense_leja_sweep_jobs(op.n, nullptr, 0, nullptr, 0, const_cast<cplx*>(op.M), out, ws->jobs, 1, tol,
                                      ws->status, nullptr, ws, st);
}

}  // namespace magnus
