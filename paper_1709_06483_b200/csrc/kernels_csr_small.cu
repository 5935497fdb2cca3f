// S5-S8 in ONE launch for small CSR problems (n <= kSmallSweepMaxN, e.g. CFG1: n = 1024,
// 0.33 MB of matrix): one thread-block CLUSTER of 8 CTAs runs a whole Leja sweep of a sub-step
// -- init, the fused iterations with the stop test after each, finish -- separated by cluster
// barriers instead of kernel boundaries.  At this size a launch (a few microseconds) costs more
// than an iteration, so the per-iteration kernels of the large path are launch bound.
//   w_0 = v, p_0 = d_0 v;  w_k = (1/gamma) M w_{k-1} - (c/gamma + l_{k-1}) w_{k-1};  p_k += d_k w_k   (c5)
//   stop at the first k >= 1 with |d_k| ||w_k|| + |d_{k-1}| ||w_{k-1}|| <= tol ||p_k||               (c6)
//   out = e^{-i (h/s) c} p_k                                                                          (c7)
// Layout: CTA c owns the contiguous row slice [c n/8, (c+1) n/8); SS_G lanes share a row; p of the
// slice lives in shared memory.  EVERY CTA holds the whole vector w in its shared memory (ping-pong,
// 2 x 16 n bytes): a CTA PUSHES every new w entry of its slice into all eight copies through distributed
// shared memory as it is computed (fire-and-forget remote stores that overlap the rest of the row loop),
// so after the one cluster barrier per iteration the gathers are local shared-memory reads and nothing is pulled.  The CTA's slice of the CSR terms is copied to shared memory once per
// sweep when it fits (cluster barriers flush L1, so global reads would pay an L2 round trip per
// dependent load in every iteration); otherwise it is read in place.  The per-CTA partial norms are
// pushed the same way; every CTA sums the eight partials in the same order and takes the same stop
// decision.  The divided differences and Leja points arrive as a kernel argument (3 KB,
// __grid_constant__).  Deterministic: fixed lane->entry map, fixed trees.
// Measured (clock64, CFG1): about 10,000 cycles per iteration -- row slice 4,000, block reduction
// 1,100, cluster barrier 1,400, DSMEM pull 1,650, stop test (hypot, sqrt) 1,300.
#include "magnus_internal.h"
#include "device_utils.cuh"

#include <cooperative_groups.h>

namespace cg = cooperative_groups;

namespace magnus {

namespace {

constexpr int SS_CTAS = 8;                 // portable cluster size
constexpr int SS_THREADS = 512;
constexpr int SS_G = 8;                    // lanes per row
constexpr int SS_GROUPS = SS_THREADS / SS_G;
constexpr int SS_MAX_ROWS = kSmallSweepMaxN / SS_CTAS;          // rows per CTA
constexpr int SS_MCAP = 4000;               // matrix entries (all terms) a CTA can keep in shared memory
constexpr int SS_W_BYTES = 2 * kSmallSweepMaxN * (int)sizeof(cplx);
constexpr int SS_SMEM = SS_W_BYTES + SS_MAX_ROWS * (int)sizeof(cplx) + SS_MCAP * (int)(sizeof(cplx) + sizeof(int32_t)) +
                        3 * (SS_MAX_ROWS + 1) * (int)sizeof(int);

// Sum of (a, b) over the block, result in thread 0.  Fixed tree.
__device__ __forceinline__ void block_reduce_sum2_ss(double& a, double& b, double* sa, double* sb) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += shfl_down_d(a, o);
    b += shfl_down_d(b, o);
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0) {
    sa[warp] = a;
    sb[warp] = b;
  }
  __syncthreads();
  if (warp == 0) {
    a = lane < SS_THREADS / 32 ? sa[lane] : 0.0;
    b = lane < SS_THREADS / 32 ? sb[lane] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      a += shfl_down_d(a, o);
      b += shfl_down_d(b, o);
    }
  }
}

// jobs[0..njobs): the exponentials of a planned batch, applied to psi in order (psi is read once and
// stays in shared memory from job to job; every job still writes its result to global memory, so that
// psi holds the state before a job that fails).  status[e] is written per job; the loop stops at the
// first job that does not meet tol within its m_max (status[e].pad = 1).
__global__ void __cluster_dims__(SS_CTAS, 1, 1) __launch_bounds__(SS_THREADS, 1)
    csr_leja_sweep_small_kernel(CsrOp op, const cplx* v, cplx* out, const SweepJob* __restrict__ jobs, int njobs,
                                const double* __restrict__ leja_l, double tol, LejaStatus* status,
                                const LejaStatus* gate) {
  extern __shared__ __align__(16) unsigned char ss_smem[];
  __shared__ double sa[SS_THREADS / 32], sb[SS_THREADS / 32];
  __shared__ double part[2][SS_CTAS][2];            // [iteration parity][CTA](sw, sp): every CTA writes its entry in all copies
  __shared__ double s_norm0;
  __shared__ double s_l[kMaxDegree + 1];            // Leja points (c2)
  __shared__ double s_absd[kMaxDegree + 1];         // |d_k| of the current job
  cg::cluster_group cluster = cg::this_cluster();
  const int rank = (int)cluster.block_rank();
  if (status->pad) return;                          // an earlier sub-step did not converge (cluster-uniform)
  if (gate && !gate->done) return;                  // an earlier job of the plan failed: psi stays as that job found it
  cplx* wbuf[2] = {reinterpret_cast<cplx*>(ss_smem), reinterpret_cast<cplx*>(ss_smem) + kSmallSweepMaxN};
  // element i of buffer b in EVERY CTA of the cluster (own included) <- x
  auto push_w = [&](int b, int i, cplx x) {
    cplx* local = wbuf[b] + i;
#pragma unroll
    for (int c = 0; c < SS_CTAS; ++c) *cluster.map_shared_rank(local, c) = x;
  };
  const int tid = threadIdx.x, grp = tid / SS_G, sub = tid % SS_G;
  const int n = (int)op.n;
  const int per = (n + SS_CTAS - 1) / SS_CTAS;
  const int r0 = min(n, rank * per), r1 = min(n, r0 + per);
  for (int k = tid; k <= kMaxDegree; k += SS_THREADS) s_l[k] = leja_l[k];

  // the CTA's slice of every term -> shared memory (values, columns, local row pointers)
  cplx* prow = reinterpret_cast<cplx*>(ss_smem + SS_W_BYTES);    // p of the CTA's rows (kept out of registers so that
  cplx* mval = prow + SS_MAX_ROWS;                               // the pass loop need not be unrolled: code size)
  int32_t* mcol = reinterpret_cast<int32_t*>(mval + SS_MCAP);
  int* mrp = reinterpret_cast<int*>(mcol + SS_MCAP);           // [term][SS_MAX_ROWS + 1], offsets into mval/mcol
  int total = 0;
  for (int t = 0; t < op.nterms; ++t) total += op.t[t].rp[r1] - op.t[t].rp[r0];
  const bool cached = total <= SS_MCAP;                         // CTA-uniform
  if (cached) {
    int off = 0;
    for (int t = 0; t < op.nterms; ++t) {
      const CsrTerm& T = op.t[t];
      const int b = T.rp[r0], len = T.rp[r1] - b;
      for (int e = tid; e < len; e += SS_THREADS) {
        mval[off + e] = T.v[b + e];
        mcol[off + e] = T.ci[b + e];
      }
      for (int r = tid; r <= r1 - r0; r += SS_THREADS) mrp[t * (SS_MAX_ROWS + 1) + r] = off + T.rp[r0 + r] - b;
      off += len;
    }
  }

  // every CTA copies the whole v
  for (int i = tid; i < n; i += SS_THREADS) wbuf[0][i] = v[i];
  int cur = 0;
  __syncthreads();
  cluster.sync();                                   // everybody's buffers exist before remote writes start

#pragma unroll 1
  for (int e = 0; e < njobs; ++e) {
    const SweepJob& J = jobs[e];
    const int m_max = J.m_max, nterms = min(J.nterms, op.nterms);
    const double inv_gamma = J.inv_gamma, c_over_gamma = J.c_over_gamma;
    cplx coef[3];
#pragma unroll
    for (int t = 0; t < 3; ++t) coef[t] = J.coef[t];
    // S5 (fixed-order norm, identical in all CTAs); p_0 for the CTA's own rows
    double s0 = 0.0, s1 = 0.0;
    for (int i = tid; i < n; i += SS_THREADS) {
      const cplx x = wbuf[cur][i];
      s0 += x.x * x.x + x.y * x.y;
    }
    block_reduce_sum2_ss(s0, s1, sa, sb);
    if (tid == 0) s_norm0 = s0;
    for (int k = tid; k <= m_max; k += SS_THREADS) s_absd[k] = hypot(J.d[k].x, J.d[k].y);
    __syncthreads();
    s0 = s_norm0;
    const cplx d0 = J.d[0];
    for (int r = r0 + tid; r < r1; r += SS_THREADS) prow[r - r0] = cmul(d0, wbuf[cur][r]);
    double e_prev = s_absd[0] * sqrt(s0);
    double err = 0.0, sw = 0.0, sp = 0.0;
    int k = 0;
    bool done = false;
    __syncthreads();                                // part[0] is rewritten by iteration 2 at the earliest, but keep S5 whole

    while (!done && k < m_max) {
      ++k;
      const cplx dk = J.d[k];
      const double shift = c_over_gamma + s_l[k - 1];
      const cplx* w_in = wbuf[cur];
      double bw = 0.0, bp = 0.0;
#pragma unroll 1
      for (int j = 0; j * SS_GROUPS < per; ++j) {     // S6 on the CTA's row slice
        const int row = r0 + grp + j * SS_GROUPS;
        const bool valid = row < r1;
        cplx y = make_double2(0.0, 0.0);
        for (int t = 0; t < nterms; ++t) {
          const CsrTerm& T = op.t[t];
          cplx a = make_double2(0.0, 0.0);
          if (valid) {
            if (cached) {
              const int* lrp = mrp + t * (SS_MAX_ROWS + 1) + (row - r0);
              const int qe = lrp[1];
              for (int q = lrp[0] + sub; q < qe; q += SS_G) cfma(a, mval[q], w_in[mcol[q]]);
            } else {
              const int qe = T.rp[row + 1];
              for (int q = T.rp[row] + sub; q < qe; q += SS_G) cfma(a, T.v[q], w_in[T.ci[q]]);
            }
          }
          const cplx ca = cmul(coef[t], a);
          y.x += ca.x;
          y.y += ca.y;
        }
#pragma unroll
        for (int o = SS_G / 2; o > 0; o >>= 1) {
          y.x += shfl_xor_d(y.x, o);
          y.y += shfl_xor_d(y.y, o);
        }
        if (valid && sub == 0) {
          const cplx wi = w_in[row];
          cplx wn;
          wn.x = inv_gamma * y.x - shift * wi.x;
          wn.y = inv_gamma * y.y - shift * wi.y;
          cplx pi = prow[row - r0];
          cfma(pi, dk, wn);
          prow[row - r0] = pi;
          bw += wn.x * wn.x + wn.y * wn.y;
          bp += pi.x * pi.x + pi.y * pi.y;
          push_w(cur ^ 1, row, wn);
        }
      }
      block_reduce_sum2_ss(bw, bp, sa, sb);
      if (tid < SS_CTAS) {                            // thread c pushes this CTA's partials into CTA c's copy
        const double bw0 = __shfl_sync(0xffu, bw, 0), bp0 = __shfl_sync(0xffu, bp, 0);
        double* remote = cluster.map_shared_rank(&part[k & 1][rank][0], tid);
        remote[0] = bw0;
        remote[1] = bp0;
      }
      cluster.sync();                                 // every CTA's slice of the new w and its partials have arrived
      sw = 0.0;
      sp = 0.0;
#pragma unroll
      for (int c = 0; c < SS_CTAS; ++c) {             // same order in every CTA: same decision
        sw += part[k & 1][c][0];
        sp += part[k & 1][c][1];
      }
      const double e_k = s_absd[k] * sqrt(sw);        // S7
      err = e_k + e_prev;
      e_prev = e_k;
      done = err <= tol * sqrt(sp);
      cur ^= 1;
    }
    if (rank == 0 && tid == 0) {
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
    if (!done) break;                                 // cluster-uniform: psi (global) is the state before this job
    // S8: the result becomes the next job's input: pushed into the buffer that was this iteration's input (nobody
    // reads it any more: every CTA is past the last barrier), visible everywhere after one more barrier.
    const cplx phase = J.phase;
    const bool more = e + 1 < njobs;
    for (int r = r0 + tid; r < r1; r += SS_THREADS) {
      const cplx o = cmul(phase, prow[r - r0]);
      out[r] = o;
      if (more) push_w(cur ^ 1, r, o);
    }
    if (more) {
      cluster.sync();
      cur ^= 1;
    }
  }
  cluster.sync();                                   // no CTA leaves while its shared memory may still be written
}

}  // namespace

int launch_csr_leja_sweep_small_jobs(const CsrOp& op, cplx* psi, const SweepJob* jobs, int njobs, const double* leja_l,
                                     double tol, LejaStatus* status, const LejaStatus* gate, Workspace* ws,
                                     cudaStream_t st) {
  // per launch (cheap): the attribute is per device, a process-wide flag would miss a second GPU
  if (cudaFuncSetAttribute(csr_leja_sweep_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SS_SMEM) !=
      cudaSuccess)
    return MAGNUS_ECUDA;
  csr_leja_sweep_small_kernel<<<SS_CTAS, SS_THREADS, SS_SMEM, st>>>(op, psi, psi, jobs, njobs, leja_l, tol, status,
                                                                    gate);
  ws->launches += 1;
  return cudaGetLastError() == cudaSuccess ? MAGNUS_OK : MAGNUS_ECUDA;
}

// one sweep (leja_expmv, sub-steps, the fall-back after a failed batch): a one-job batch through the job slot 0
int launch_csr_leja_sweep_small(const CsrOp& op, const cplx* v, cplx* out, double inv_gamma, double c_over_gamma,
                                double tol, int m_max, cplx phase, const SweepTable& tab, Workspace* ws,
                                cudaStream_t st) {
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
  if (cudaFuncSetAttribute(csr_leja_sweep_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SS_SMEM) !=
      cudaSuccess)
    return MAGNUS_ECUDA;
  csr_leja_sweep_small_kernel<<<SS_CTAS, SS_THREADS, SS_SMEM, st>>>(op, v, out, ws->jobs, 1, ws->leja_l, tol,
                                                                    ws->status, nullptr);
  ws->launches += 1;
  return cudaGetLastError() == cudaSuccess ? MAGNUS_OK : MAGNUS_ECUDA;
}

}  // namespace magnus
