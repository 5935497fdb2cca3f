// Shortcut "tight spectral interval" (reported separately from the mandated Gershgorin path).
// P:190 only asks for "an estimate on the spectrum"; NS fixes Gershgorin for the mandated path.  On dense random
// Hermitian matrices Gershgorin over-estimates the spectral radius 20x (n = 2048) to 57x (n = 16384), which
// costs 1.6-3x more Leja iterations.  Here the interval of an exponential comes from m steps of the Lanczos
// process on M started at the vector v that is about to be propagated (reading ti):
//   q_1 = v / ||v||;  for j = 1..m:  u = M q_j - beta_{j-1} q_{j-1};  alpha_j = Re(q_j^H u);
//                                    r = u - alpha_j q_j;  beta_j = ||r||;  q_{j+1} = r / beta_j,
//   [theta_min(T) - beta_m, theta_max(T) + beta_m],  T = tridiag(alpha; beta_1..beta_{m-1}).
// The product M q_j is the library's fused Leja iteration kernel run as a plain mat-vec (1/gamma = 1, shift = 0,
// d_k = 0); this file holds the vector kernels around it.  All scalars stay on the device until the m steps are
// over (no host round trip per step); sums are fixed trees + a fixed-order sum of block partials by the last block.
// scal[0] = ||v||, scal[1] = beta_{j-1}, scal[2 + j] = alpha_j, scal[2 + m + j] = beta_j  (j = 0..m-1).
#include "magnus_internal.h"
#include "device_utils.cuh"
#include "leja_finalize.cuh"

namespace magnus {

namespace {

constexpr int LZ_THREADS = 256;

// sum of the first component of the block partials -> thread 0 of the calling (last) block
__device__ __forceinline__ double sum_partials_warp0(const double* partials, int nblk) {
  double s = 0.0;
  if (threadIdx.x < 32) {
    for (int b = threadIdx.x; b < nblk; b += 32) s += __ldcg(partials + 2 * b);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += shfl_down_d(s, o);
  }
  return s;
}

__global__ void __launch_bounds__(LZ_THREADS) lanczos_norm_kernel(const cplx* __restrict__ v, int64_t n, double* partials,
                                                                   unsigned* ticket, double* scal) {
  double s = 0.0, t = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const cplx x = v[i];
    s += x.x * x.x + x.y * x.y;
  }
  block_reduce_sum2<LZ_THREADS>(s, t);
  if (threadIdx.x == 0) partials[2 * blockIdx.x] = s;
  if (last_block_ticket(ticket)) {
    const double tot = sum_partials_warp0(partials, gridDim.x);
    if (threadIdx.x == 0) {
      scal[0] = sqrt(tot);
      scal[1] = 0.0;
    }
  }
}

// q = v / ||v||, q_prev = 0
__global__ void __launch_bounds__(LZ_THREADS) lanczos_start_kernel(const cplx* __restrict__ v, cplx* __restrict__ q,
                                                                    cplx* __restrict__ qprev, int64_t n,
                                                                    const double* __restrict__ scal) {
  const double nv = scal[0], inv = nv > 0.0 ? 1.0 / nv : 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const cplx x = v[i];
    q[i] = make_double2(x.x * inv, x.y * inv);
    qprev[i] = make_double2(0.0, 0.0);
  }
}

// u -= beta_{j-1} q_{j-1};  alpha_j = Re(q_j^H u)
__global__ void __launch_bounds__(LZ_THREADS) lanczos_alpha_kernel(cplx* __restrict__ u, const cplx* __restrict__ q,
                                                                    const cplx* __restrict__ qprev, int64_t n, double* scal,
                                                                    int j, double* partials, unsigned* ticket) {
  const double bp = scal[1];
  double s = 0.0, t = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    cplx x = u[i];
    const cplx p = qprev[i], y = q[i];
    x.x -= bp * p.x;
    x.y -= bp * p.y;
    u[i] = x;
    s += y.x * x.x + y.y * x.y;
  }
  block_reduce_sum2<LZ_THREADS>(s, t);
  if (threadIdx.x == 0) partials[2 * blockIdx.x] = s;
  if (last_block_ticket(ticket)) {
    const double tot = sum_partials_warp0(partials, gridDim.x);
    if (threadIdx.x == 0) scal[2 + j] = tot;
  }
}

// r = u - alpha_j q_j (written over q_{j-1}, which is no longer needed);  beta_j = ||r||
__global__ void __launch_bounds__(LZ_THREADS) lanczos_beta_kernel(const cplx* __restrict__ u, const cplx* __restrict__ q,
                                                                   cplx* __restrict__ r, int64_t n, double* scal, int j, int m,
                                                                   double* partials, unsigned* ticket) {
  const double al = scal[2 + j];
  double s = 0.0, t = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const cplx x = u[i], y = q[i];
    const cplx z = make_double2(x.x - al * y.x, x.y - al * y.y);
    r[i] = z;
    s += z.x * z.x + z.y * z.y;
  }
  block_reduce_sum2<LZ_THREADS>(s, t);
  if (threadIdx.x == 0) partials[2 * blockIdx.x] = s;
  if (last_block_ticket(ticket)) {
    const double tot = sum_partials_warp0(partials, gridDim.x);
    if (threadIdx.x == 0) {
      const double be = sqrt(tot);
      scal[2 + m + j] = be;
      scal[1] = be;
    }
  }
}

// q_{j+1} = r / beta_j in place (0 if beta_j = 0: the host cuts T off there anyway)
__global__ void __launch_bounds__(LZ_THREADS) lanczos_scale_kernel(cplx* __restrict__ r, int64_t n,
                                                                    const double* __restrict__ scal) {
  const double be = scal[1], inv = be > 0.0 ? 1.0 / be : 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    cplx x = r[i];
    x.x *= inv;
    x.y *= inv;
    r[i] = x;
  }
}

int lz_grid(int64_t n) {
  int64_t g = (n + LZ_THREADS * 4 - 1) / (LZ_THREADS * 4);
  if (g < 1) g = 1;
  const int64_t cap = (int64_t)device_sm_count() * 8;
  if (g > cap) g = cap;
  if (g > kMaxPartials) g = kMaxPartials;
  return (int)g;
}

}  // namespace

void launch_lanczos_start(const cplx* v, cplx* q, cplx* qprev, int64_t n, double* scal, Workspace* ws, cudaStream_t st) {
  const int g = lz_grid(n);
  lanczos_norm_kernel<<<g, LZ_THREADS, 0, st>>>(v, n, ws->partials, ws->tickets, scal);
  lanczos_start_kernel<<<g, LZ_THREADS, 0, st>>>(v, q, qprev, n, scal);
  ws->launches += 2;
}

// after u = M q_j: alpha_j, r (over qprev), beta_j, q_{j+1} = r / beta_j (in place, in the qprev buffer)
void launch_lanczos_step(cplx* u, const cplx* q, cplx* qprev, int64_t n, double* scal, int j, int m, Workspace* ws,
                         cudaStream_t st) {
  const int g = lz_grid(n);
  lanczos_alpha_kernel<<<g, LZ_THREADS, 0, st>>>(u, q, qprev, n, scal, j, ws->partials, ws->tickets);
  lanczos_beta_kernel<<<g, LZ_THREADS, 0, st>>>(u, q, qprev, n, scal, j, m, ws->partials, ws->tickets);
  lanczos_scale_kernel<<<g, LZ_THREADS, 0, st>>>(qprev, n, scal);
  ws->launches += 3;
}

}  // namespace magnus
