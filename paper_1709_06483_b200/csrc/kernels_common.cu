// Vector-level kernels of the Leja recurrence shared by the CSR and dense
// paths: rows S5 (init), S7 (stop test) and S8 (finish) of the scope table.
// P:n = PAPER.md line n; c1..c7 = readings in DESIGN.md section 3.
#include "magnus_internal.h"
#include "device_utils.cuh"

namespace magnus {

// S5 (fragment lines 1-2): w = v; p = d0 v; partial sum |v|^2 per block.
__global__ void __launch_bounds__(256) leja_init_kernel(const cplx* __restrict__ v, cplx* __restrict__ w,
                                                         cplx* __restrict__ p, int64_t n, cplx d0,
                                                         double* __restrict__ partials) {
  double s = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const cplx x = v[i];
    w[i] = x;
    p[i] = cmul(d0, x);
    s += x.x * x.x + x.y * x.y;
  }
  double t = 0.0;
  block_reduce_sum2<256>(s, t);
  if (threadIdx.x == 0) {
    partials[2 * blockIdx.x] = s;
    partials[2 * blockIdx.x + 1] = 0.0;
  }
}

// S7 ("early termination criterion"; c6).  One block.  Sums the per-block
// partials in a fixed order (deterministic: no floating-point atomics), then
//   k = 0 (after init):  e_prev = |d_0| ||v||
//   k >= 1            :  e_k = |d_k| ||w_k||;  done if e_k + e_{k-1} <= tol ||p_k||
__global__ void __launch_bounds__(256) leja_finalize_kernel(const double* __restrict__ partials, int nblk,
                                                             double abs_dk, double tol, int is_init,
                                                             LejaStatus* __restrict__ st) {
  if (!is_init && st->done) return;
  double sw = 0.0, sp = 0.0;
  for (int b = threadIdx.x; b < nblk; b += 256) {
    sw += partials[2 * b];
    sp += partials[2 * b + 1];
  }
  block_reduce_sum2<256>(sw, sp);
  if (threadIdx.x == 0) {
    if (is_init) {
      st->done = 0;
      st->k = 0;
      st->e_prev = abs_dk * sqrt(sw);
      st->norm_w2 = sw;
      st->norm_p2 = 0.0;
    } else {
      const double e_k = abs_dk * sqrt(sw);
      const double err = e_k + st->e_prev;
      st->k += 1;
      st->iters += 1;
      st->err_est = err;
      st->norm_w2 = sw;
      st->norm_p2 = sp;
      st->e_prev = e_k;
      if (err <= tol * sqrt(sp)) st->done = 1;
    }
  }
}

// S8 (c7): out = e^{-i (h/s) c} p.
__global__ void __launch_bounds__(256) scale_copy_kernel(const cplx* __restrict__ in, cplx* __restrict__ out, int64_t n,
                                                          cplx phase) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    out[i] = cmul(phase, in[i]);
}

// Final min / max over the per-block Gershgorin bounds (row S3).  One block.
// in: [2*b] = block min of (Re M_ii - R_i), [2*b+1] = block max of (Re M_ii + R_i);
// out[0], out[1] = global min, max.  min/max are exact, so order does not matter.
__global__ void __launch_bounds__(256) minmax_finalize_kernel(const double* __restrict__ in, int nblk,
                                                               double* __restrict__ out) {
  double lo = INFINITY, hi = -INFINITY;
  for (int b = threadIdx.x; b < nblk; b += 256) {
    lo = fmin(lo, in[2 * b]);
    hi = fmax(hi, in[2 * b + 1]);
  }
  block_reduce_minmax<256>(lo, hi);
  if (threadIdx.x == 0) {
    out[0] = lo;
    out[1] = hi;
  }
}

static int vec_grid(int64_t n) {
  int64_t g = (n + 256 * 4 - 1) / (256 * 4);
  if (g < 1) g = 1;
  if (g > 148 * 8) g = 148 * 8;
  return (int)g;
}

void launch_leja_init(const cplx* v, cplx* w, cplx* p, int64_t n, cplx d0, double abs_d0, Workspace* ws,
                      cudaStream_t st) {
  const int g = vec_grid(n);
  leja_init_kernel<<<g, 256, 0, st>>>(v, w, p, n, d0, ws->partials);
  leja_finalize_kernel<<<1, 256, 0, st>>>(ws->partials, g, abs_d0, 0.0, 1, ws->status);
  ws->launches += 2;
}

void launch_leja_finalize(int nblk, double abs_dk, double tol, Workspace* ws, cudaStream_t st) {
  leja_finalize_kernel<<<1, 256, 0, st>>>(ws->partials, nblk, abs_dk, tol, 0, ws->status);
  ws->launches += 1;
}

void launch_scale_copy(const cplx* in, cplx* out, int64_t n, cplx phase, cudaStream_t st, Workspace* ws) {
  scale_copy_kernel<<<vec_grid(n), 256, 0, st>>>(in, out, n, phase);
  ws->launches += 1;
}

void launch_leja_finish(const cplx* p, cplx* out, int64_t n, cplx phase, cudaStream_t st, Workspace* ws) {
  launch_scale_copy(p, out, n, phase, st, ws);
}

void launch_minmax_finalize(int nblk, Workspace* ws, cudaStream_t st) {
  minmax_finalize_kernel<<<1, 256, 0, st>>>(ws->gersh, nblk, ws->gersh + 2 * kMaxPartials);
  ws->launches += 1;
}

int workspace_alloc(Workspace* ws, int64_t n) {
  ws->n = n;
  const size_t vb = sizeof(cplx) * (size_t)n;
  if (cudaMalloc(&ws->w[0], vb) != cudaSuccess) return MAGNUS_ENOMEM;
  if (cudaMalloc(&ws->w[1], vb) != cudaSuccess) return MAGNUS_ENOMEM;
  if (cudaMalloc(&ws->p, vb) != cudaSuccess) return MAGNUS_ENOMEM;
  if (cudaMalloc(&ws->partials, sizeof(double) * 2 * kMaxPartials) != cudaSuccess) return MAGNUS_ENOMEM;
  if (cudaMalloc(&ws->gersh, sizeof(double) * (2 * kMaxPartials + 2)) != cudaSuccess) return MAGNUS_ENOMEM;
  if (cudaMalloc(&ws->status, sizeof(LejaStatus)) != cudaSuccess) return MAGNUS_ENOMEM;
  if (cudaMallocHost(&ws->status_host, sizeof(LejaStatus)) != cudaSuccess) return MAGNUS_ENOMEM;
  if (cudaMallocHost(&ws->ab_host, 2 * sizeof(double)) != cudaSuccess) return MAGNUS_ENOMEM;
  for (int i = 0; i < 4; ++i)
    if (cudaEventCreate(&ws->ev[i]) != cudaSuccess) return MAGNUS_ECUDA;
  return MAGNUS_OK;
}

void workspace_free(Workspace* ws) {
  cudaFree(ws->w[0]);
  cudaFree(ws->w[1]);
  cudaFree(ws->p);
  cudaFree(ws->partials);
  cudaFree(ws->gersh);
  cudaFree(ws->status);
  if (ws->status_host) cudaFreeHost(ws->status_host);
  if (ws->ab_host) cudaFreeHost(ws->ab_host);
  for (int i = 0; i < 4; ++i)
    if (ws->ev[i]) cudaEventDestroy(ws->ev[i]);
  *ws = Workspace();
}

}  // namespace magnus
