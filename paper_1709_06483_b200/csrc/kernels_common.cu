// Vector-level kernels of the Leja recurrence shared by the CSR and dense
// paths: rows S5 (init), S7 (stop test) and S8 (finish) of the scope table.
// P:n = PAPER.md line n; c1..c7 = readings in DESIGN.md section 3.
#include "magnus_internal.h"
#include "device_utils.cuh"
#include "leja_finalize.cuh"

namespace magnus {

// S5 (fragment lines 1-2): w = v; p = d0 v; partial sum |v|^2 per block.
__global__ void __launch_bounds__(256) leja_init_kernel(const cplx* __restrict__ v, cplx* __restrict__ w,
                                                         cplx* __restrict__ p, int64_t n, cplx d0, double abs_d0,
                                                         double* __restrict__ partials, LejaStatus* status,
                                                         unsigned* ticket) {
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
  if (last_block_ticket(ticket)) leja_finalize_warp0(partials, gridDim.x, abs_d0, 0.0, true, status);   // e_0 = |d_0| ||v||
}

// S7 (the stop test) runs in the last block of the init / iteration kernels: leja_finalize.cuh.

// S8 (c7): out = e^{-i (h/s) c} p.  in == out is allowed (gamma = 0 on an in-place step): no __restrict__.
__global__ void __launch_bounds__(256) scale_copy_kernel(const cplx* in, cplx* out, int64_t n, cplx phase) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    out[i] = cmul(phase, in[i]);
}

int device_sm_count() {
  static int cached[64] = {0};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
  if (cached[dev] == 0) {
    int v = 0;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) v = 148;
    cached[dev] = v;
  }
  return cached[dev];
}

static int vec_grid(int64_t n) {
  int64_t g = (n + 256 * 4 - 1) / (256 * 4);
  if (g < 1) g = 1;
  if (g > (int64_t)device_sm_count() * 8) g = (int64_t)device_sm_count() * 8;
  return (int)g;
}

void launch_leja_init(const cplx* v, cplx* w, cplx* p, int64_t n, cplx d0, double abs_d0, Workspace* ws,
                      cudaStream_t st) {
  const int g = vec_grid(n);
  leja_init_kernel<<<g, 256, 0, st>>>(v, w, p, n, d0, abs_d0, ws->partials, ws->status, ws->tickets);
  ws->launches += 1;
}

void launch_scale_copy(const cplx* in, cplx* out, int64_t n, cplx phase, cudaStream_t st, Workspace* ws) {
  scale_copy_kernel<<<vec_grid(n), 256, 0, st>>>(in, out, n, phase);
  ws->launches += 1;
}

void launch_leja_finish(const cplx* p, cplx* out, int64_t n, cplx phase, cudaStream_t st, Workspace* ws) {
  launch_scale_copy(p, out, n, phase, st, ws);
}

int workspace_alloc(Workspace* ws, int64_t n, cudaStream_t st) {
  ws->n = n;
  const size_t vb = sizeof(cplx) * (size_t)n;
  if (cudaMalloc(&ws->w[0], vb) != cudaSuccess) return MAGNUS_ENOMEM;
  if (cudaMalloc(&ws->w[1], vb) != cudaSuccess) return MAGNUS_ENOMEM;
  if (cudaMalloc(&ws->p, vb) != cudaSuccess) return MAGNUS_ENOMEM;
  if (cudaMalloc(&ws->partials, sizeof(double) * 2 * kMaxPartials) != cudaSuccess) return MAGNUS_ENOMEM;
  if (cudaMalloc(&ws->gersh, sizeof(double) * (2 * kMaxPartials + 2)) != cudaSuccess) return MAGNUS_ENOMEM;
  if (cudaMalloc(&ws->status, sizeof(LejaStatus)) != cudaSuccess) return MAGNUS_ENOMEM;
  if (cudaMalloc(&ws->tickets, 2 * sizeof(unsigned)) != cudaSuccess) return MAGNUS_ENOMEM;
  // on the caller's stream: a legacy-stream memset would not be ordered before kernels on a non-blocking stream
  if (cudaMemsetAsync(ws->tickets, 0, 2 * sizeof(unsigned), st) != cudaSuccess) return MAGNUS_ECUDA;
  if (cudaMallocHost(&ws->status_host, sizeof(LejaStatus)) != cudaSuccess) return MAGNUS_ENOMEM;
  if (cudaMallocHost(&ws->ab_host, 2 * sizeof(double)) != cudaSuccess) return MAGNUS_ENOMEM;
  for (int i = 0; i < 4; ++i)
    if (cudaEventCreate(&ws->ev[i]) != cudaSuccess) return MAGNUS_ECUDA;
  return MAGNUS_OK;
}

// Buffers of the planned-batch path; allocated once per workspace, on first use: ONE device block and ONE pinned
// block carved into the arrays (a pinned allocation costs about a millisecond, which a small problem notices).
namespace {
struct PlanLayout {
  size_t jobs, status, ab, coef, leja, bar, partials, total_dev, total_host;
  PlanLayout() {
    size_t o = 0;
    auto take = [&](size_t bytes) { const size_t at = o; o += (bytes + 255) / 256 * 256; return at; };
    jobs = take(sizeof(SweepJob) * kJobCap);
    status = take(sizeof(LejaStatus) * kPlanCap);
    ab = take(sizeof(double) * 2 * kPlanCap);
    coef = take(sizeof(double) * 4 * kPlanCap);
    total_host = o;                       // the host mirror stops here
    leja = take(sizeof(double) * (kMaxDegree + 1));
    bar = take(256);
    partials = take(sizeof(double) * 4 * kMaxPartials);
    total_dev = o;
  }
};
}  // namespace

int ensure_sweep_jobs(Workspace* ws, cudaStream_t st) {
  if (ws->jobs) return MAGNUS_OK;
  const PlanLayout L;
  char* dev = nullptr;
  char* host = nullptr;
  bool ok = cudaMalloc(&dev, L.total_dev) == cudaSuccess && cudaMallocHost(&host, L.total_host) == cudaSuccess;
  for (int i = 0; ok && i < 2 * kJobRing; ++i) ok = cudaEventCreate(&ws->ring_ev[i]) == cudaSuccess;
  if (ok)
    ok = cudaMemsetAsync(dev + L.bar, 0, 256, st) == cudaSuccess &&      // leja_points() is a process-lifetime table
         cudaMemcpyAsync(dev + L.leja, leja_points(), sizeof(double) * (kMaxDegree + 1), cudaMemcpyHostToDevice, st) == cudaSuccess;
  if (!ok) {
    cudaGetLastError();
    cudaFree(dev);
    if (host) cudaFreeHost(host);
    return MAGNUS_ENOMEM;
  }
  ws->jobs = reinterpret_cast<SweepJob*>(dev + L.jobs);
  ws->status_arr = reinterpret_cast<LejaStatus*>(dev + L.status);
  ws->ab_arr = reinterpret_cast<double*>(dev + L.ab);
  ws->coef_arr = reinterpret_cast<double*>(dev + L.coef);
  ws->leja_l = reinterpret_cast<double*>(dev + L.leja);
  ws->grid_bar = reinterpret_cast<unsigned*>(dev + L.bar);
  ws->sweep_partials = reinterpret_cast<double*>(dev + L.partials);
  ws->jobs_host = reinterpret_cast<SweepJob*>(host + L.jobs);
  ws->status_arr_host = reinterpret_cast<LejaStatus*>(host + L.status);
  ws->ab_arr_host = reinterpret_cast<double*>(host + L.ab);
  ws->coef_arr_host = reinterpret_cast<double*>(host + L.coef);
  return MAGNUS_OK;
}

void workspace_free(Workspace* ws) {
  stream_maps_free(ws);
  cudaFree(ws->jobs);                                   // the one device block of ensure_sweep_jobs starts here
  for (int i = 0; i < 2 * kJobRing; ++i)
    if (ws->ring_ev[i]) cudaEventDestroy(ws->ring_ev[i]);
  if (ws->jobs_host) cudaFreeHost(ws->jobs_host);       // ... and the one pinned block here
  cudaFree(ws->w[0]);
  cudaFree(ws->w[1]);
  cudaFree(ws->p);
  cudaFree(ws->partials);
  cudaFree(ws->gersh);
  cudaFree(ws->status);
  cudaFree(ws->tickets);
  if (ws->status_host) cudaFreeHost(ws->status_host);
  if (ws->ab_host) cudaFreeHost(ws->ab_host);
  for (int i = 0; i < 4; ++i)
    if (ws->ev[i]) cudaEventDestroy(ws->ev[i]);
  *ws = Workspace();
}

}  // namespace magnus
