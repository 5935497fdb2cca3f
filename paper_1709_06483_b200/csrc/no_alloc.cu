// magnus_leja_iteration_dense_noalloc -- the fused dense Leja iteration (row S6) for callers that
// must not allocate.
//
// Who that is: a process whose device memory is already spoken for -- a PyTorch job whose caching allocator has
// taken the GPU, a service running under a fixed memory budget, a plug-in loaded into somebody else's CUDA
// context -- cannot count on cudaMalloc succeeding, and a loop with a latency bound cannot pay for it either:
// cudaMalloc / cudaFree take driver locks and cudaFree waits for the whole device.  Every other entry point of
// this library that reduces over the grid (magnus_leja_iteration, magnus_gershgorin, leja_expmv, a handle) gets
// its per-block partial sums and its last-block ticket from a workspace it allocates.  This one keeps them in a
// fixed array that is part of the library image instead, so the call itself allocates nothing: no cudaMalloc,
// cudaMallocHost, cudaFree, event or stream creation, and no library routine that would.
//
// Price and rules (also in include/magnus.h):
//   * the array is kNoAllocScratchBytes = 65,792 bytes, present on EVERY GPU on which this library's module gets
//     loaded, from that load until the process exits, whether or not this entry point is ever called;
//   * it bounds the problem: n <= MAGNUS_NOALLOC_MAX_N = 32768 (one 8-row block per partial slot, 4096 slots);
//     larger n is refused with MAGNUS_EINVAL and a message, never truncated;
//   * one array per device, shared by every call: two calls that can run at the same time on one device (different
//     streams, different host threads) race on the partial sums and the ticket and produce wrong norms or a
//     missing result.  Serialise them (one stream, or events);
//   * the array keeps what the last call left.  The partial slots need no clearing (every block of a launch
//     overwrites its own slot before anybody reads it); the ticket must be zero when a launch starts, so every
//     call enqueues a memset of the ticket block ahead of its kernel -- a launch that died half-way cannot poison
//     the next one;
//   * the first call on a device looks up the array's device address (cudaGetSymbolAddress, which may load the
//     module).  Make that first call per device outside any stream capture; later calls only enqueue a memset and a
//     kernel on the caller's stream.
//
// The arithmetic is the one of dense_leja_iter_kernel (kernels_dense.cu): one warp per row, lanes stride the row
// with 128-bit streaming loads, 8 loads in flight, two accumulators, shuffle tree; for n <= 32768 the existing
// launcher also uses one block per 8 rows, so w_out, p AND the two sums come out bit-identical to
// magnus_leja_iteration on a dense matrix.  No stop test here (no LejaStatus): the sums go to the caller's buffer.
#include <mutex>

#include "magnus_internal.h"
#include "device_utils.cuh"

constexpr int kNaWarps = 8;                                        // rows per block, one warp each
constexpr int kNaMaxBlocks = MAGNUS_NOALLOC_MAX_N / kNaWarps;      // 4096 partial slots
constexpr int kNaTicketDoubles = 32;                               // a 256-byte block of its own for the ticket
constexpr int kNaLoads = 8;                                        // independent 128-bit loads in flight per lane

// THE scratch: [0, 2*kNaMaxBlocks) per-block (sum |w+|^2, sum |p|^2); the ticket (an unsigned) sits at
// element 2*kNaMaxBlocks.  In host code this name is only a handle for cudaGetSymbolAddress -- it is NOT a device
// address and must never be passed to a kernel; device code below does not name it either, it gets the looked-up
// pointer, so there is exactly one way the address travels.
static __device__ __align__(256) double g_noalloc_scratch[2 * kNaMaxBlocks + kNaTicketDoubles];
constexpr size_t kNoAllocScratchBytes = sizeof(double) * (2 * kNaMaxBlocks + kNaTicketDoubles);
static_assert(kNoAllocScratchBytes == 65792, "documented size of the static scratch");

namespace magnus {

namespace {


__global__ void __launch_bounds__(kNaWarps * 32)
dense_leja_iter_noalloc_kernel(int64_t n, const cplx* __restrict__ M, int64_t ld, const cplx* __restrict__ w_in,
                               cplx* __restrict__ w_out, cplx* __restrict__ p, double inv_gamma, double shift, cplx dk,
                               double* partials, unsigned* ticket, double* __restrict__ sums_out) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint64_t pol = policy_evict_first();
  const int64_t row = (int64_t)blockIdx.x * kNaWarps + warp;
  double sw = 0.0, sp = 0.0;
  if (row < n) {
    const cplx* __restrict__ m = M + row * ld;
    cplx acc[2] = {make_double2(0.0, 0.0), make_double2(0.0, 0.0)};
    int64_t j = lane;
    for (; j + 32 * (kNaLoads - 1) < n; j += 32 * kNaLoads) {
      cplx mv[kNaLoads], xv[kNaLoads];
#pragma unroll
      for (int u = 0; u < kNaLoads; ++u) mv[u] = ld_stream(m + j + 32 * u, pol);
#pragma unroll
      for (int u = 0; u < kNaLoads; ++u) xv[u] = w_in[j + 32 * u];
#pragma unroll
      for (int u = 0; u < kNaLoads; ++u) cfma(acc[u & 1], mv[u], xv[u]);
    }
    for (; j < n; j += 32) cfma(acc[0], ld_stream(m + j, pol), w_in[j]);
    cplx y = make_double2(acc[0].x + acc[1].x, acc[0].y + acc[1].y);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      y.x += shfl_xor_d(y.x, o);
      y.y += shfl_xor_d(y.y, o);
    }
    if (lane == 0) {
      const cplx wi = w_in[row];
      cplx wn;
      wn.x = inv_gamma * y.x - shift * wi.x;
      wn.y = inv_gamma * y.y - shift * wi.y;
      w_out[row] = wn;
      cplx pi = p[row];
      cfma(pi, dk, wn);
      p[row] = pi;
      sw = wn.x * wn.x + wn.y * wn.y;
      sp = pi.x * pi.x + pi.y * pi.y;
    }
  }
  block_reduce_sum2<kNaWarps * 32>(sw, sp);
  __shared__ int is_last;
  if (threadIdx.x == 0) {
    partials[2 * blockIdx.x] = sw;
    partials[2 * blockIdx.x + 1] = sp;
    __threadfence();
    is_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);   // the memset ahead of the launch set it to 0
    __threadfence();
  }
  __syncthreads();
  if (!is_last || threadIdx.x >= 32) return;
  // last block to finish, warp 0: sums in slot order (lane-strided, then a shuffle tree), whichever block this is
  double tw = 0.0, tp = 0.0;
  for (int b = threadIdx.x; b < (int)gridDim.x; b += 32) {
    tw += __ldcg(partials + 2 * b);
    tp += __ldcg(partials + 2 * b + 1);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    tw += shfl_down_d(tw, o);
    tp += shfl_down_d(tp, o);
  }
  if (threadIdx.x == 0) {
    sums_out[0] = tw;
    sums_out[1] = tp;
  }
}

// Device address of g_noalloc_scratch per device ordinal, looked up once with that device current.
constexpr int kNaMaxDevices = 64;
std::mutex g_na_mutex;
double* g_na_ptr[kNaMaxDevices] = {};

int noalloc_scratch_ptr(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) {
    set_error("magnus_leja_iteration_dense_noalloc: no current CUDA device (%s); no CPU fallback", cudaGetErrorString(e));
    cudaGetLastError();
    return MAGNUS_ECUDA;
  }
  if (dev < 0 || dev >= kNaMaxDevices) {
    set_error("magnus_leja_iteration_dense_noalloc: device ordinal %d outside 0..%d", dev, kNaMaxDevices - 1);
    return MAGNUS_EINVAL;
  }
  std::lock_guard<std::mutex> lock(g_na_mutex);
  if (!g_na_ptr[dev]) {
    double* ptr = nullptr;
    e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch);   // the current device's copy of the array
    if (e != cudaSuccess || !ptr) {
      set_error("magnus_leja_iteration_dense_noalloc: cudaGetSymbolAddress failed on device %d: %s", dev,
                cudaGetErrorString(e));
      cudaGetLastError();
      return MAGNUS_ECUDA;
    }
    g_na_ptr[dev] = ptr;
  }
  *out = g_na_ptr[dev];
  return MAGNUS_OK;
}

bool aligned16(const void* p) { return ((uintptr_t)p & 15u) == 0; }

}  // namespace
}  // namespace magnus

using namespace magnus;

extern "C" int magnus_leja_iteration_dense_noalloc(int64_t n, const void* M, int64_t ld, const void* w_in, void* w_out,
                                                   void* p, double inv_gamma, double shift, double d_re, double d_im,
                                                   void* stream, double* sums_dev) {
  if (n <= 0) { set_error("magnus_leja_iteration_dense_noalloc: n must be positive"); return MAGNUS_EINVAL; }
  if (n > MAGNUS_NOALLOC_MAX_N) {
    set_error("magnus_leja_iteration_dense_noalloc: n = %lld exceeds MAGNUS_NOALLOC_MAX_N = %d, the size the library's "
              "static scratch (%zu bytes per GPU) is laid out for; use magnus_leja_iteration, which allocates",
              (long long)n, MAGNUS_NOALLOC_MAX_N, kNoAllocScratchBytes);
    return MAGNUS_EINVAL;
  }
  if (ld == 0) ld = n;
  if (ld < n) { set_error("magnus_leja_iteration_dense_noalloc: ld < n"); return MAGNUS_EINVAL; }
  if (!M || !w_in || !w_out || !p || !sums_dev || w_in == w_out || p == w_in || p == w_out) {
    set_error("magnus_leja_iteration_dense_noalloc: null or aliased vector / matrix pointer");
    return MAGNUS_EINVAL;
  }
  if (!aligned16(M) || !aligned16(w_in) || !aligned16(w_out) || !aligned16(p) || ((uintptr_t)sums_dev & 7u)) {
    set_error("magnus_leja_iteration_dense_noalloc: complex128 pointers must be 16-byte aligned, sums_dev 8-byte");
    return MAGNUS_EINVAL;
  }
  double* scratch = nullptr;
  const int rc = noalloc_scratch_ptr(&scratch);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  double* partials = scratch;
  unsigned* ticket = (unsigned*)(scratch + 2 * kNaMaxBlocks);
  cudaError_t e = cudaMemsetAsync(ticket, 0, sizeof(double) * kNaTicketDoubles, st);
  if (e == cudaSuccess) {
    const int grid = (int)((n + kNaWarps - 1) / kNaWarps);
    dense_leja_iter_noalloc_kernel<<<grid, kNaWarps * 32, 0, st>>>(n, (const cplx*)M, ld, (const cplx*)w_in,
                                                                   (cplx*)w_out, (cplx*)p, inv_gamma, shift,
                                                                   make_double2(d_re, d_im), partials, ticket, sums_dev);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) {
    set_error("magnus_leja_iteration_dense_noalloc: enqueue failed: %s", cudaGetErrorString(e));
    return MAGNUS_ECUDA;
  }
  return MAGNUS_OK;
}
