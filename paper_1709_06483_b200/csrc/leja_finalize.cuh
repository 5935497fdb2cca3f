// S7 fused into the producing kernels: the LAST block of a launch to finish (atomic ticket, no
// spinning) sums the per-block partials in a fixed order and applies the stop test
// ("early termination criterion"; reading c6), so an iteration is one launch.
// Deterministic: the ticket only decides WHICH block does the sum, never its order.
#ifndef MAGNUS_LEJA_FINALIZE_CUH
#define MAGNUS_LEJA_FINALIZE_CUH

#include "magnus_internal.h"
#include "device_utils.cuh"

namespace magnus {

// Call after thread 0 of the block has stored its partials.  Returns true (block-uniform) in
// exactly one block per launch, after every other block's partials are visible.  The counter
// wraps to 0 by itself (atomicInc), ready for the next launch.
__device__ __forceinline__ bool last_block_ticket(unsigned* counter) {
  __shared__ int is_last;
  if (threadIdx.x == 0) {
    __threadfence();
    const unsigned t = atomicInc(counter, gridDim.x - 1);
    is_last = (t == gridDim.x - 1);
    __threadfence();
  }
  __syncthreads();
  return is_last != 0;
}

// Warp 0 of the last block: fixed-order sums of partials[2b], partials[2b+1], b < nblk (lane-strided,
// then a shuffle tree -- independent of the block size of the calling kernel), then
//   is_init:  e_prev = |d_0| ||v||
//   else:     e_k = |d_k| ||w_k||; done if e_k + e_{k-1} <= tol ||p_k||
__device__ __forceinline__ void leja_finalize_warp0(const double* partials, int nblk, double abs_dk, double tol,
                                                    bool is_init, LejaStatus* st) {
  if (threadIdx.x >= 32) return;
  double sw = 0.0, sp = 0.0;
  for (int b = threadIdx.x; b < nblk; b += 32) {
    sw += __ldcg(partials + 2 * b);
    sp += __ldcg(partials + 2 * b + 1);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    sw += shfl_down_d(sw, o);
    sp += shfl_down_d(sp, o);
  }
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

// Same for the Gershgorin bounds: out[0] = min over blocks of in[2b], out[1] = max of in[2b+1].
__device__ __forceinline__ void minmax_finalize_warp0(const double* in, int nblk, double* out) {
  if (threadIdx.x >= 32) return;
  double lo = INFINITY, hi = -INFINITY;
  for (int b = threadIdx.x; b < nblk; b += 32) {
    lo = fmin(lo, __ldcg(in + 2 * b));
    hi = fmax(hi, __ldcg(in + 2 * b + 1));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lo = fmin(lo, shfl_down_d(lo, o));
    hi = fmax(hi, shfl_down_d(hi, o));
  }
  if (threadIdx.x == 0) {
    out[0] = lo;
    out[1] = hi;
  }
}

}  // namespace magnus
#endif
