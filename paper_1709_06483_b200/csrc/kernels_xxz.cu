// Shortcut (SURVEY 8f-4 "matrix-free XXZ apply", reported separately from the mandated CSR path): the fused Leja
// iteration (row S6) for the periodic XXZ chain in a transverse field WITHOUT a stored matrix.
//   H0 = sum over the N periodic nearest-neighbour bonds of  jxy (sx sx + sy sy) + jz sz sz,   H1 = hx sum_i sx_i
// (the structure of the paper's Example 2, and of BASELINE configs 1, 3, 5).  In the sz basis
// (site j on bit N - j; bonds (bit b, bit b-1), b = N-1..1, plus the periodic bond (bit N-1, bit 0)) row r holds
//   the diagonal jz (N - 2k), k = antiparallel bonds of r,
//   2 jxy at r ^ (pair mask) for every antiparallel bond,   and   g hx at r ^ (1 << b) for every bit b,
// so the matrix entries are recomputed from the bits of r and an iteration moves vector bytes only:
//   w+_r = (1/gamma) (M w)_r - shift w_r,   p_r += d_k w+_r,   partial sums of |w+|^2, |p|^2   (c5).
// A lane is a row, a warp 32 consecutive rows: flips of bits 0..4 are warp shuffles of the lane's own w, flips of
// higher bits are coalesced 512-byte gathers (the 32 partners are consecutive).  Deterministic: fixed order of the
// terms (single flips by ascending bit, then bonds by descending bit, then the periodic bond), fixed reduction trees.
#include "magnus_internal.h"
#include "device_utils.cuh"
#include "leja_finalize.cuh"

namespace magnus {

namespace {

__device__ __forceinline__ cplx shfl_xor_c(cplx v, int m) {
  return make_double2(__shfl_xor_sync(0xffffffffu, v.x, m), __shfl_xor_sync(0xffffffffu, v.y, m));
}

__global__ void __launch_bounds__(256) xxz_leja_iter_kernel(XxzOp op, const cplx* __restrict__ w_in,
                                                             cplx* __restrict__ w_out, cplx* __restrict__ p,
                                                             double inv_gamma, double shift, cplx dk, double abs_dk,
                                                             double tol, LejaStatus* status, double* partials,
                                                             unsigned* ticket) {
  if (status->done) return;
  const int N = op.nspins, lane = threadIdx.x & 31;
  const int64_t n = (int64_t)1 << N;
  const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  const int low = N < 5 ? N : 5;                      // bits whose flip stays inside the warp's 32 rows
  double sw = 0.0, sp = 0.0;
  for (int64_t base = warp0 << 5; base < n; base += nwarps << 5) {
    const int64_t r = base + lane;
    const bool valid = r < n;                         // n < 32 only for N < 5
    const cplx wi = valid ? w_in[r] : make_double2(0.0, 0.0);
    // H1: single flips, ascending bit
    cplx s1 = make_double2(0.0, 0.0);
    for (int b = 0; b < low; ++b) {
      const cplx x = shfl_xor_c(wi, 1 << b);
      s1.x += x.x;
      s1.y += x.y;
    }
#pragma unroll 8
    for (int b = 5; b < N; ++b) {
      const cplx x = w_in[r ^ ((int64_t)1 << b)];
      s1.x += x.x;
      s1.y += x.y;
    }
    // H0: bonds (bit b, bit b-1), descending b; antiparallel pairs flip with amplitude 2 jxy
    cplx s2 = make_double2(0.0, 0.0);
    int k = 0;
#pragma unroll 8
    for (int b = N - 1; b >= 6; --b) {                // both bits above the lane bits: the same for the whole warp
      const bool anti = (((r >> b) ^ (r >> (b - 1))) & 1) != 0;
      if (anti) {
        const cplx x = w_in[r ^ ((int64_t)3 << (b - 1))];
        s2.x += x.x;
        s2.y += x.y;
        ++k;
      }
    }
    if (N > 5) {                                      // bond (5, 4): the partner sits in the neighbouring 32-row block
      const bool anti = (((r >> 5) ^ (r >> 4)) & 1) != 0;
      cplx x = make_double2(0.0, 0.0);
      if (anti) x = w_in[r ^ 0x30];
      s2.x += x.x;
      s2.y += x.y;
      k += anti;
    }
    for (int b = low - 1; b >= 1; --b) {              // both bits inside the warp: shuffles
      const bool anti = (((r >> b) ^ (r >> (b - 1))) & 1) != 0;
      const cplx x = shfl_xor_c(wi, 3 << (b - 1));
      if (anti) {
        s2.x += x.x;
        s2.y += x.y;
        ++k;
      }
    }
    {                                                 // periodic bond (bit N-1, bit 0)
      const bool anti = (((r >> (N - 1)) ^ r) & 1) != 0;
      cplx x = make_double2(0.0, 0.0);
      if (N <= 5) {
        const cplx t = shfl_xor_c(wi, (1 << (N - 1)) | 1);
        if (anti) x = t;
      } else if (anti) {
        x = w_in[r ^ (((int64_t)1 << (N - 1)) | 1)];
      }
      s2.x += x.x;
      s2.y += x.y;
      k += anti;
    }
    if (valid) {
      const double dg = op.jz * (double)(N - 2 * k);
      cplx y;
      y.x = fma(op.asingle, s1.x, fma(op.apair, s2.x, dg * wi.x));
      y.y = fma(op.asingle, s1.y, fma(op.apair, s2.y, dg * wi.y));
      cplx wn;
      wn.x = inv_gamma * y.x - shift * wi.x;
      wn.y = inv_gamma * y.y - shift * wi.y;
      cplx pi = p[r];
      cfma(pi, dk, wn);
      w_out[r] = wn;
      p[r] = pi;
      sw += wn.x * wn.x + wn.y * wn.y;
      sp += pi.x * pi.x + pi.y * pi.y;
    }
  }
  block_reduce_sum2<256>(sw, sp);
  if (threadIdx.x == 0) {
    partials[2 * blockIdx.x] = sw;
    partials[2 * blockIdx.x + 1] = sp;
  }
  if (last_block_ticket(ticket)) leja_finalize_warp0(partials, gridDim.x, abs_dk, tol, false, status);   // S7
}

}  // namespace

int launch_xxz_leja_iter(const XxzOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma, double shift,
                         cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st) {
  const int64_t n = (int64_t)1 << op.nspins;
  int64_t g = (n + 255) / 256;
  const int64_t cap = (int64_t)device_sm_count() * 8;
  if (g > cap) g = cap;
  xxz_leja_iter_kernel<<<(int)g, 256, 0, st>>>(op, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws->status,
                                               ws->partials, ws->tickets);
  ws->launches += 1;
  return (int)g;
}

// Gershgorin bounds of H0 + g H1 (c4) in closed form: a row with k antiparallel bonds has the centre jz (N - 2k)
// and the radius 2 |jxy| k + |g hx| N; on a ring k is even and at most N (N even) or N - 1 (N odd).
void xxz_gershgorin(const XxzOp& op, double* a, double* b) {
  const int N = op.nspins;
  double lo = INFINITY, hi = -INFINITY;
  for (int k = 0; k <= N; k += 2) {
    const double c = op.jz * (double)(N - 2 * k), r = std::fabs(op.apair) * (double)k + std::fabs(op.asingle) * (double)N;
    lo = std::fmin(lo, c - r);
    hi = std::fmax(hi, c + r);
  }
  *a = lo;
  *b = hi;
}

}  // namespace magnus
