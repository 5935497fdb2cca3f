// S6 -- fused Leja iteration, CSR "row-block" kernel tuned for the spin-chain
// structure (about N+1 stored entries per row, column = row XOR a small set of
// masks), but valid for any CSR matrix.
//
// Problem with the textbook mappings on this structure: lanes-along-a-row reads
// the matrix coalesced but gathers w from 32 different cache lines per
// instruction (one L1 wavefront per stored entry, which is slower than HBM can
// deliver the matrix); one-thread-per-row gathers w coalesced (32 consecutive
// rows with the same XOR mask touch 512 contiguous bytes) but reads the matrix
// with a row-length stride.  This kernel does both coalesced:
//   1. a warp owns 32 consecutive rows; their entries are one contiguous range of
//      the CSR arrays, which the warp streams HBM -> shared memory with 16-byte
//      cp.async (values) and 4-byte cp.async (columns), L2 evict-first;
//   2. the shared-memory slot of entry e is e + e/8 (one 16-byte pad every
//      128 bytes), so that the row-strided reads of step 3 spread over the banks;
//   3. lane l walks row r0+l out of shared memory and gathers w[col] from
//      global/L1 -- for equal slot numbers the 32 lanes hit one or a few aligned
//      512-byte segments;
//   4. the lane finishes its row: w+ = inv_gamma*y - shift*w, p += d_k w+, and
//      accumulates |w+|^2, |p|^2 (coalesced 16-byte accesses).
// Deterministic: fixed row->warp map, sequential sum along a row, fixed trees.
#include "magnus_internal.h"
#include "device_utils.cuh"
#include "leja_finalize.cuh"

namespace magnus {

namespace {

constexpr int RB_WARPS = 4;                     // warps per CTA
constexpr int RB_CAP = 768;                     // entries per warp staging buffer
constexpr int RB_SLOTS = RB_CAP + RB_CAP / 8;   // padded
constexpr int RB_BYTES_PER_WARP = RB_SLOTS * (int)(sizeof(cplx) + sizeof(int32_t));
constexpr int RB_SMEM = RB_WARPS * RB_BYTES_PER_WARP;
constexpr int RB_UNROLL = 8;

// POL  1: p and w+ move with an L2 evict-first hint (they are streamed once per launch and never gathered), so
//         that of all the traffic only w competes for L2 residency (n large: w itself exceeds L2)
// TB    the 32-row blocks are visited in an order that interleaves 2^TB contiguous chunks of the row range:
//         partners of a row under a flip of one of the top TB index bits are then in flight at the same time
// PIPE  1: the gathers of the next batch of RB_UNROLL entries are issued before the FMAs of the current one
template <int POL, int TB, int PIPE>
__global__ void __launch_bounds__(RB_WARPS * 32, 3)
    csr_leja_iter_rowblock_kernel(CsrOp op, const cplx* __restrict__ w_in, cplx* __restrict__ w_out,
                                  cplx* __restrict__ p, double inv_gamma, double shift, cplx dk,
                                  double abs_dk, double tol, LejaStatus* status, double* partials,
                                  unsigned* ticket) {
  if (status->done) return;
  extern __shared__ __align__(16) unsigned char rb_smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  cplx* sv = reinterpret_cast<cplx*>(rb_smem + (size_t)warp * RB_BYTES_PER_WARP);
  int32_t* sc = reinterpret_cast<int32_t*>(sv + RB_SLOTS);
  const uint64_t pol = policy_evict_first();
  const int64_t n = op.n;
  const int64_t nblocks = (n + 31) >> 5;
  const int64_t chunk = (nblocks + (1 << TB) - 1) >> TB;      // blocks per interleaved chunk
  const int64_t nslots = chunk << TB;
  const int64_t total_warps = (int64_t)gridDim.x * RB_WARPS;
  double sw = 0.0, sp = 0.0;

  for (int64_t slot = (int64_t)blockIdx.x * RB_WARPS + warp; slot < nslots; slot += total_warps) {
    const int64_t blk = TB == 0 ? slot : (slot & ((1 << TB) - 1)) * chunk + (slot >> TB);
    if (blk >= nblocks) continue;
    const int64_t row = (blk << 5) + lane;
    const bool valid = row < n;
    cplx y = make_double2(0.0, 0.0);
    // issued now, consumed after the last term: row pointers of every term and this row's w, p
    // (round-1 ncu: 20 % of the stall samples were these dependent loads)
    int rs_t[3], re_t[3];
#pragma unroll
    for (int t = 0; t < 3; ++t) {
      rs_t[t] = re_t[t] = 0;
      if (t < op.nterms) {
        rs_t[t] = op.t[t].rp[valid ? row : n];
        re_t[t] = op.t[t].rp[valid ? row + 1 : n];
      }
    }
    cplx wi = make_double2(0.0, 0.0), pi = make_double2(0.0, 0.0);
    if (valid) {
      wi = w_in[row];
      pi = POL ? ld_hint(p + row, pol) : p[row];
    }
#pragma unroll
    for (int t = 0; t < 3; ++t) {
      if (t >= op.nterms) break;
      const int32_t* __restrict__ ci = op.t[t].ci;
      const cplx* __restrict__ vv = op.t[t].v;
      const int rs = rs_t[t];
      const int re = re_t[t];
      cplx a = make_double2(0.0, 0.0);
      int first = 0;   // first lane (row) of the block not yet consumed
      while (first < 32) {
        const int base = __shfl_sync(0xffffffffu, rs, first);
        const bool fits = (re - base) <= RB_CAP;            // monotone in the lane: re ascends
        const unsigned nofit = ~__ballot_sync(0xffffffffu, fits || lane < first);
        const int last = nofit ? (__ffs(nofit) - 1) : 32;   // first lane whose row does not fit any more
        if (last == first) {
          // one row longer than the staging buffer: the whole warp strides over it
          const int e0 = base, e1 = __shfl_sync(0xffffffffu, re, first);
          cplx b = make_double2(0.0, 0.0);
          for (int q = e0 + lane; q < e1; q += 32) cfma(b, ld_stream(vv + q, pol), w_in[ld_stream_i32(ci + q, pol)]);
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) {
            b.x += shfl_xor_d(b.x, o);
            b.y += shfl_xor_d(b.y, o);
          }
          if (lane == first) {
            a.x += b.x;
            a.y += b.y;
          }
          first += 1;
          continue;
        }
        const int len = __shfl_sync(0xffffffffu, re, last - 1) - base;
        for (int e = lane; e < len; e += 32) {
          const int s = rb_slot(e);
          cp_async16(sv + s, vv + base + e, pol);
          cp_async4(sc + s, ci + base + e, pol);
        }
        cp_async_wait_all();
        __syncwarp();
        const bool mine = lane >= first && lane < last;
        const int qs = rs - base;
        const int mylen = mine ? re - rs : 0;
        const int maxlen = __reduce_max_sync(0xffffffffu, mylen);
        const int64_t safe = valid ? row : 0;
        if (PIPE) {
          // two batches in flight: gathers of batch b+1 are requested before batch b is consumed
          cplx xa[RB_UNROLL], xb[RB_UNROLL];
#pragma unroll
          for (int u = 0; u < RB_UNROLL; ++u) {
            const bool ok = u < mylen;
            xa[u] = w_in[ok ? (int64_t)sc[rb_slot(qs + u)] : safe];
          }
          for (int j = 0; j < maxlen; j += 2 * RB_UNROLL) {
#pragma unroll
            for (int u = 0; u < RB_UNROLL; ++u) {
              const bool ok = j + RB_UNROLL + u < mylen;
              xb[u] = w_in[ok ? (int64_t)sc[rb_slot(qs + j + RB_UNROLL + u)] : safe];
            }
#pragma unroll
            for (int u = 0; u < RB_UNROLL; ++u) {
              const bool ok = j + u < mylen;
              const cplx m = ok ? sv[rb_slot(qs + j + u)] : make_double2(0.0, 0.0);
              cfma(a, m, xa[u]);
            }
#pragma unroll
            for (int u = 0; u < RB_UNROLL; ++u) {
              const bool ok = j + 2 * RB_UNROLL + u < mylen;
              xa[u] = w_in[ok ? (int64_t)sc[rb_slot(qs + j + 2 * RB_UNROLL + u)] : safe];
            }
#pragma unroll
            for (int u = 0; u < RB_UNROLL; ++u) {
              const bool ok = j + RB_UNROLL + u < mylen;
              const cplx m = ok ? sv[rb_slot(qs + j + RB_UNROLL + u)] : make_double2(0.0, 0.0);
              cfma(a, m, xb[u]);
            }
          }
        } else {
          for (int j = 0; j < maxlen; j += RB_UNROLL) {
            cplx xv[RB_UNROLL], mv[RB_UNROLL];
#pragma unroll
            for (int u = 0; u < RB_UNROLL; ++u) {
              const bool ok = j + u < mylen;
              const int s = ok ? rb_slot(qs + j + u) : 0;
              mv[u] = ok ? sv[s] : make_double2(0.0, 0.0);
              const int64_t c = ok ? (int64_t)sc[s] : safe;
              xv[u] = w_in[c];
            }
#pragma unroll
            for (int u = 0; u < RB_UNROLL; ++u) cfma(a, mv[u], xv[u]);
          }
        }
        __syncwarp();   // everyone done reading before the buffer is refilled
        first = last;
      }
      const cplx ca = cmul(op.t[t].coef, a);
      y.x += ca.x;
      y.y += ca.y;
    }
    if (valid) {
      cplx wn;
      wn.x = inv_gamma * y.x - shift * wi.x;
      wn.y = inv_gamma * y.y - shift * wi.y;
      cfma(pi, dk, wn);
      if (POL) {
        st_hint(w_out + row, wn, pol);
        st_hint(p + row, pi, pol);
      } else {
        w_out[row] = wn;
        p[row] = pi;
      }
      sw += wn.x * wn.x + wn.y * wn.y;
      sp += pi.x * pi.x + pi.y * pi.y;
    }
  }
  block_reduce_sum2<RB_WARPS * 32>(sw, sp);
  if (threadIdx.x == 0) {
    partials[2 * blockIdx.x] = sw;
    partials[2 * blockIdx.x + 1] = sp;
  }
  if (last_block_ticket(ticket)) leja_finalize_warp0(partials, gridDim.x, abs_dk, tol, false, status);   // S7
}

template <int POL, int TB, int PIPE>
int launch_variant(const CsrOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma, double shift, cplx dk,
                   double abs_dk, double tol, Workspace* ws, cudaStream_t st) {
  auto kern = csr_leja_iter_rowblock_kernel<POL, TB, PIPE>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, RB_SMEM) != cudaSuccess) return -1;
  const int64_t nblocks = (op.n + 31) >> 5;
  int64_t g = (nblocks + RB_WARPS - 1) / RB_WARPS;
  const int64_t cap = (int64_t)device_sm_count() * 3;
  if (g > cap) g = cap;
  kern<<<(int)g, RB_WARPS * 32, RB_SMEM, st>>>(op, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws->status,
                                               ws->partials, ws->tickets);
  ws->launches += 1;
  return (int)g;
}

}  // namespace

bool csr_rowblock_supported(const CsrOp& op) { return op.n >= 32768; }

int launch_csr_leja_iter_rowblock(const CsrOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma,
                                  double shift, cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st) {
#define RB_ARGS op, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws, st
  switch (ws->csr_kernel) {   // experimental variants (round-2 sweep): 1000 + 100 POL + 10 TB + PIPE
    case 1001: return launch_variant<0, 0, 1>(RB_ARGS);
    case 1100: return launch_variant<1, 0, 0>(RB_ARGS);
    case 1101: return launch_variant<1, 0, 1>(RB_ARGS);
    case 1020: return launch_variant<0, 2, 0>(RB_ARGS);
    case 1120: return launch_variant<1, 2, 0>(RB_ARGS);
    case 1130: return launch_variant<1, 3, 0>(RB_ARGS);
    case 1140: return launch_variant<1, 4, 0>(RB_ARGS);
    case 1121: return launch_variant<1, 2, 1>(RB_ARGS);
    case 1131: return launch_variant<1, 3, 1>(RB_ARGS);
    case 1141: return launch_variant<1, 4, 1>(RB_ARGS);
    default: return launch_variant<0, 0, 0>(RB_ARGS);
  }
#undef RB_ARGS
}

}  // namespace magnus
