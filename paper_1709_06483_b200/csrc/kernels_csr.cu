// CSR kernels: Gershgorin bounds of M = sum_t coef_t A_t (row S3), the fused
// Leja iteration (row S6) and the setup-time sparse commutator (row S0).
// P:n = PAPER.md line n; c1..c7 = readings in DESIGN.md section 3.
#include "magnus_internal.h"
#include "device_utils.cuh"
#include "leja_finalize.cuh"

#include <cub/device/device_scan.cuh>
#include <limits.h>

namespace magnus {

// ---------------------------------------------------------------------------
// S3 -- Gershgorin bounds ("an estimate on the spectrum of the matrix"; c4):
// lo_i = Re M_ii - R_i, hi_i = Re M_ii + R_i, R_i = sum_{j != i} |M_ij| with
// M_ij the SUMMED entry over the terms.  One thread walks one row with a k-way
// merge over the (ascending) column lists, so overlapping patterns are summed
// before the modulus is taken.  Block min/max go to ws->gersh.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256) csr_gershgorin_kernel(CsrOp op, double* out, unsigned* ticket, double* fin) {
  double lo = INFINITY, hi = -INFINITY;
  for (int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; row < op.n;
       row += (int64_t)gridDim.x * blockDim.x) {
    int q[3], e[3];
#pragma unroll
    for (int t = 0; t < 3; ++t) {
      q[t] = t < op.nterms ? op.t[t].rp[row] : 0;
      e[t] = t < op.nterms ? op.t[t].rp[row + 1] : 0;
    }
    double R = 0.0, d = 0.0;
    while (true) {
      int c = INT_MAX;
#pragma unroll
      for (int t = 0; t < 3; ++t)
        if (t < op.nterms && q[t] < e[t]) c = min(c, op.t[t].ci[q[t]]);
      if (c == INT_MAX) break;
      cplx z = make_double2(0.0, 0.0);
#pragma unroll
      for (int t = 0; t < 3; ++t)
        if (t < op.nterms && q[t] < e[t] && op.t[t].ci[q[t]] == c) {
          const cplx prod = cmul(op.t[t].coef, op.t[t].v[q[t]]);
          z.x += prod.x;
          z.y += prod.y;
          ++q[t];
        }
      if ((int64_t)c == row) d = z.x; else R += cabs_fast(z);
    }
    lo = fmin(lo, d - R);
    hi = fmax(hi, d + R);
  }
  block_reduce_minmax<256>(lo, hi);
  if (threadIdx.x == 0) {
    out[2 * blockIdx.x] = lo;
    out[2 * blockIdx.x + 1] = hi;
  }
  if (last_block_ticket(ticket)) minmax_finalize_warp0(out, gridDim.x, fin);
}

// The same bounds for large n with every access coalesced: a warp owns 32 consecutive rows,
// streams the contiguous entry ranges of ALL terms for those rows into shared memory with
// cp.async (as the row-block Leja kernel does for one term), then lane l runs the same k-way
// merge as above over row l out of shared memory.  Same arithmetic and summation order as
// csr_gershgorin_kernel.  A row block whose entries do not fit the buffer is merged straight
// from global memory.
const int GS_WARPS = 6;
const int GS_CAP = 1600;                    // staged entries per warp, all terms together
const int GS_SLOTS = GS_CAP + GS_CAP / 8;
const int GS_BYTES_PER_WARP = GS_SLOTS * (int)(sizeof(cplx) + sizeof(int32_t));
const int GS_SMEM = GS_WARPS * GS_BYTES_PER_WARP;

__global__ void __launch_bounds__(GS_WARPS * 32, 1) csr_gershgorin_staged_kernel(CsrOp op, double* out, unsigned* ticket,
                                                                                 double* fin) {
  extern __shared__ __align__(16) unsigned char gs_smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  cplx* sv = reinterpret_cast<cplx*>(gs_smem + (size_t)warp * GS_BYTES_PER_WARP);
  int32_t* sc = reinterpret_cast<int32_t*>(sv + GS_SLOTS);
  const uint64_t pol = policy_evict_first();
  const int64_t n = op.n;
  const int64_t nblocks = (n + 31) >> 5;
  const int64_t total_warps = (int64_t)gridDim.x * GS_WARPS;
  double lo = INFINITY, hi = -INFINITY;
  for (int64_t blk = (int64_t)blockIdx.x * GS_WARPS + warp; blk < nblocks; blk += total_warps) {
    const int64_t row = (blk << 5) + lane;
    const bool valid = row < n;
    int rs[3], re[3], base[3], off[3];
    int total = 0;
#pragma unroll
    for (int t = 0; t < 3; ++t) {
      rs[t] = re[t] = base[t] = off[t] = 0;
      if (t < op.nterms) {
        rs[t] = op.t[t].rp[valid ? row : n];
        re[t] = op.t[t].rp[valid ? row + 1 : n];
        base[t] = __shfl_sync(0xffffffffu, rs[t], 0);
        off[t] = total;
        total += __shfl_sync(0xffffffffu, re[t], 31) - base[t];
      }
    }
    const bool staged = total <= GS_CAP;
    if (staged) {
#pragma unroll
      for (int t = 0; t < 3; ++t) {
        if (t < op.nterms) {
          const int len = (t + 1 < op.nterms ? off[t + 1] : total) - off[t];
          const cplx* __restrict__ vv = op.t[t].v + base[t];
          const int32_t* __restrict__ ci = op.t[t].ci + base[t];
          for (int e = lane; e < len; e += 32) {
            const int s = rb_slot(off[t] + e);
            cp_async16(sv + s, vv + e, pol);
            cp_async4(sc + s, ci + e, pol);
          }
        }
      }
      cp_async_wait_all();
      __syncwarp();
    }
    int q[3], e[3];
#pragma unroll
    for (int t = 0; t < 3; ++t) {
      q[t] = staged ? off[t] + rs[t] - base[t] : rs[t];
      e[t] = staged ? off[t] + re[t] - base[t] : re[t];
    }
    double R = 0.0, d = 0.0;
    while (true) {
      int c = INT_MAX;
      int cc[3];
#pragma unroll
      for (int t = 0; t < 3; ++t) {
        cc[t] = INT_MAX;
        if (t < op.nterms && q[t] < e[t]) cc[t] = staged ? sc[rb_slot(q[t])] : op.t[t].ci[q[t]];
        c = min(c, cc[t]);
      }
      if (c == INT_MAX) break;
      cplx z = make_double2(0.0, 0.0);
#pragma unroll
      for (int t = 0; t < 3; ++t)
        if (cc[t] == c) {
          const cplx v = staged ? sv[rb_slot(q[t])] : op.t[t].v[q[t]];
          const cplx prod = cmul(op.t[t].coef, v);
          z.x += prod.x;
          z.y += prod.y;
          ++q[t];
        }
      if ((int64_t)c == row) d = z.x; else R += cabs_fast(z);
    }
    if (staged) __syncwarp();   // everyone done reading before the buffer is refilled
    if (valid) {
      lo = fmin(lo, d - R);
      hi = fmax(hi, d + R);
    }
  }
  block_reduce_minmax<GS_WARPS * 32>(lo, hi);
  if (threadIdx.x == 0) {
    out[2 * blockIdx.x] = lo;
    out[2 * blockIdx.x + 1] = hi;
  }
  if (last_block_ticket(ticket)) minmax_finalize_warp0(out, gridDim.x, fin);
}

int launch_csr_gershgorin(const CsrOp& op, Workspace* ws, cudaStream_t st) {
  if (op.n >= 32768) {
    // per launch (cheap): the attribute is per device, a process-wide flag would miss a second GPU
    cudaFuncSetAttribute(csr_gershgorin_staged_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, GS_SMEM);
    const int sms = device_sm_count();
    csr_gershgorin_staged_kernel<<<sms, GS_WARPS * 32, GS_SMEM, st>>>(op, ws->gersh, ws->tickets + 1, gersh_final(ws));
    ws->launches += 1;
    return sms;
  }
  int64_t g = (op.n + 255) / 256;
  if (g > (int64_t)device_sm_count() * 8) g = (int64_t)device_sm_count() * 8;
  csr_gershgorin_kernel<<<(int)g, 256, 0, st>>>(op, ws->gersh, ws->tickets + 1, gersh_final(ws));
  ws->launches += 1;
  return (int)g;
}

// ---------------------------------------------------------------------------
// S3 with cached row statistics.  When no column of a row is stored in more than one term
// (checked once at magnus_create by csr_terms_disjoint), the modulus of the summed entry
// separates, |sum_t c_t v_t| = |c_t| |v_t| for the one term that holds it, so
//   R_i = sum_t |c_t| r_i^t,  r_i^t = sum_{j != i} |A_t,ij|;   Re M_ii = sum_t Re(c_t A_t,ii)
// and the bounds of every exponential follow from the per-term vectors r^t, diag^t (computed
// once) in one pass over 24 n bytes per term instead of the whole matrix.  Same quantity as
// csr_gershgorin_kernel up to summation order, which the interval snapping (c4) absorbs.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256) csr_rowstats_kernel(CsrTerm T, int64_t n, double* __restrict__ r,
                                                            cplx* __restrict__ diag) {
  for (int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; row < n; row += (int64_t)gridDim.x * blockDim.x) {
    double R = 0.0;
    cplx d = make_double2(0.0, 0.0);
    for (int q = T.rp[row]; q < T.rp[row + 1]; ++q) {
      const cplx v = T.v[q];
      if ((int64_t)T.ci[q] == row) d = v; else R += cabs_fast(v);
    }
    r[row] = R;
    diag[row] = d;
  }
}

// flag |= 1 if some (row, column) is stored in more than one of the terms
__global__ void __launch_bounds__(256) csr_overlap_kernel(CsrOp op, int* __restrict__ flag) {
  bool hit = false;
  for (int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; row < op.n;
       row += (int64_t)gridDim.x * blockDim.x) {
    int q[3], e[3];
#pragma unroll
    for (int t = 0; t < 3; ++t) {
      q[t] = t < op.nterms ? op.t[t].rp[row] : 0;
      e[t] = t < op.nterms ? op.t[t].rp[row + 1] : 0;
    }
    while (true) {
      int c = INT_MAX;
#pragma unroll
      for (int t = 0; t < 3; ++t)
        if (t < op.nterms && q[t] < e[t]) c = min(c, op.t[t].ci[q[t]]);
      if (c == INT_MAX) break;
      int cnt = 0;
#pragma unroll
      for (int t = 0; t < 3; ++t)
        if (t < op.nterms && q[t] < e[t] && op.t[t].ci[q[t]] == c) {
          ++cnt;
          ++q[t];
        }
      hit |= cnt > 1;
    }
  }
  if (hit) atomicOr(flag, 1);
}

struct RowStats {
  const double* r[3];
  const cplx* diag[3];
  cplx coef[3];
  int nterms;
};

__global__ void __launch_bounds__(256) csr_gershgorin_cached_kernel(RowStats S, int64_t n, double* out,
                                                                     unsigned* ticket, double* fin) {
  double lo = INFINITY, hi = -INFINITY;
  double ac[3];
#pragma unroll
  for (int t = 0; t < 3; ++t) ac[t] = t < S.nterms ? cabs_fast(S.coef[t]) : 0.0;
  for (int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; row < n; row += (int64_t)gridDim.x * blockDim.x) {
    double R = 0.0, d = 0.0;
#pragma unroll
    for (int t = 0; t < 3; ++t)
      if (t < S.nterms) {
        const cplx dg = S.diag[t][row];
        R = fma(ac[t], S.r[t][row], R);
        d += S.coef[t].x * dg.x - S.coef[t].y * dg.y;
      }
    lo = fmin(lo, d - R);
    hi = fmax(hi, d + R);
  }
  block_reduce_minmax<256>(lo, hi);
  if (threadIdx.x == 0) {
    out[2 * blockIdx.x] = lo;
    out[2 * blockIdx.x + 1] = hi;
  }
  if (last_block_ticket(ticket)) minmax_finalize_warp0(out, gridDim.x, fin);
}

static int row_grid256(int64_t n) {
  int64_t g = (n + 255) / 256;
  if (g > (int64_t)device_sm_count() * 8) g = (int64_t)device_sm_count() * 8;
  return (int)g;
}

void launch_csr_rowstats(const CsrTerm& T, int64_t n, double* r, cplx* diag, cudaStream_t st) {
  csr_rowstats_kernel<<<row_grid256(n), 256, 0, st>>>(T, n, r, diag);
}

void launch_csr_overlap(const CsrOp& op, int* flag, cudaStream_t st) {
  csr_overlap_kernel<<<row_grid256(op.n), 256, 0, st>>>(op, flag);
}

int launch_csr_gershgorin_cached(const CsrOp& op, const double* const* r, const cplx* const* diag, Workspace* ws,
                                 cudaStream_t st) {
  RowStats S;
  S.nterms = op.nterms;
  for (int t = 0; t < 3; ++t) {
    S.r[t] = r[t < op.nterms ? t : 0];
    S.diag[t] = diag[t < op.nterms ? t : 0];
    S.coef[t] = op.t[t < op.nterms ? t : 0].coef;
  }
  const int g = row_grid256(op.n);
  csr_gershgorin_cached_kernel<<<g, 256, 0, st>>>(S, op.n, ws->gersh, ws->tickets + 1, gersh_final(ws));
  ws->launches += 1;
  return g;
}

// The same bounds for a whole planned batch in ONE launch: block e takes exponential e, whose term
// coefficients are (1, g_e, -i kappa_e) = coefs[4e], coefs[4e+1], nterms = (int)coefs[4e+2].  Small n only
// (a block walks all rows); the arithmetic per row is that of csr_gershgorin_cached_kernel.
__global__ void __launch_bounds__(256) csr_gershgorin_cached_batch_kernel(RowStats S, int64_t n,
                                                                           const double* __restrict__ coefs,
                                                                           double* __restrict__ ab_out) {
  const int e = blockIdx.x;
  const double g = coefs[4 * e], kappa = coefs[4 * e + 1];
  const int nterms = (int)coefs[4 * e + 2];
  cplx coef[3] = {make_double2(1.0, 0.0), make_double2(g, 0.0), make_double2(0.0, -kappa)};
  double ac[3];
#pragma unroll
  for (int t = 0; t < 3; ++t) ac[t] = t < nterms ? cabs_fast(coef[t]) : 0.0;
  double lo = INFINITY, hi = -INFINITY;
  for (int64_t row = threadIdx.x; row < n; row += blockDim.x) {
    double R = 0.0, d = 0.0;
#pragma unroll
    for (int t = 0; t < 3; ++t)
      if (t < nterms) {
        const cplx dg = S.diag[t][row];
        R = fma(ac[t], S.r[t][row], R);
        d += coef[t].x * dg.x - coef[t].y * dg.y;
      }
    lo = fmin(lo, d - R);
    hi = fmax(hi, d + R);
  }
  block_reduce_minmax<256>(lo, hi);
  if (threadIdx.x == 0) {
    ab_out[2 * e] = lo;
    ab_out[2 * e + 1] = hi;
  }
}

void launch_csr_gershgorin_cached_batch(int64_t n, const double* const* r, const cplx* const* diag, int nterms_max,
                                        const double* coefs_dev, int E, double* ab_out, Workspace* ws, cudaStream_t st) {
  RowStats S;
  S.nterms = nterms_max;
  for (int t = 0; t < 3; ++t) {
    S.r[t] = r[t < nterms_max ? t : 0];
    S.diag[t] = diag[t < nterms_max ? t : 0];
    S.coef[t] = make_double2(0.0, 0.0);
  }
  csr_gershgorin_cached_batch_kernel<<<E, 256, 0, st>>>(S, n, coefs_dev, ab_out);
  ws->launches += 1;
}

// ---------------------------------------------------------------------------
// S6 -- fused Leja iteration, generic kernel (any CSR): G lanes share one row.
//   y_i   = sum_t coef_t sum_q A_t.v[q] w[A_t.ci[q]]            (SpMV of H(t) formed on the fly)
//   w+_i  = inv_gamma y_i - shift w_i                            (fragment line 4; c5)
//   p_i  += d_k w+_i                                             (fragment line 5)
//   block partials of sum |w+|^2 and sum |p|^2                  (for S7)
// Lanes of a row read consecutive 16-byte values (coalesced 128-bit loads with
// L1 no-allocate / L2 evict-first), reduce with a shuffle tree, lane 0 does the
// vector update.  Deterministic: fixed lane->entry map and fixed trees.
// ---------------------------------------------------------------------------
template <int G>
__global__ void __launch_bounds__(256) csr_leja_iter_generic(CsrOp op, const cplx* __restrict__ w_in,
                                                              cplx* __restrict__ w_out, cplx* __restrict__ p,
                                                              double inv_gamma, double shift, cplx dk,
                                                              double abs_dk, double tol, LejaStatus* status,
                                                              double* partials, unsigned* ticket) {
  if (status->done) return;
  constexpr int ROWS = 256 / G;
  const int sub = threadIdx.x % G;
  const int rib = threadIdx.x / G;
  const uint64_t pol = policy_evict_first();
  double sw = 0.0, sp = 0.0;
  for (int64_t base = (int64_t)blockIdx.x * ROWS; base < op.n; base += (int64_t)gridDim.x * ROWS) {
    const int64_t row = base + rib;
    const bool valid = row < op.n;
    cplx y = make_double2(0.0, 0.0);
#pragma unroll
    for (int t = 0; t < 3; ++t) {
      if (t < op.nterms) {
        const CsrTerm& T = op.t[t];
        int qs = 0, qe = 0;
        if (valid) {
          qs = T.rp[row];
          qe = T.rp[row + 1];
        }
        cplx a = make_double2(0.0, 0.0);
        for (int q = qs + sub; q < qe; q += G) {
          const cplx v = ld_stream(T.v + q, pol);
          const int c = ld_stream_i32(T.ci + q, pol);
          const cplx x = w_in[c];
          cfma(a, v, x);
        }
        const cplx ca = cmul(T.coef, a);
        y.x += ca.x;
        y.y += ca.y;
      }
    }
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) {
      y.x += shfl_xor_d(y.x, o);
      y.y += shfl_xor_d(y.y, o);
    }
    if (valid && sub == 0) {
      const cplx wi = w_in[row];
      cplx wn;
      wn.x = inv_gamma * y.x - shift * wi.x;
      wn.y = inv_gamma * y.y - shift * wi.y;
      w_out[row] = wn;
      cplx pi = p[row];
      cfma(pi, dk, wn);
      p[row] = pi;
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

template <int G>
static int launch_generic(const CsrOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma, double shift,
                          cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st) {
  constexpr int ROWS = 256 / G;
  int64_t g = (op.n + ROWS - 1) / ROWS;
  if (g > (int64_t)device_sm_count() * 8) g = (int64_t)device_sm_count() * 8;
  csr_leja_iter_generic<G><<<(int)g, 256, 0, st>>>(op, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol,
                                                    ws->status, ws->partials, ws->tickets);
  ws->launches += 1;
  return (int)g;
}

int launch_csr_leja_iter_rowblock(const CsrOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma,
                                  double shift, cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st);
bool csr_rowblock_supported(const CsrOp& op);

int launch_csr_leja_iter(const CsrOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma, double shift,
                         cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st) {
  if (op.slice && (ws->csr_kernel == 0 || slice_layout_kind(ws->csr_kernel) != 0))
    return launch_csr_leja_iter_slice(op, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws, st);
  if (ws->csr_kernel == 4 && csr_rowtma_supported(op)) {
    const int g = launch_csr_leja_iter_rowtma(op, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws, st);
    if (g > 0) return g;
  }
  if ((ws->csr_kernel == 3 || (ws->csr_kernel >= 20000 && ws->csr_kernel < 30000)) && csr_stream_supported(op)) {
    const int g = launch_csr_leja_iter_stream(op, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws, st);
    if (g > 0) return g;
  }
  if (ws->csr_kernel == 2 || ws->csr_kernel >= 1000 || (ws->csr_kernel == 0 && csr_rowblock_supported(op)))
    return launch_csr_leja_iter_rowblock(op, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws, st);
  // lanes per row from the mean stored entries per row and term
  double mean = 0.0;
  for (int t = 0; t < op.nterms; ++t) mean += (double)op.t[t].nnz;
  mean /= (double)op.n * (double)op.nterms;
  if (mean > 48.0) return launch_generic<32>(op, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws, st);
  if (mean > 24.0) return launch_generic<16>(op, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws, st);
  if (mean > 6.0) return launch_generic<8>(op, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws, st);
  if (mean > 3.0) return launch_generic<4>(op, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws, st);
  return launch_generic<2>(op, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws, st);
}

// ---------------------------------------------------------------------------
// S0 -- sparse commutator C = A B - B A at setup time ("the commutators
// ... are computed directly on the device"; P:262 l.6-8).  One block per row:
// expand all products a_ik b_kj and -b_ik a_kj into shared memory, bitonic-sort
// by column, sum equal columns in sorted order, drop exact zeros.  Pass 1
// counts, an exclusive scan gives row_ptr, pass 2 writes.
// ---------------------------------------------------------------------------
const int kCommCap = 2048;     // candidate products per row held in shared memory
const int kCommThreads = 128;

struct CsrRaw {
  const int32_t* rp;
  const int32_t* ci;
  const cplx* v;
};

__device__ __forceinline__ void comm_expand(const CsrRaw& A, const CsrRaw& B, int64_t row, double sign, int* keys,
                                            cplx* vals, int& base, int* overflow) {
  // += sign * sum_k A(row,k) B(k,:)
  const int ps = A.rp[row], pe = A.rp[row + 1];
  for (int pp = ps; pp < pe; ++pp) {
    const int k = A.ci[pp];
    const cplx a = A.v[pp];
    const int qs = B.rp[k], len = B.rp[k + 1] - qs;
    if (base + len > kCommCap) {
      if (threadIdx.x == 0) *overflow = 1;
      base = kCommCap + 1;
      return;
    }
    for (int t = threadIdx.x; t < len; t += kCommThreads) {
      const cplx b = B.v[qs + t];
      cplx prod = cmul(a, b);
      prod.x *= sign;
      prod.y *= sign;
      keys[base + t] = B.ci[qs + t];
      vals[base + t] = prod;
    }
    base += len;
  }
}

// Bitonic sorting network over 32 R keys held R per lane (element e = lane R + r), ascending.  Strides below R
// are compare-exchanges between registers of a lane, the others exchange with lane ^ (stride / R) by shuffle;
// everything is unrolled at compile time, so the network touches no memory.
template <int R, typename T>
__device__ __forceinline__ void warp_bitonic_sort(T (&k)[R], int lane) {
#pragma unroll
  for (int size = 2; size <= 32 * R; size <<= 1) {
#pragma unroll
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      if (stride < R) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
          if (r & stride) continue;
          const bool asc = size < R ? (r & size) == 0 : (lane & (size / R)) == 0;   // size == 32 R: always ascending
          const T a = k[r], b = k[r | stride];
          const T lo = a < b ? a : b, hi = a < b ? b : a;
          k[r] = asc ? lo : hi;
          k[r | stride] = asc ? hi : lo;
        }
      } else {
        const int lm = stride / R;
        const bool lower = (lane & lm) == 0;
        const bool asc = (lane & (size / R)) == 0;
#pragma unroll
        for (int r = 0; r < R; ++r) {
          const T o = __shfl_xor_sync(0xffffffffu, k[r], lm);
          const bool take_min = lower == asc;
          k[r] = take_min ? (o < k[r] ? o : k[r]) : (o > k[r] ? o : k[r]);
        }
      }
    }
  }
}

// keys[0..total) of a warp: (column << 32 | position) -> the same, sorted; T = unsigned packs the key as
// column * 1024 + position for the network and unpacks it again
template <int R, typename T, bool DUMMY>
__device__ __forceinline__ void sort_keys(unsigned long long* skey, int total, int lane) {
  T k[R];
#pragma unroll
  for (int r = 0; r < R; ++r) {
    const int e = lane * R + r;
    if (e < total) {
      const unsigned long long full = skey[e];
      k[r] = sizeof(T) == 4 ? (T)(((unsigned)(full >> 32) << 10) | ((unsigned)full & 1023u)) : (T)full;
    } else {
      k[r] = (T)~(T)0;
    }
  }
  warp_bitonic_sort<R, T>(k, lane);
  __syncwarp();
#pragma unroll
  for (int r = 0; r < R; ++r) {
    const int e = lane * R + r;
    if (e < total)
      skey[e] = sizeof(T) == 4 ? (((unsigned long long)((unsigned)k[r] >> 10) << 32) | ((unsigned)k[r] & 1023u))
                               : (unsigned long long)k[r];
  }
}

// Row i of C = A B - B A is a linear combination of sparse rows: + a_ik B_k for the entries of A's row i and
// - b_ik A_k for those of B's row i, L = len A_i + len B_i source rows ("lists").  ONE WARP per row:
//   1. every lane looks up its lists (lane, lane + 32, ...) and a warp scan gives each list its place in a
//      per-warp candidate buffer in shared memory;
//   2. expand: the lane copies its lists there -- key = (column << 32) | position, value = +-coefficient times
//      entry -- all loads independent of one another;
//   3. the warp sorts the 64-bit keys with a bitonic network in REGISTERS (16 or 32 keys per lane, shuffles
//      between lanes, fully unrolled);
//   4. every lane takes a contiguous piece of the sorted keys, sums each run of equal columns that starts in
//      its piece IN POSITION ORDER (positions are unique, so the sorted order and therefore every sum is
//      fixed: the A-part in k order, then the B-part in k order), drops exact zeros, and a warp scan places
//      the survivors, which are already in column order.
// The spin chains need (N/2 + 1) N 2 candidates per row (624 at N = 24); a row with more than kSortCap
// candidates or more than kCommLists lists is left to the CTA-wide sorting kernel below.
// Two tiers of the warp kernel: candidate buffers of 512 entries for all rows (14 warps per SM), and of 1024 for the
// rows the first tier hands on through a second worklist (the chains' rows with many antiparallel bonds).
const int kCommLists = 256;
const int kMergeWarps = 2;
const int kSortCap = 1024;    // largest candidate buffer (second tier)
const int kCommTmp = 32;      // entries of a row of C the warp kernel parks in the temporary buffer
template <int CAP>
constexpr int merge_smem() { return kMergeWarps * (CAP * (int)(sizeof(cplx) + sizeof(unsigned long long)) + 3 * kCommLists * (int)sizeof(int)); }

// counts[row] = entries of row i of C; the entries themselves go to tmp_ci / tmp_v at row * kCommTmp (the gather
// kernel moves them to their CSR place once the row pointers are known).  A row this kernel does not take --
// too many lists, more than kSortCap candidates, or more than kCommTmp entries -- is appended to `work` (work[0] =
// how many) for the CTA-wide kernel; a row with more than CAP but at most kSortCap candidates to `work2` for the
// second tier.  FROM_LIST: the rows are those of `rows_in` (rows_in[0] = how many) instead of 0..n-1.
template <int CAP, bool FROM_LIST>
__global__ void __launch_bounds__(kMergeWarps * 32) csr_commutator_merge_kernel(CsrRaw A, CsrRaw B, int64_t n,
                                                                                int32_t* __restrict__ counts,
                                                                                int32_t* __restrict__ tmp_ci,
                                                                                cplx* __restrict__ tmp_v, int* work,
                                                                                int* work2, const int* rows_in) {
  constexpr bool WRITE = false;
  extern __shared__ __align__(16) unsigned char cm_smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  cplx* sval = reinterpret_cast<cplx*>(cm_smem) + warp * CAP;
  unsigned long long* skey = reinterpret_cast<unsigned long long*>(cm_smem + kMergeWarps * CAP * sizeof(cplx)) + warp * CAP;
  int* lq = reinterpret_cast<int*>(cm_smem + kMergeWarps * CAP * (sizeof(cplx) + sizeof(unsigned long long))) +
            warp * 3 * kCommLists;
  int* llen = lq + kCommLists;
  int* lo = llen + kCommLists;
  const int64_t nwarps = (int64_t)gridDim.x * kMergeWarps;
  const bool narrow = n <= ((int64_t)1 << 22);
  const int64_t nrows_todo = FROM_LIST ? rows_in[0] : n;
  for (int64_t it = (int64_t)blockIdx.x * kMergeWarps + warp; it < nrows_todo; it += nwarps) {
    const int64_t row = FROM_LIST ? rows_in[1 + it] : it;
    const int pa = A.rp[row], lenA = A.rp[row + 1] - pa, pb = B.rp[row], lenB = B.rp[row + 1] - pb;
    const int L = lenA + lenB;
    int total = 0;
    if (L <= kCommLists) {
      __syncwarp();
      for (int t0 = 0; t0 < L; t0 += 32) {               // 1. the lists and their places
        const int t = t0 + lane;
        int q = 0, len = 0;
        if (t < L) {
          const bool fromA = t < lenA;                   // + a_ik B_k  or  - b_ik A_k
          const int k = fromA ? A.ci[pa + t] : B.ci[pb + t - lenA];
          const CsrRaw& S = fromA ? B : A;
          q = S.rp[k];
          len = S.rp[k + 1] - q;
        }
        int inc = len;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
          const int up = __shfl_up_sync(0xffffffffu, inc, d);
          if (lane >= d) inc += up;
        }
        if (t < L) {
          lq[t] = q;
          llen[t] = len;
          lo[t] = total + inc - len;
        }
        total += __shfl_sync(0xffffffffu, inc, 31);
      }
    }
    if (L > kCommLists || total > kSortCap) {            // warp-uniform: the CTA-wide kernel takes this row
      if (lane == 0) {
        counts[row] = 0;
        work[1 + atomicAdd(work, 1)] = (int)row;
      }
      continue;
    }
    if (total > CAP) {                                   // warp-uniform: the second tier takes this row
      if (lane == 0) {
        counts[row] = 0;
        work2[1 + atomicAdd(work2, 1)] = (int)row;
      }
      continue;
    }
    __syncwarp();
    for (int t = lane; t < L; t += 32) {                 // 2. expand
      const bool fromA = t < lenA;
      const CsrRaw& S = fromA ? B : A;
      cplx coef = fromA ? A.v[pa + t] : B.v[pb + t - lenA];
      if (!fromA) {
        coef.x = -coef.x;
        coef.y = -coef.y;
      }
      const int q = lq[t], len = llen[t], o = lo[t];
#pragma unroll 4
      for (int j = 0; j < len; ++j) {
        skey[o + j] = ((unsigned long long)(unsigned)S.ci[q + j] << 32) | (unsigned)(o + j);
        sval[o + j] = cmul(coef, S.v[q + j]);
      }
    }
    __syncwarp();
    // 3. sort the keys: into registers (lane-contiguous), network, back to shared memory.  When column and
    // position fit 32 bits together (n * 1024 <= 2^32) the network runs on 32-bit keys (min / max per exchange).
    if (narrow) {
      if (CAP <= 16 * 32 || total <= 16 * 32) sort_keys<16, unsigned, WRITE>(skey, total, lane);
      else sort_keys<32, unsigned, WRITE>(skey, total, lane);
    } else {
      if (CAP <= 16 * 32 || total <= 16 * 32) sort_keys<16, unsigned long long, WRITE>(skey, total, lane);
      else sort_keys<32, unsigned long long, WRITE>(skey, total, lane);
    }
    __syncwarp();
    // 4. runs of equal columns; a lane owns the runs that start in its piece
    const int per = (total + 31) >> 5, s0 = min(total, lane * per), s1 = min(total, s0 + per);
    int cnt = 0;
    for (int p = s0; p < s1; ++p) {
      const unsigned c = (unsigned)(skey[p] >> 32);
      if (p > 0 && (unsigned)(skey[p - 1] >> 32) == c) continue;
      cplx z = sval[(unsigned)skey[p]];
      for (int u = p + 1; u < total && (unsigned)(skey[u] >> 32) == c; ++u) {
        const cplx y = sval[(unsigned)skey[u]];
        z.x += y.x;
        z.y += y.y;
      }
      if (z.x != 0.0 || z.y != 0.0) ++cnt;
    }
    int inc = cnt;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int up = __shfl_up_sync(0xffffffffu, inc, d);
      if (lane >= d) inc += up;
    }
    const int nrow = __shfl_sync(0xffffffffu, inc, 31);
    if (nrow > kCommTmp) {                               // warp-uniform
      if (lane == 0) {
        counts[row] = 0;
        work[1 + atomicAdd(work, 1)] = (int)row;
      }
      continue;
    }
    if (lane == 0) counts[row] = nrow;
    int o = inc - cnt;
    int32_t* oc = tmp_ci + row * kCommTmp;
    cplx* ov = tmp_v + row * kCommTmp;
    for (int p = s0; p < s1; ++p) {
      const unsigned c = (unsigned)(skey[p] >> 32);
      if (p > 0 && (unsigned)(skey[p - 1] >> 32) == c) continue;
      cplx z = sval[(unsigned)skey[p]];
      for (int u = p + 1; u < total && (unsigned)(skey[u] >> 32) == c; ++u) {
        const cplx y = sval[(unsigned)skey[u]];
        z.x += y.x;
        z.y += y.y;
      }
      if (z.x != 0.0 || z.y != 0.0) {
        oc[o] = (int)c;
        ov[o] = z;
        ++o;
      }
    }
  }
}

// rows the warp kernel finished: tmp -> CSR place (one warp per row)
__global__ void __launch_bounds__(256) csr_commutator_gather_kernel(int64_t n, const int32_t* __restrict__ counts,
                                                                     const int32_t* __restrict__ rp,
                                                                     const int32_t* __restrict__ tmp_ci,
                                                                     const cplx* __restrict__ tmp_v,
                                                                     int32_t* __restrict__ ci_out, cplx* __restrict__ v_out) {
  const int lane = threadIdx.x & 31;
  const int64_t row = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (row >= n) return;
  const int o = rp[row], len = rp[row + 1] - o;
  if (len > kCommTmp) return;   // a row of the CTA-wide kernel, which writes after this kernel (so does it for its
                                // shorter rows: what is copied here for them is overwritten)
  for (int j = lane; j < len; j += 32) {
    ci_out[o + j] = tmp_ci[row * kCommTmp + j];
    v_out[o + j] = tmp_v[row * kCommTmp + j];
  }
}

template <bool WRITE>
__global__ void __launch_bounds__(kCommThreads) csr_commutator_kernel(CsrRaw A, CsrRaw B, int64_t n,
                                                                       int32_t* __restrict__ counts,
                                                                       const int32_t* __restrict__ rp_out,
                                                                       int32_t* __restrict__ ci_out,
                                                                       cplx* __restrict__ v_out, int* overflow,
                                                                       const int* __restrict__ work) {
  __shared__ int keys[kCommCap];
  __shared__ cplx vals[kCommCap];
  __shared__ int scan[kCommThreads + 1];
  (void)n;
  const int nwork = work[0];                     // the rows the warp kernel left over
  for (int wi = blockIdx.x; wi < nwork; wi += gridDim.x) {
    const int64_t row = work[1 + wi];
    int total = 0;
    comm_expand(A, B, row, 1.0, keys, vals, total, overflow);
    if (total <= kCommCap) comm_expand(B, A, row, -1.0, keys, vals, total, overflow);
    if (total > kCommCap) {   // row too dense for the shared-memory path: flagged, host reports EINVAL
      if (!WRITE && threadIdx.x == 0) counts[row] = 0;
      __syncthreads();
      continue;
    }
    int cap = 1;
    while (cap < total) cap <<= 1;
    for (int t = total + threadIdx.x; t < cap; t += kCommThreads) keys[t] = INT_MAX;
    __syncthreads();
    // bitonic sort on (key); equal keys end in a network-determined (fixed) order
    for (int k = 2; k <= cap; k <<= 1) {
      for (int j = k >> 1; j > 0; j >>= 1) {
        for (int t = threadIdx.x; t < cap; t += kCommThreads) {
          const int u = t ^ j;
          if (u > t) {
            const bool up = (t & k) == 0;
            const int kt = keys[t], ku = keys[u];
            if ((kt > ku) == up) {
              keys[t] = ku;
              keys[u] = kt;
              const cplx tv = vals[t];
              vals[t] = vals[u];
              vals[u] = tv;
            }
          }
        }
        __syncthreads();
      }
    }
    // each thread owns a contiguous slice; a "head" starts a run of equal columns
    const int per = (total + kCommThreads - 1) / kCommThreads;
    const int s0 = min(total, threadIdx.x * per), s1 = min(total, s0 + per);
    int cnt = 0;
    for (int t = s0; t < s1; ++t) {
      if (t == 0 || keys[t] != keys[t - 1]) {
        cplx z = vals[t];
        for (int u = t + 1; u < total && keys[u] == keys[t]; ++u) {
          z.x += vals[u].x;
          z.y += vals[u].y;
        }
        if (z.x != 0.0 || z.y != 0.0) ++cnt;
      }
    }
    scan[threadIdx.x + 1] = cnt;
    if (threadIdx.x == 0) scan[0] = 0;
    __syncthreads();
    if (threadIdx.x == 0)
      for (int t = 1; t <= kCommThreads; ++t) scan[t] += scan[t - 1];
    __syncthreads();
    if (!WRITE) {
      if (threadIdx.x == 0) counts[row] = scan[kCommThreads];
    } else {
      int o = rp_out[row] + scan[threadIdx.x];
      for (int t = s0; t < s1; ++t) {
        if (t == 0 || keys[t] != keys[t - 1]) {
          cplx z = vals[t];
          for (int u = t + 1; u < total && keys[u] == keys[t]; ++u) {
            z.x += vals[u].x;
            z.y += vals[u].y;
          }
          if (z.x != 0.0 || z.y != 0.0) {
            ci_out[o] = keys[t];
            v_out[o] = z;
            ++o;
          }
        }
      }
    }
    __syncthreads();
  }
}

// Builds C = AB - BA into freshly cudaMalloc'ed arrays (caller frees).
int csr_commutator_build(const CsrRaw& A, const CsrRaw& B, int64_t n, int32_t** rp_out, int32_t** ci_out,
                         cplx** v_out, int64_t* nnz_out, cudaStream_t st) {
  int32_t* counts = nullptr;
  int32_t* rp = nullptr;
  int* overflow = nullptr;
  int* work = nullptr;          // [0] = rows left to the CTA-wide kernel, then the rows
  int* work2 = nullptr;         // the same for the second tier of the warp kernel
  int32_t* tmp_ci = nullptr;
  cplx* tmp_v = nullptr;
  void* tmp = nullptr;
  size_t tmp_bytes = 0;
  int rc = MAGNUS_OK;
  *rp_out = nullptr;
  *ci_out = nullptr;
  *v_out = nullptr;
  if (cudaMalloc(&counts, sizeof(int32_t) * (size_t)(n + 1)) != cudaSuccess ||
      cudaMalloc(&rp, sizeof(int32_t) * (size_t)(n + 1)) != cudaSuccess ||
      cudaMalloc(&overflow, sizeof(int)) != cudaSuccess ||
      cudaMalloc(&work, sizeof(int) * (size_t)(n + 1)) != cudaSuccess ||
      cudaMalloc(&work2, sizeof(int) * (size_t)(n + 1)) != cudaSuccess ||
      cudaMalloc(&tmp_ci, sizeof(int32_t) * (size_t)n * kCommTmp) != cudaSuccess ||
      cudaMalloc(&tmp_v, sizeof(cplx) * (size_t)n * kCommTmp) != cudaSuccess) {
    cudaGetLastError();
    set_error("sparse commutator: workspace allocation failed (n=%lld)", (long long)n);
    rc = MAGNUS_ENOMEM;
  }
  const int64_t gmax = (int64_t)device_sm_count() * 16;
  const int64_t mrows = (n + kMergeWarps - 1) / kMergeWarps;
  const int mgrid = (int)(mrows < gmax ? mrows : gmax);
  int h_over = 0, h_work = 0, grid = 1;
  int32_t h_nnz = 0;
  if (rc == MAGNUS_OK) {
    cudaMemsetAsync(overflow, 0, sizeof(int), st);
    cudaMemsetAsync(work, 0, sizeof(int), st);
    cudaMemsetAsync(work2, 0, sizeof(int), st);
    cudaMemsetAsync(counts + n, 0, sizeof(int32_t), st);
    cudaFuncSetAttribute(csr_commutator_merge_kernel<512, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, merge_smem<512>());
    cudaFuncSetAttribute(csr_commutator_merge_kernel<kSortCap, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         merge_smem<kSortCap>());
    csr_commutator_merge_kernel<512, false><<<mgrid, kMergeWarps * 32, merge_smem<512>(), st>>>(A, B, n, counts, tmp_ci, tmp_v,
                                                                                              work, work2, nullptr);
    // second tier: its row count is on the device, so the grid is sized for the machine and strides over the list
    csr_commutator_merge_kernel<kSortCap, true><<<device_sm_count() * 4, kMergeWarps * 32, merge_smem<kSortCap>(), st>>>(
        A, B, n, counts, tmp_ci, tmp_v, work, work2, work2);
    cudaMemcpyAsync(&h_work, work, sizeof(int), cudaMemcpyDeviceToHost, st);
    if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = MAGNUS_ECUDA;
    grid = (int)(h_work < gmax ? (h_work > 0 ? h_work : 1) : gmax);
    if (rc == MAGNUS_OK && h_work)   // rows with too many source rows, candidates or entries: expand / sort / merge
      csr_commutator_kernel<false><<<grid, kCommThreads, 0, st>>>(A, B, n, counts, nullptr, nullptr, nullptr, overflow,
                                                                  work);
    if (rc == MAGNUS_OK) {
      cub::DeviceScan::ExclusiveSum(nullptr, tmp_bytes, counts, rp, (int)(n + 1), st);
      if (cudaMalloc(&tmp, tmp_bytes) != cudaSuccess) rc = MAGNUS_ENOMEM;
    }
  }
  if (rc == MAGNUS_OK) {
    cub::DeviceScan::ExclusiveSum(tmp, tmp_bytes, counts, rp, (int)(n + 1), st);
    cudaMemcpyAsync(&h_over, overflow, sizeof(int), cudaMemcpyDeviceToHost, st);
    cudaMemcpyAsync(&h_nnz, rp + n, sizeof(int32_t), cudaMemcpyDeviceToHost, st);
    if (cudaStreamSynchronize(st) != cudaSuccess) rc = MAGNUS_ECUDA;
  }
  if (rc == MAGNUS_OK && h_over) {
    set_error("sparse commutator: a row needs more than %d candidate products", kCommCap);
    rc = MAGNUS_EINVAL;
  }
  int32_t* ci = nullptr;
  cplx* v = nullptr;
  if (rc == MAGNUS_OK) {
    const size_t cap = h_nnz > 0 ? (size_t)h_nnz : 1;
    if (cudaMalloc(&ci, sizeof(int32_t) * cap) != cudaSuccess || cudaMalloc(&v, sizeof(cplx) * cap) != cudaSuccess)
      rc = MAGNUS_ENOMEM;
  }
  if (rc == MAGNUS_OK) {
    const int64_t gblocks = (n * 32 + 255) / 256;
    csr_commutator_gather_kernel<<<(unsigned)gblocks, 256, 0, st>>>(n, counts, rp, tmp_ci, tmp_v, ci, v);
    if (h_work) csr_commutator_kernel<true><<<grid, kCommThreads, 0, st>>>(A, B, n, nullptr, rp, ci, v, overflow, work);
    if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = MAGNUS_ECUDA;
  }
  cudaFree(counts);
  cudaFree(overflow);
  cudaFree(work);
  cudaFree(work2);
  cudaFree(tmp_ci);
  cudaFree(tmp_v);
  cudaFree(tmp);
  if (rc != MAGNUS_OK) {
    cudaFree(rp);
    cudaFree(ci);
    cudaFree(v);
    return rc;
  }
  *rp_out = rp;
  *ci_out = ci;
  *v_out = v;
  *nnz_out = h_nnz;
  return MAGNUS_OK;
}

int csr_commutator_owned(const magnus_matrix* A, const magnus_matrix* B, int32_t** rp, int32_t** ci, cplx** v,
                         int64_t* nnz, cudaStream_t st) {
  CsrRaw a{A->row_ptr, A->col_idx, (const cplx*)A->values}, b{B->row_ptr, B->col_idx, (const cplx*)B->values};
  return csr_commutator_build(a, b, A->n, rp, ci, v, nnz, st);
}

int csr_commutator(const magnus_matrix* A, const magnus_matrix* B, int64_t cap, int64_t* nnz_out, int32_t* rp_out,
                   int32_t* ci_out, cplx* v_out, cudaStream_t st) {
  int32_t* rp = nullptr;
  int32_t* ci = nullptr;
  cplx* v = nullptr;
  int64_t nnz = 0;
  int rc = csr_commutator_owned(A, B, &rp, &ci, &v, &nnz, st);
  if (rc != MAGNUS_OK) return rc;
  *nnz_out = nnz;
  if (cap > 0) {
    if (cap < nnz) {
      set_error("magnus_commutator_csr: capacity %lld < nnz %lld", (long long)cap, (long long)nnz);
      rc = MAGNUS_EINVAL;
    } else {
      cudaMemcpyAsync(rp_out, rp, sizeof(int32_t) * (size_t)(A->n + 1), cudaMemcpyDeviceToDevice, st);
      cudaMemcpyAsync(ci_out, ci, sizeof(int32_t) * (size_t)nnz, cudaMemcpyDeviceToDevice, st);
      cudaMemcpyAsync(v_out, v, sizeof(cplx) * (size_t)nnz, cudaMemcpyDeviceToDevice, st);
      if (cudaStreamSynchronize(st) != cudaSuccess) rc = MAGNUS_ECUDA;
    }
  }
  cudaFree(rp);
  cudaFree(ci);
  cudaFree(v);
  return rc;
}

// ---------------------------------------------------------------------------
// Sampled Hermitian check (magnus_create with check_hermitian): for a strided
// sample of rows, every stored (i,j) must have a stored (j,i) = conj, found by
// binary search.  Reports the largest violation.
// ---------------------------------------------------------------------------
__global__ void csr_hermitian_check_kernel(CsrRaw A, int64_t n, int64_t stride, double* __restrict__ worst) {
  double bad = 0.0;
  for (int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; s * stride < n;
       s += (int64_t)gridDim.x * blockDim.x) {
    const int64_t i = s * stride;
    for (int q = A.rp[i]; q < A.rp[i + 1]; ++q) {
      const int j = A.ci[q];
      const cplx a = A.v[q];
      int lo = A.rp[j], hi = A.rp[j + 1] - 1;
      cplx b = make_double2(0.0, 0.0);
      while (lo <= hi) {
        const int mid = (lo + hi) >> 1;
        const int c = A.ci[mid];
        if (c == (int)i) {
          b = A.v[mid];
          break;
        }
        if (c < (int)i) lo = mid + 1; else hi = mid - 1;
      }
      bad = fmax(bad, fmax(fabs(a.x - b.x), fabs(a.y + b.y)));
    }
  }
  double dummy = -INFINITY;
  double neg = -bad;
  block_reduce_minmax<256>(neg, dummy);
  if (threadIdx.x == 0) worst[blockIdx.x] = -neg;
}

int csr_hermitian_check(const magnus_matrix* A, cudaStream_t st, double* max_violation) {
  CsrRaw a{A->row_ptr, A->col_idx, (const cplx*)A->values};
  const int64_t n = A->n;
  const int64_t stride = n > 65536 ? n / 65536 : 1;
  const int grid = 64;
  double* worst = nullptr;
  if (cudaMalloc(&worst, sizeof(double) * grid) != cudaSuccess) return MAGNUS_ENOMEM;
  csr_hermitian_check_kernel<<<grid, 256, 0, st>>>(a, n, stride, worst);
  double h[64];
  cudaMemcpyAsync(h, worst, sizeof(double) * grid, cudaMemcpyDeviceToHost, st);
  const cudaError_t e = cudaStreamSynchronize(st);
  cudaFree(worst);
  if (e != cudaSuccess) return MAGNUS_ECUDA;
  double m = 0.0;
  for (int i = 0; i < grid; ++i) m = h[i] > m ? h[i] : m;
  *max_violation = m;
  return MAGNUS_OK;
}

}  // namespace magnus
