// S6 -- fused Leja iteration on a SLICE-MAJOR copy of the CSR operator (csr_kernel = 5).
//
// The row-block kernel (kernels_csr_rowblock.cu) streams the CSR range of 32 rows into shared
// memory so that a lane can walk "its" row while the warp's global reads stay coalesced; ncu shows
// it limited by what fits into shared memory between request and last use (profiles/
// r2_csr_kernel_study.md).  Here the handle owns a re-ordered copy of the operator, built once
// in magnus_create, in which the coalesced order IS the storage order, so the kernel needs no
// staging at all and the register file holds what is in flight:
//
//   * a SLICE is 32 consecutive rows; the entries of all terms (H0, H1 and, for M4, C = [H0,H1])
//     of a slice are stored together, term after term;
//   * inside a term the entries of a slice are grouped into SLOTS.  A slot holds at most one
//     entry per row, all with the same diagonal offset (column - row): the slots of a slice are
//     found by a 32-way merge of its rows on that key.  A slot is stored as a 32-bit row mask
//     plus its entries packed in row order, values and columns in two parallel arrays -- no
//     padding, 20 bytes per stored entry exactly as in CSR;
//   * lane l of the warp that owns the slice is row l.  For a slot with mask m it reads entry
//     popc(m & lanes below l): active lanes read consecutive addresses (128-bit values, 32-bit
//     columns), and because all entries of a slot share col - row, the gather of w touches one
//     contiguous piece of w (on the spin chains col = row XOR mask: col - row is +-mask).
//
// The warp runs a software pipeline over the slots of its slices, eight at a time: the column
// indices of batch b+1 are requested while the values and the w-gathers of batch b are in
// flight, across term and slice boundaries (the next 32 slot masks are prefetched too).
// Per-iteration HBM traffic: 20 B per stored entry + 64 B per row (w, w+, p) + 4 B per slot and
// 24 B per slice of bookkeeping (instead of CSR's 4 B per row and term of row pointers).
// Deterministic: fixed row -> lane map, per-row sums in slot order (ascending col - row inside a
// term), fixed reduction trees.  The summation order differs from CSR order by a permutation
// inside a row, so results agree with the other kernels to rounding, not bit for bit.
#include "magnus_internal.h"
#include "device_utils.cuh"
#include "leja_finalize.cuh"

#include <climits>

namespace magnus {

namespace {

constexpr int SL_WARPS = 4;     // warps per CTA
constexpr int SL_PAD = 8;       // the slots of every term of a slice are padded (zero masks) to a multiple of this
constexpr int SL_CAP = 512;     // slots of one slice the per-warp mask buffer holds; a layout with a larger slice is refused

struct SliceView {
  int64_t n, nslices;
  const int4* meta;            // per slice: {first slot (global), slots, first slot of term 1, of term 2 (slice-relative)}
  const int64_t* ent_ptr;      // [nslices + 1] first entry of the slice in ci / v
  const unsigned* slot_mask;
  const int32_t* ci;
  const cplx* v;
  cplx coef[3];
};

// Predicated loads whose destination is preset inside the asm block: the compiler sees one producer, so the
// load stays asynchronous (a C++ "x = ok ? load : 0" becomes load + select and the select waits for the load).
// No L2 cache-policy operand: it has to sit in a uniform register and cost two R2UR per load (ncu), and the
// evict-first hint made no difference on this workload (profiles/r2_csr_kernel_study.md).
__device__ __forceinline__ cplx ld_stream_if(const cplx* p, unsigned ok) {
  cplx r;
  asm("{\n .reg .pred q;\n setp.ne.b32 q, %3, 0;\n mov.f64 %0, 0d0000000000000000;\n mov.f64 %1, 0d0000000000000000;\n"
      " @q ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];\n}"
      : "=d"(r.x), "=d"(r.y)
      : "l"(p), "r"(ok));
  return r;
}
// column index, or `other` (the lane's own row: a harmless gather target) for a lane without an entry in the slot
__device__ __forceinline__ int ld_stream_i32_if(const int32_t* p, unsigned ok, int other) {
  int r;
  asm("{\n .reg .pred q;\n setp.ne.b32 q, %2, 0;\n mov.b32 %0, %3;\n"
      " @q ld.global.nc.L1::no_allocate.s32 %0, [%1];\n}"
      : "=r"(r)
      : "l"(p), "r"(ok), "r"(other));
  return r;
}

struct SliceDesc {
  unsigned eb;  // first entry of the slice (the layout is refused beyond 2^32 stored entries)
  int sb;       // first slot of the slice in slot_mask
  int ns;       // slots (padded: a multiple of SL_PAD, at least SL_PAD)
  int b1, b2;   // first slot of term 1 / of term 2
};

// per-warp buffer of a slice's slots: .x = row mask (arrives by cp.async), .y = entries of the slice before the slot
__device__ __forceinline__ void stage_masks(const SliceView& L, const SliceDesc& D, uint2* buf, int lane) {
  const unsigned* __restrict__ src = L.slot_mask + D.sb;
#pragma unroll 1
  for (int k = lane; k < D.ns; k += 32) {
    const unsigned dst = (unsigned)__cvta_generic_to_shared(&buf[k].x);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src + k) : "memory");
  }
}
// after the masks have landed: running entry offsets, 32 slots per warp scan
__device__ __forceinline__ void scan_masks(uint2* buf, int ns, int lane) {
  int run = 0;
  for (int k0 = 0; k0 < ns; k0 += 32) {
    const int k = k0 + lane;
    const int cnt = k < ns ? __popc(buf[k].x) : 0;
    int inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int up = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += up;
    }
    if (k < ns) buf[k].y = (unsigned)(run + inc - cnt);
    run += __shfl_sync(0xffffffffu, inc, 31);
  }
  __syncwarp();
}

// C stage: column indices of the SL_U slots whose masks start at mk; run = entries of the slice before them
template <int SL_U>
__device__ __forceinline__ void issue_cols(const int32_t* __restrict__ ci, unsigned eb, const uint2* mk, unsigned lbit,
                                           unsigned lt, int row, int (&cn)[SL_U]) {
#pragma unroll
  for (int u = 0; u < SL_U; u += 2) {
    const uint4 q = *reinterpret_cast<const uint4*>(mk + u);   // two slots: {mask, start, mask, start}
    cn[u] = ld_stream_i32_if(ci + (eb + q.y + __popc(q.x & lt)), q.x & lbit, row);
    cn[u + 1] = ld_stream_i32_if(ci + (eb + q.w + __popc(q.z & lt)), q.z & lbit, row);
  }
}

// SL_U slots per batch, MINB resident CTAs per SM (register budget 65536 / (128 MINB) per thread)
template <int SL_U, int MINB>
__global__ void __launch_bounds__(SL_WARPS * 32, MINB)
    csr_leja_iter_slice_kernel(SliceView L, const cplx* __restrict__ w_in, cplx* __restrict__ w_out,
                               cplx* __restrict__ p, double inv_gamma, double shift, cplx dk, double abs_dk,
                               double tol, LejaStatus* status, double* partials, unsigned* ticket) {
  if (status->done) return;
  __shared__ __align__(16) uint2 s_mask[SL_WARPS][2][SL_CAP];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const unsigned lbit = 1u << lane, lt = lbit - 1u;
  const int stride = (int)gridDim.x * SL_WARPS, nslices = (int)L.nslices;
  double sw = 0.0, sp = 0.0;

  int s0 = (int)blockIdx.x * SL_WARPS + warp;   // slice in the V stage
  if (s0 < nslices) {
    auto load_desc = [&](int s, SliceDesc& D) {
      const int4 m = __ldg(L.meta + s);
      D.eb = (unsigned)__ldg(L.ent_ptr + s);
      D.sb = m.x;
      D.ns = m.y;
      D.b1 = m.z;
      D.b2 = m.w;
    };
    auto own_row = [&](int s) { return (int)min(((int64_t)s << 5) + lane, L.n - 1); };
    SliceDesc D0, D1, D2;   // current slice, next, the one after (its masks are not staged yet)
    int cb = 0;             // D0's masks are in s_mask[warp][cb], D1's in the other buffer
    load_desc(s0, D0);
    stage_masks(L, D0, s_mask[warp][0], lane);
    bool have1 = s0 + stride < nslices, have2 = s0 + 2 * stride < nslices;
    D1 = D0;
    D2 = D0;
    if (have1) {
      load_desc(s0 + stride, D1);
      stage_masks(L, D1, s_mask[warp][1], lane);
    }
    if (have2) load_desc(s0 + 2 * stride, D2);
    cp_async_wait_all();
    __syncwarp();
    scan_masks(s_mask[warp][0], D0.ns, lane);
    if (have1) scan_masks(s_mask[warp][1], D1.ns, lane);

    int cn[SL_U];
    int j = 0;
    bool fresh1 = have1;   // D1's buffer is already scanned (only before the first slice switch)
    issue_cols<SL_U>(L.ci, D0.eb, s_mask[warp][0], lbit, lt, own_row(s0), cn);
    cplx a = make_double2(0.0, 0.0), y = a, wi = a, pi = a;
    int term = 0;
    {
      const int64_t row = ((int64_t)s0 << 5) + lane;
      if (row < L.n) {
        wi = w_in[row];
        pi = p[row];
      }
    }
    while (true) {
      // ---- V stage: values and w-gathers of slots j .. j+U-1 of D0
      const uint2* mv = s_mask[warp][cb] + j;
      cplx v[SL_U], x[SL_U];
#pragma unroll
      for (int u = 0; u < SL_U; u += 2) {
        const uint4 q = *reinterpret_cast<const uint4*>(mv + u);
        v[u] = ld_stream_if(L.v + (D0.eb + q.y + __popc(q.x & lt)), q.x & lbit);
        x[u] = w_in[cn[u]];   // a lane without an entry gathers its own row's w against v = 0
        v[u + 1] = ld_stream_if(L.v + (D0.eb + q.w + __popc(q.z & lt)), q.z & lbit);
        x[u + 1] = w_in[cn[u + 1]];
      }
      // ---- C stage: columns of the next batch (same slice, or the first batch of the next one)
      const int jn = j + SL_U;
      const bool last = jn >= D0.ns;
      if (!last) {
        issue_cols<SL_U>(L.ci, D0.eb, s_mask[warp][cb] + jn, lbit, lt, own_row(s0), cn);
      } else if (have1) {
        if (!fresh1) {           // D1's masks were requested a slice ago
          cp_async_wait_all();
          __syncwarp();
          scan_masks(s_mask[warp][cb ^ 1], D1.ns, lane);
        }
        fresh1 = false;
        issue_cols<SL_U>(L.ci, D1.eb, s_mask[warp][cb ^ 1], lbit, lt, own_row(s0 + stride), cn);
      }
      // ---- the batch belongs to one term (terms are padded to whole batches)
      const int tnow = (j >= D0.b1) + (j >= D0.b2);
      if (tnow != term) {
        cfma(y, L.coef[term], a);
        a = make_double2(0.0, 0.0);
        term = tnow;
      }
#pragma unroll
      for (int u = 0; u < SL_U; ++u) cfma(a, v[u], x[u]);
      j = jn;
      if (last) {
        // finish the rows of the slice
        cfma(y, L.coef[term], a);
        const int64_t row = ((int64_t)s0 << 5) + lane;
        if (row < L.n) {
          cplx wn;
          wn.x = inv_gamma * y.x - shift * wi.x;
          wn.y = inv_gamma * y.y - shift * wi.y;
          cfma(pi, dk, wn);
          w_out[row] = wn;
          p[row] = pi;
          sw += wn.x * wn.x + wn.y * wn.y;
          sp += pi.x * pi.x + pi.y * pi.y;
        }
        if (!have1) break;
        s0 += stride;
        D0 = D1;
        D1 = D2;
        have1 = have2;
        have2 = s0 + 2 * stride < nslices;
        __syncwarp();   // every lane is done with the old D0's masks
        if (have1) stage_masks(L, D1, s_mask[warp][cb], lane);
        cb ^= 1;
        if (have2) load_desc(s0 + 2 * stride, D2);
        j = 0;
        term = 0;
        a = make_double2(0.0, 0.0);
        y = a;
        const int64_t nrow = ((int64_t)s0 << 5) + lane;
        if (nrow < L.n) {
          wi = w_in[nrow];
          pi = p[nrow];
        }
      }
    }
  }
  block_reduce_sum2<SL_WARPS * 32>(sw, sp);
  if (threadIdx.x == 0) {
    partials[2 * blockIdx.x] = sw;
    partials[2 * blockIdx.x + 1] = sp;
  }
  if (last_block_ticket(ticket)) leja_finalize_warp0(partials, gridDim.x, abs_dk, tol, false, status);   // S7
}

// ---- building the layout (once per handle) ------------------------------------------------
// 32-way merge of the rows of a slice on key = column - row (ascending inside a CSR row).
// FILL = false: count slots and entries per slice; FILL = true: write masks and packed entries.
// OFFS = true: a slot is stored as the record {row mask, column - row} and no column array is written
// (the offset-slot layout of csr_kernel 6); OFFS = false: masks and a column per entry (csr_kernel 5).
// REAL (with OFFS): every stored value has a zero imaginary part (checked before), only the real parts are written.
template <bool FILL, bool OFFS, bool REAL = false>
__global__ void __launch_bounds__(128)
    slice_merge_kernel(CsrOp op, int64_t nslices, int4* meta, int64_t* ent_ptr, unsigned* slot_mask, uint2* slot_rec,
                       int32_t* ci_out, cplx* v_out, double* vr_out = nullptr) {
  const int lane = threadIdx.x & 31;
  const unsigned lt = (1u << lane) - 1u;
  const int64_t s = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (s >= nslices) return;
  const int64_t row = (s << 5) + lane;
  const bool valid = row < op.n;
  int nslots = 0, b[3] = {0, 0, 0};
  int64_t ents = 0;
  int sb = 0;
  int64_t eb = 0;
  if (FILL) {
    sb = meta[s].x;
    eb = ent_ptr[s];
  }
#pragma unroll
  for (int t = 0; t < 3; ++t) {
    b[t] = nslots;
    if (t >= op.nterms) continue;
    const int32_t* __restrict__ ci = op.t[t].ci;
    const cplx* __restrict__ vv = op.t[t].v;
    int cur = valid ? op.t[t].rp[row] : 0;
    const int end = valid ? op.t[t].rp[row + 1] : 0;
    int col = cur < end ? ci[cur] : 0;
    int key = cur < end ? col - (int)row : INT_MAX;
    while (true) {
      const int kmin = __reduce_min_sync(0xffffffffu, key);
      if (kmin == INT_MAX) break;
      const bool hit = key == kmin;
      const unsigned m = __ballot_sync(0xffffffffu, hit);
      if (FILL) {
        if (lane == 0) {
          if (OFFS) slot_rec[sb + nslots] = make_uint2(m, (unsigned)kmin);
          else slot_mask[sb + nslots] = m;
        }
        if (hit) {
          const int64_t q = eb + ents + __popc(m & lt);
          if (!OFFS) ci_out[q] = col;
          if (REAL) vr_out[q] = vv[cur].x;
          else v_out[q] = vv[cur];
        }
      }
      ents += __popc(m);
      nslots += 1;
      if (hit) {
        cur += 1;
        col = cur < end ? ci[cur] : 0;
        key = cur < end ? col - (int)row : INT_MAX;
      }
    }
    nslots = (nslots + SL_PAD - 1) / SL_PAD * SL_PAD;   // whole batches per term; the padding masks stay zero
  }
  if (nslots == 0) nslots = SL_PAD;
  if (!FILL && lane == 0) {
    meta[s] = make_int4(0, nslots, op.nterms > 1 ? b[1] : nslots, op.nterms > 2 ? b[2] : nslots);
    ent_ptr[s] = ents;
  }
}

// flag |= 1 if any stored value of the term has a non-zero imaginary part
__global__ void __launch_bounds__(256) csr_any_imag_kernel(const cplx* __restrict__ v, int64_t nnz, int* flag) {
  bool any = false;
  for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < nnz; q += (int64_t)gridDim.x * blockDim.x)
    any |= v[q].y != 0.0;
  if (__syncthreads_or(any) && threadIdx.x == 0) atomicOr(flag, 1);
}

// exclusive prefix sums of the slot and entry counts (one CTA; nslices is at most a few million)
__global__ void __launch_bounds__(1024) slice_scan_kernel(int64_t nslices, int4* meta, int64_t* ent_ptr, int64_t* totals) {
  __shared__ int64_t s_slots[1024], s_ents[1024];
  __shared__ int s_max[1024];
  const int tid = threadIdx.x;
  const int64_t per = (nslices + 1023) / 1024;
  const int64_t lo = min(nslices, (int64_t)tid * per), hi = min(nslices, lo + per);
  int64_t ns = 0, ne = 0;
  int mx = 0;
  for (int64_t s = lo; s < hi; ++s) {
    ns += meta[s].y;
    mx = max(mx, meta[s].y);
    ne += ent_ptr[s];
  }
  s_slots[tid] = ns;
  s_ents[tid] = ne;
  s_max[tid] = mx;
  __syncthreads();
  if (tid == 0) {
    int64_t as = 0, ae = 0;
    for (int i = 0; i < 1024; ++i) {
      const int64_t cs = s_slots[i], ce = s_ents[i];
      s_slots[i] = as;
      s_ents[i] = ae;
      as += cs;
      ae += ce;
      mx = max(mx, s_max[i]);
    }
    totals[0] = as;
    totals[1] = ae;
    totals[2] = mx;
    ent_ptr[nslices] = ae;
  }
  __syncthreads();
  ns = s_slots[tid];
  ne = s_ents[tid];
  for (int64_t s = lo; s < hi; ++s) {
    const int cnt = meta[s].y;
    const int64_t ce = ent_ptr[s];
    meta[s].x = (int)ns;
    ent_ptr[s] = ne;
    ns += cnt;
    ne += ce;
  }
}


// ---------------------------------------------------------------------------------------------
// csr_kernel = 6: the OFFSET-SLOT layout.  All entries of a slot share column - row, so the slot
// record {row mask, column - row} replaces the per-entry column array: per stored entry the kernel
// reads the 16-byte value and nothing else (8 bytes per slot instead of 4 bytes per entry), and the
// w-gather address row + offset is known without a dependent index load.  The warp keeps SO_U slots
// in flight per lane in a ROTATING register pipeline: slot u of the batch being consumed is
// multiplied and its registers are re-used at once for slot u of the next batch (which may belong to
// the next slice), so value and w loads are outstanding all the time instead of draining at batch
// boundaries.  Slot records reach the warp through a double-buffered per-warp shared-memory ring
// (one 16-byte cp.async per lane and slice, requested a whole slice ahead).
// Per-iteration HBM traffic: 16 B per stored entry + 8 B per slot + 24 B per slice + 64 B per row.
// ---------------------------------------------------------------------------------------------
constexpr int SO_CAP = 256;    // slots of one slice a ring buffer holds; a layout with a larger slice is refused

struct SliceViewO {
  int64_t n, nslices;
  const int4* meta;            // per slice: {first slot (global), slots, first slot of term 1, of term 2}
  const int64_t* ent_ptr;      // [nslices + 1]
  const uint2* rec;            // per slot {row mask, column - row}
  const cplx* v;               // values, or
  const double* vr;            // ... their real parts when every imaginary part is zero (real layout: 8 B per entry)
  cplx coef[3];
};

// value type in flight: complex, or the real part alone
template <bool REAL> struct SlotVal { typedef cplx type; };
template <> struct SlotVal<true> { typedef double type; };
__device__ __forceinline__ double ld_stream_real_if(const double* p, unsigned ok) {
  double r;
  asm("{\n .reg .pred q;\n setp.ne.b32 q, %2, 0;\n mov.f64 %0, 0d0000000000000000;\n"
      " @q ld.global.nc.L1::no_allocate.f64 %0, [%1];\n}"
      : "=d"(r)
      : "l"(p), "r"(ok));
  return r;
}
// acc += v x for a real v: the two products the complex form adds with a zero imaginary part are left out, the
// result is the same to the bit
__device__ __forceinline__ void slot_fma(cplx& acc, double v, cplx x) {
  acc.x = fma(v, x.x, acc.x);
  acc.y = fma(v, x.y, acc.y);
}
__device__ __forceinline__ void slot_fma(cplx& acc, cplx v, cplx x) { cfma(acc, v, x); }

__device__ __forceinline__ cplx ld_stream_hint_if(const cplx* p, unsigned ok, uint64_t pol) {
  cplx r;
  asm("{\n .reg .pred q;\n setp.ne.b32 q, %3, 0;\n mov.f64 %0, 0d0000000000000000;\n mov.f64 %1, 0d0000000000000000;\n"
      " @q ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0, %1}, [%2], %4;\n}"
      : "=d"(r.x), "=d"(r.y)
      : "l"(p), "r"(ok), "l"(pol));
  return r;
}
__device__ __forceinline__ cplx ld_cached_hint_if(const cplx* p, unsigned ok, uint64_t pol) {
  cplx r;
  asm("{\n .reg .pred q;\n setp.ne.b32 q, %3, 0;\n mov.f64 %0, 0d0000000000000000;\n mov.f64 %1, 0d0000000000000000;\n"
      " @q ld.global.nc.L2::cache_hint.v2.f64 {%0, %1}, [%2], %4;\n}"
      : "=d"(r.x), "=d"(r.y)
      : "l"(p), "r"(ok), "l"(pol));
  return r;
}
__device__ __forceinline__ cplx ld_cached_if(const cplx* p, unsigned ok) {
  cplx r;
  asm("{\n .reg .pred q;\n setp.ne.b32 q, %3, 0;\n mov.f64 %0, 0d0000000000000000;\n mov.f64 %1, 0d0000000000000000;\n"
      " @q ld.global.nc.v2.f64 {%0, %1}, [%2];\n}"
      : "=d"(r.x), "=d"(r.y)
      : "l"(p), "r"(ok));
  return r;
}

// POL: 0 no L2 hints; 1 matrix values evict-first; 2 also w gathers evict-last.  SO_U slots in flight per lane.
template <int SO_U, int MINB, int POL, bool REAL>
__global__ void __launch_bounds__(SL_WARPS * 32, MINB)
    csr_leja_iter_sliceoff_kernel(SliceViewO L, const cplx* __restrict__ w_in, cplx* __restrict__ w_out,
                                  cplx* __restrict__ p, double inv_gamma, double shift, cplx dk, double abs_dk,
                                  double tol, LejaStatus* status, double* partials, unsigned* ticket) {
  static_assert(SL_PAD % SO_U == 0, "batches must not straddle terms (terms are padded to SL_PAD slots)");
  if (status->done) return;
  __shared__ __align__(16) uint2 s_rec[SL_WARPS][2][SO_CAP];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const unsigned lbit = 1u << lane, lt = lbit - 1u;
  const int stride = (int)gridDim.x * SL_WARPS, nslices = (int)L.nslices;
  double sw = 0.0, sp = 0.0;

  const uint64_t pol_v = POL >= 1 ? policy_evict_first() : 0, pol_w = POL >= 2 ? policy_evict_last() : 0;
  int sI = (int)blockIdx.x * SL_WARPS + warp;   // slice on the issue side
  if (sI < nslices) {
    struct Desc { int64_t eb; int sb, ns, b1, b2; };
    auto load_desc = [&](int s, Desc& D) {
      const int4 m = __ldg(L.meta + s);
      D.eb = __ldg(L.ent_ptr + s);
      D.sb = m.x;
      D.ns = m.y;
      D.b1 = m.z;
      D.b2 = m.w;
    };
    auto stage = [&](const Desc& D, uint2* buf) {   // two records per 16-byte copy
      for (int k = 2 * lane; k < D.ns; k += 64) {
        const unsigned dst = (unsigned)__cvta_generic_to_shared(buf + k);
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(L.rec + D.sb + k) : "memory");
      }
    };
    Desc DI, DN, D2;     // slice being issued, the next one (records staged), the one after (descriptor only)
    load_desc(sI, DI);
    stage(DI, s_rec[warp][0]);
    bool haveN = sI + stride < nslices, have2 = sI + 2 * stride < nslices;
    DN = DI;
    D2 = DI;
    if (haveN) {
      load_desc(sI + stride, DN);
      stage(DN, s_rec[warp][1]);
    }
    if (have2) load_desc(sI + 2 * stride, D2);
    cp_async_wait_all();
    __syncwarp();

    // issue side
    int bufI = 0, jI = 0;
    unsigned runI = 0;                       // entries of the slice before slot jI
    typedef typename SlotVal<REAL>::type val_t;
    const val_t* vbI = (REAL ? (const val_t*)L.vr : (const val_t*)L.v) + DI.eb;
    int64_t rowI = ((int64_t)sI << 5) + lane;
    bool issuing = true;
    // consume side (one batch behind)
    int jC = 0, nsC = DI.ns, b1C = DI.b1, b2C = DI.b2, term = 0;
    int64_t rowC = rowI;
    cplx a = make_double2(0.0, 0.0), y = a, wi = a, pi = a;
    if (rowC < L.n) {
      wi = w_in[rowC];
      pi = p[rowC];
    }
    val_t v[SO_U];
    cplx x[SO_U];
    auto issue_slot = [&](int u) {
      const uint2 r = s_rec[warp][bufI][jI + u];
      const unsigned ok = r.x & lbit;
      if constexpr (REAL) {
        v[u] = ld_stream_real_if(vbI + (runI + __popc(r.x & lt)), ok);
      } else {
        v[u] = POL >= 1 ? ld_stream_hint_if(vbI + (runI + __popc(r.x & lt)), ok, pol_v)
                        : ld_stream_if(vbI + (runI + __popc(r.x & lt)), ok);
      }
      x[u] = POL >= 2 ? ld_cached_hint_if(w_in + (rowI + (int)r.y), ok, pol_w)
                      : ld_cached_if(w_in + (rowI + (int)r.y), ok);
      runI += __popc(r.x);
    };
#pragma unroll
    for (int u = 0; u < SO_U; ++u) issue_slot(u);
    jI = SO_U;

    while (true) {
      // ---- issue side: next batch of the same slice, or the first batch of the next slice
      if (jI >= DI.ns) {
        if (haveN) {
          sI += stride;
          DI = DN;
          DN = D2;
          haveN = have2;
          have2 = sI + 2 * stride < nslices;
          cp_async_wait_all();   // the new slice's records were requested a slice ago
          __syncwarp();          // ... and every lane is done with the old slice's
          if (haveN) stage(DN, s_rec[warp][bufI]);
          bufI ^= 1;
          if (have2) load_desc(sI + 2 * stride, D2);
          jI = 0;
          runI = 0;
          vbI = (REAL ? (const val_t*)L.vr : (const val_t*)L.v) + DI.eb;
          rowI = ((int64_t)sI << 5) + lane;
        } else {
          issuing = false;
        }
      }
      // ---- consume side: the batch belongs to one term (terms are padded to whole batches)
      const int tnow = (jC >= b1C) + (jC >= b2C);
      if (tnow != term) {
        cfma(y, L.coef[term], a);
        a = make_double2(0.0, 0.0);
        term = tnow;
      }
      if (issuing) {
#pragma unroll
        for (int u = 0; u < SO_U; ++u) {
          slot_fma(a, v[u], x[u]);
          issue_slot(u);
        }
        jI += SO_U;
      } else {
#pragma unroll
        for (int u = 0; u < SO_U; ++u) slot_fma(a, v[u], x[u]);
      }
      jC += SO_U;
      if (jC >= nsC) {
        // finish the rows of the slice
        cfma(y, L.coef[term], a);
        if (rowC < L.n) {
          cplx wn;
          wn.x = inv_gamma * y.x - shift * wi.x;
          wn.y = inv_gamma * y.y - shift * wi.y;
          cfma(pi, dk, wn);
          w_out[rowC] = wn;
          p[rowC] = pi;
          sw += wn.x * wn.x + wn.y * wn.y;
          sp += pi.x * pi.x + pi.y * pi.y;
        }
        if (!issuing) break;
        // the issue side is exactly one batch ahead: it has just entered the slice consumed next
        jC = 0;
        nsC = DI.ns;
        b1C = DI.b1;
        b2C = DI.b2;
        rowC = rowI;
        term = 0;
        a = make_double2(0.0, 0.0);
        y = a;
        if (rowC < L.n) {
          wi = w_in[rowC];
          pi = p[rowC];
        }
      }
    }
  }
  block_reduce_sum2<SL_WARPS * 32>(sw, sp);
  if (threadIdx.x == 0) {
    partials[2 * blockIdx.x] = sw;
    partials[2 * blockIdx.x + 1] = sp;
  }
  if (last_block_ticket(ticket)) leja_finalize_warp0(partials, gridDim.x, abs_dk, tol, false, status);   // S7
}

}  // namespace

void slice_layout_free(SliceLayout* L) {
  if (!L) return;
  cudaFree(L->meta);
  cudaFree(L->ent_ptr);
  cudaFree(L->slot_mask);
  cudaFree(L->slot_rec);
  cudaFree(L->ci);
  cudaFree(L->v);
  cudaFree(L->vr);
  *L = SliceLayout();
}

// Returns MAGNUS_OK and a filled layout, or an error code with *out left empty (callers fall back to
// the CSR kernels: the layout is an optimisation, never a requirement).  Synchronises the stream once.
// offsets = true builds the offset-slot layout of csr_kernel 6 (slot records, no column array).
// allow_real (offset-slot layout only; the shortcut MAGNUS_SHORTCUT_REAL_VALUES): when no stored value of any term has
// an imaginary part -- a real symmetric operator, e.g. the spin chains -- only the real parts are stored (8 B per
// entry) and the kernel multiplies by them; the results are the same to the bit.
int slice_layout_build(const CsrOp& op, SliceLayout* out, cudaStream_t st, bool offsets, bool allow_real) {
  *out = SliceLayout();
  SliceLayout L;
  L.n = op.n;
  L.nslices = (op.n + 31) >> 5;
  L.nterms = op.nterms;
  L.offsets = offsets;
  int64_t* totals = nullptr;
  int64_t host_totals[4] = {0, 0, 0, 0};
  bool ok = cudaMalloc(&L.meta, sizeof(int4) * (size_t)L.nslices) == cudaSuccess &&
            cudaMalloc(&L.ent_ptr, sizeof(int64_t) * (size_t)(L.nslices + 1)) == cudaSuccess &&
            cudaMalloc(&totals, 4 * sizeof(int64_t)) == cudaSuccess;
  const int64_t blocks = (L.nslices * 32 + 127) / 128;
  if (ok) {
    cudaMemsetAsync(totals, 0, 4 * sizeof(int64_t), st);
    if (offsets && allow_real)
      for (int t = 0; t < op.nterms; ++t) {
        int64_t g = (op.t[t].nnz + 255) / 256;
        if (g > (int64_t)device_sm_count() * 16) g = (int64_t)device_sm_count() * 16;
        if (g > 0) csr_any_imag_kernel<<<(int)g, 256, 0, st>>>(op.t[t].v, op.t[t].nnz, reinterpret_cast<int*>(totals + 3));
      }
    slice_merge_kernel<false, false><<<(unsigned)blocks, 128, 0, st>>>(op, L.nslices, L.meta, L.ent_ptr, nullptr, nullptr,
                                                                       nullptr, nullptr);
    slice_scan_kernel<<<1, 1024, 0, st>>>(L.nslices, L.meta, L.ent_ptr, totals);
    ok = cudaMemcpyAsync(host_totals, totals, sizeof host_totals, cudaMemcpyDeviceToHost, st) == cudaSuccess &&
         cudaStreamSynchronize(st) == cudaSuccess;
  }
  if (ok) {
    ok = host_totals[0] < ((int64_t)1 << 31) && host_totals[2] <= (offsets ? SO_CAP : SL_CAP) &&
         host_totals[1] < ((int64_t)1 << 32);
  }
  if (ok) {
    L.nslots = host_totals[0];
    L.nent = host_totals[1];
    L.real_values = offsets && allow_real && host_totals[3] == 0;
    const size_t ns = (size_t)(L.nslots > 0 ? L.nslots : 1), ne = (size_t)(L.nent > 0 ? L.nent : 1);
    ok = L.real_values ? cudaMalloc(&L.vr, sizeof(double) * ne) == cudaSuccess : cudaMalloc(&L.v, sizeof(cplx) * ne) == cudaSuccess;
    if (ok && offsets) {
      ok = cudaMalloc(&L.slot_rec, sizeof(uint2) * ns) == cudaSuccess &&
           cudaMemsetAsync(L.slot_rec, 0, sizeof(uint2) * ns, st) == cudaSuccess;
    } else if (ok) {
      ok = cudaMalloc(&L.slot_mask, sizeof(unsigned) * ns) == cudaSuccess &&
           cudaMalloc(&L.ci, sizeof(int32_t) * ne) == cudaSuccess &&
           cudaMemsetAsync(L.slot_mask, 0, sizeof(unsigned) * ns, st) == cudaSuccess;
    }
  }
  if (ok) {
    if (offsets && L.real_values)
      slice_merge_kernel<true, true, true><<<(unsigned)blocks, 128, 0, st>>>(op, L.nslices, L.meta, L.ent_ptr, nullptr,
                                                                             L.slot_rec, nullptr, nullptr, L.vr);
    else if (offsets)
      slice_merge_kernel<true, true><<<(unsigned)blocks, 128, 0, st>>>(op, L.nslices, L.meta, L.ent_ptr, nullptr,
                                                                       L.slot_rec, nullptr, L.v);
    else
      slice_merge_kernel<true, false><<<(unsigned)blocks, 128, 0, st>>>(op, L.nslices, L.meta, L.ent_ptr, L.slot_mask,
                                                                        nullptr, L.ci, L.v);
    ok = cudaGetLastError() == cudaSuccess;
  }
  cudaFree(totals);
  if (!ok) {
    cudaGetLastError();
    slice_layout_free(&L);
    return MAGNUS_ENOMEM;
  }
  *out = L;
  return MAGNUS_OK;
}

int launch_csr_leja_iter_slice(const CsrOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma, double shift,
                               cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st) {
  const SliceLayout& S = *op.slice;
  if (S.offsets) {
    SliceViewO L;
    L.n = S.n;
    L.nslices = S.nslices;
    L.meta = S.meta;
    L.ent_ptr = S.ent_ptr;
    L.rec = S.slot_rec;
    L.v = S.v;
    L.vr = S.vr;
    for (int t = 0; t < 3; ++t) L.coef[t] = t < op.nterms ? op.t[t].coef : make_double2(0.0, 0.0);
    // tuning code 6000 + 100 POL + 10 [4 slots in flight instead of 8] + MINB (default 6004: no hints, 8 slots,
    // 4 CTAs = 16 warps per SM)
    int code = ws->csr_kernel >= 6000 && ws->csr_kernel < 7000 ? ws->csr_kernel - 6000 : 4;
    if (code >= 500) code -= 500;       // 6500..6999: the same tuning codes on real-part storage (see slice_layout_build)
    const int minb = code % 10, pol = code / 100, u = (code / 10) % 10 ? 4 : 8;
    const bool real = S.real_values;
#define SO_LAUNCH(U, MINB, POL)                                                                                      \
  SO_LAUNCH_(U, MINB, POL, false)                                                                                    \
  SO_LAUNCH_(U, MINB, POL, true)
#define SO_LAUNCH_(U, MINB, POL, REAL)                                                                               \
  if (u == U && minb == MINB && pol == POL && real == REAL) {                                                        \
    int64_t g = (S.nslices + SL_WARPS - 1) / SL_WARPS;                                                               \
    const int64_t cap = (int64_t)device_sm_count() * MINB;                                                           \
    if (g > cap) g = cap;                                                                                            \
    csr_leja_iter_sliceoff_kernel<U, MINB, POL, REAL><<<(int)g, SL_WARPS * 32, 0, st>>>(                             \
        L, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws->status, ws->partials, ws->tickets);                \
    ws->launches += 1;                                                                                               \
    return (int)g;                                                                                                   \
  }
    SO_LAUNCH(8, 4, 0)
    SO_LAUNCH(8, 3, 0)
    SO_LAUNCH(8, 4, 1)
    SO_LAUNCH(8, 4, 2)
    SO_LAUNCH(8, 5, 0)
    SO_LAUNCH(4, 5, 0)
    SO_LAUNCH(4, 6, 0)
    SO_LAUNCH(4, 7, 0)
    SO_LAUNCH(4, 8, 0)
#undef SO_LAUNCH
#undef SO_LAUNCH_
    return -1;
  }
  SliceView L;
  L.n = S.n;
  L.nslices = S.nslices;
  L.meta = S.meta;
  L.ent_ptr = S.ent_ptr;
  L.slot_mask = S.slot_mask;
  L.ci = S.ci;
  L.v = S.v;
  for (int t = 0; t < 3; ++t) L.coef[t] = t < op.nterms ? op.t[t].coef : make_double2(0.0, 0.0);
  int code = ws->csr_kernel >= 5000 && ws->csr_kernel < 6000 ? ws->csr_kernel - 5000 : 84;   // 10 U + MINB
#define SL_LAUNCH(U, MINB)                                                                                         \
  if (code == 10 * U + MINB) {                                                                                     \
    int64_t g = (S.nslices + SL_WARPS - 1) / SL_WARPS;                                                             \
    const int64_t cap = (int64_t)device_sm_count() * MINB;                                                         \
    if (g > cap) g = cap;                                                                                          \
    csr_leja_iter_slice_kernel<U, MINB><<<(int)g, SL_WARPS * 32, 0, st>>>(L, w_in, w_out, p, inv_gamma, shift, dk,  \
                                                                         abs_dk, tol, ws->status, ws->partials,   \
                                                                         ws->tickets);                            \
    ws->launches += 1;                                                                                             \
    return (int)g;                                                                                                 \
  }
  SL_LAUNCH(8, 4)
  SL_LAUNCH(8, 3)
  SL_LAUNCH(4, 5)
  SL_LAUNCH(4, 6)
  SL_LAUNCH(4, 8)
#undef SL_LAUNCH
  return -1;
}

}  // namespace magnus
