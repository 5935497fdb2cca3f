// S6 -- fused Leja iteration for large CSR operators: the "stream" kernel (sm_100a).
//
//   y_i  = sum_t coef_t sum_q A_t.v[q] w[A_t.ci[q]]      (SpMV of H(t) = sum_t coef_t A_t, formed on the fly)
//   w+_i = inv_gamma y_i - shift w_i                      (fragment line 4; c5)
//   p_i += d_k w+_i                                       (fragment line 5)
//   block partials of sum |w+|^2, sum |p|^2; stop test in the last block (S7; c6)
//
// One persistent CTA per SM, warp specialised:
//   * warp 0: the PRODUCER.  A unit of work is a block of 32 consecutive rows; the stored entries of those rows
//     are ONE contiguous range of each term's CSR arrays.  The value array of a term is described to the TMA as a
//     2-D tensor of rows of 8 entries (128 bytes), the index array as rows of 32 indices (128 bytes), and every
//     (unit, term) is fetched by a few tensor copies (cp.async.bulk.tensor, SASS UTMALDG) whose BOX IS WIDER THAN
//     THE TENSOR ROW (9 resp. 36 elements per row): the out-of-bounds column is zero-filled, so the data lands in
//     shared memory already padded by 16 bytes per 128 -- the layout that makes the row-strided reads of the
//     consumers free of bank conflicts at the spin chain's 24 entries per row -- without a single thread
//     instruction or L1 wavefront spent on staging.  Completion is counted in bytes on the stage's mbarrier
//     (SASS SYNCS).  The ring of stages lets the HBM stream run ahead of the consumers; L2 evict-first on the
//     stream (read once per launch).
//   * warps 1..NC: CONSUMERS, one warp per unit, lane l = row l.  For one entry slot the 32 lanes gather w at
//     32 consecutive rows under (mostly) one column offset: 512 contiguous bytes, the cheapest gather the L1 can
//     serve.  Entries are consumed in batches of 8; the gathered w of the next batches is in flight in registers
//     ahead of the FMAs, across unit boundaries, so the gather pipeline never drains.  A stage is handed back
//     (mbarrier arrive) right after its last read.
//   * the unit order is the natural row order, all CTAs in lockstep (unit u of the launch goes to CTA u mod grid),
//     so the gathered window of w is compact in L2.
// (unit, term)s whose entries exceed the stage capacity, or that touch the tail of an array that does not fill a
// tensor row, are read straight from global memory ("direct"); correctness never depends on the ring.
// Deterministic: fixed unit->warp map, sequential sum along a row in a fixed order, fixed trees.
#include "magnus_internal.h"
#include "device_utils.cuh"
#include "leja_finalize.cuh"

#include <cuda.h>

#include <new>

namespace magnus {

namespace {

constexpr int ST_THREADS_MAX = 32 * 10;   // 1 producer + up to 9 consumer warps (200 registers per thread)
constexpr int ST_SMEM_BUDGET = 220 * 1024;       // ring bytes (the rest of the 227 KB: barriers, reduction scratch)
constexpr int ST_MAX_STAGES = 16;
constexpr int ST_ROW_BYTES = 144;                // one padded tensor row in shared memory: 128 data + 16 pad
constexpr int ST_NVH = 16;                       // box heights of the value copies: (i + 1) * granule tensor rows

// One tensor copy per array and (unit, term): the box is the smallest of a few heights that covers the rows needed
// (the surplus rows belong to the next units, which other SMs fetch at about the same time: L2 hits).
struct StreamMaps {
  CUtensorMap v[3][ST_NVH];
  int vg;                         // granule: box i is (i + 1) * vg tensor rows high (a multiple of 8)
};

__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  unsigned ok = 0;
  const unsigned a = smem_addr(bar);
  while (!ok) {
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
        : "=r"(ok)
        : "r"(a), "r"(parity)
        : "memory");
  }
}
// TMA tile copy global -> shared: box of the tensor map starting at tensor row `row`, completion on an mbarrier
__device__ __forceinline__ void tma_rows_g2s(unsigned dst_smem, const CUtensorMap* map, int row, uint64_t* bar,
                                             uint64_t pol) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], "
      "[%4], %5;" ::"r"(dst_smem),
      "l"(map), "r"(0), "r"(row), "r"(smem_addr(bar)), "l"(pol)
      : "memory");
}

__device__ __forceinline__ void st_release_cta(long long* p, long long v) {
  asm volatile("st.release.cta.shared::cta.s64 [%0], %1;" ::"r"(smem_addr(p)), "l"(v) : "memory");
}
__device__ __forceinline__ long long ld_acquire_cta(const long long* p) {
  long long v;
  asm volatile("ld.acquire.cta.shared::cta.s64 %0, [%1];" : "=l"(v) : "r"(smem_addr(p)) : "memory");
  return v;
}

__device__ __forceinline__ void prefetch_l2(const void* p) {
  asm volatile("prefetch.global.L2::evict_last [%0];" ::"l"(p));
}
__device__ __forceinline__ void cp_async16_shared(unsigned dst_smem, const void* src, uint64_t pol) {
  asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(dst_smem), "l"(src), "l"(pol)
               : "memory");
}

// shared-memory loads through 32-bit shared-space addresses
__device__ __forceinline__ int lds_i32(unsigned addr) {
  int v;
  asm("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ cplx lds_c128(unsigned addr) {
  cplx v;
  asm("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
  return v;
}

struct StreamCfg {
  int cap;        // stage capacity in entries (one term of one 32-row unit), a multiple of 32
  int nstages;
  int ncons;      // consumer warps (one unit each)
  int pol;        // 1: p and w+ move with L2 evict-first hints
  int pfd;        // L2 prefetch distance in units (0 = none)
};

// Tensor rows a stage holds: values (8 entries per row; a range of cap entries touches at most cap/8 + 1 rows),
// indices (32 per row), each rounded up to the 8-row granularity of the boxes.
__host__ __device__ __forceinline__ int stage_vrows(int cap) { return ((cap / 8 + 1) + 7) & ~7; }
__host__ __device__ __forceinline__ int stage_crows(int cap) { return ((cap / 32 + 1) + 7) & ~7; }
__host__ __device__ __forceinline__ int stage_bytes_of(int cap) {
  return (stage_vrows(cap) + stage_crows(cap)) * ST_ROW_BYTES;      // a multiple of 1152 = 9 * 128
}

template <int NT, int NB, int MAXT>
__global__ void __launch_bounds__(MAXT, 1)
    csr_leja_iter_stream_kernel(CsrOp op, const __grid_constant__ StreamMaps maps, const cplx* __restrict__ w_in,
                                cplx* __restrict__ w_out, cplx* __restrict__ p, double inv_gamma, double shift,
                                cplx dk, double abs_dk, double tol, LejaStatus* status, double* partials,
                                unsigned* ticket, StreamCfg cfg) {
  if (status->done) return;
  extern __shared__ __align__(128) unsigned char st_smem[];
  __shared__ __align__(8) uint64_t full_bar[ST_MAX_STAGES];
  __shared__ __align__(8) uint64_t empty_bar[ST_MAX_STAGES];
  __shared__ double red_w[ST_THREADS_MAX / 32], red_p[ST_THREADS_MAX / 32];
  __shared__ long long produced[3];   // per term: units whose stage has been armed by that term's producer

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int NS = cfg.nstages;
  const int sbytes = stage_bytes_of(cfg.cap);
  const unsigned smem_base = smem_addr(st_smem);
  const unsigned coff = (unsigned)(stage_vrows(cfg.cap) * ST_ROW_BYTES);   // index region inside a stage
  const int64_t n = op.n;
  const int64_t nunits = (n + 31) >> 5;
  // units of this CTA: u = blockIdx.x + i * gridDim.x, i < my_units; stage sequence number of (i, t): i NT + t
  const int64_t my_units = nunits > blockIdx.x ? (nunits - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;

  if (threadIdx.x == 0) {
    produced[0] = produced[1] = produced[2] = 0;
    for (int s = 0; s < NS; ++s) {
      mbar_init(&full_bar[s], 33);
      mbar_init(&empty_bar[s], 1);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  double sw = 0.0, sp = 0.0;
  const uint64_t pol = policy_evict_first();

  if (warp < NT) {
    // ------------------------------------------------------------------ producers, one warp per term
    // Row pointers of 32 units are fetched at once, one unit per lane (a unit's two pointers are a dependent HBM
    // round trip: paid once per 32 units, and the next batch is requested before this one is issued); lane 0
    // then arms the stage barriers and issues the tensor copies of its term, one stage per (unit, term).
    const int t = warp;
    int s = t % NS;                                   // stage of (unit 0, term t); NT stages further per unit
    unsigned ph = (unsigned)((t / NS) & 1);
    int nrs = 0, nre = 0;
    auto fetch = [&](int64_t i) {
      nrs = nre = 0;
      if (i < my_units) {
        const int64_t r0 = ((int64_t)blockIdx.x + i * gridDim.x) << 5;
        const int64_t r1 = r0 + 32 < n ? r0 + 32 : n;
        nrs = __ldg(op.t[t].rp + r0);
        nre = __ldg(op.t[t].rp + r1);
      }
    };
    fetch(lane);
    for (int64_t base = 0; base < my_units; base += 32) {
      const int crs = nrs, cre = nre;
      fetch(base + 32 + lane);
      const int cnt = my_units - base < 32 ? (int)(my_units - base) : 32;
      for (int j = 0; j < cnt; ++j) {
        const int rs = __shfl_sync(0xffffffffu, crs, j);
        const int re = __shfl_sync(0xffffffffu, cre, j);
        if (cfg.pfd > 0) {
          // HBM -> L2 prefetch of the (unit, term) pfd units ahead, one 128-byte line per lane and instruction:
          // the tensor copy into shared memory then finds its data in L2, so a ring stage is occupied for an L2
          // round trip instead of an HBM one, and the same ring sustains a higher rate
          const int jj = j + cfg.pfd;
          const int prs = __shfl_sync(0xffffffffu, jj < 32 ? crs : nrs, jj & 31);
          const int pre = __shfl_sync(0xffffffffu, jj < 32 ? cre : nre, jj & 31);
          if (base + jj < my_units && pre > prs) {
            const char* v0 = reinterpret_cast<const char*>(op.t[t].v + prs);
            const char* v1 = reinterpret_cast<const char*>(op.t[t].v + pre);
            for (const char* a = v0 + 128 * lane; a < v1; a += 128 * 32) prefetch_l2(a);
            const char* c0 = reinterpret_cast<const char*>(op.t[t].ci + prs);
            const char* c1 = reinterpret_cast<const char*>(op.t[t].ci + pre);
            for (const char* a = c0 + 128 * lane; a < c1; a += 128 * 32) prefetch_l2(a);
          }
        }
        const int len = re - rs;
        const bool direct = len > cfg.cap || re > ((int)op.t[t].nnz & ~31);
        if (lane == 0) {
          // the slot's previous occupant (sequence number q - NS, another term's) must have been armed before
          // the parity of its "consumed" phase means anything to this warp
          const int64_t q = (base + j) * NT + t;
          if (q >= NS) {
            const int64_t qq = q - NS;
            while (ld_acquire_cta(&produced[qq % NT]) <= qq / NT) {
            }
          }
          mbar_wait(&empty_bar[s], ph ^ 1u);
        }
        __syncwarp();
        // 33 arrivals complete a stage: lane 0's (with the byte count of the tensor copy) and one per lane
        if (len > 0 && !direct) {
          const unsigned dst = smem_base + (unsigned)(s * sbytes);
          if (lane == 0) {
            // values: ONE tensor copy, the smallest box that covers the rows (the TMA's cost is per copy)
            const int q0 = rs >> 3;
            const int nv = ((re + 7) >> 3) - q0;
            const int iv = (nv + maps.vg - 1) / maps.vg - 1;
            mbar_arrive_expect_tx(&full_bar[s], (unsigned)((iv + 1) * maps.vg * ST_ROW_BYTES));
            tma_rows_g2s(dst, &maps.v[t][iv], q0, &full_bar[s], pol);
          }
          // column indices: 16-byte cp.async by the 32 lanes into the same padded layout (a copy of a few KB
          // would cost the TMA as much as the 12 KB of values)
          const int x0 = rs & ~31;
          for (int c4 = (rs >> 2) + lane; c4 < ((re + 3) >> 2); c4 += 32) {
            const int x = 4 * c4 - x0;
            cp_async16_shared(dst + coff + 4u * (unsigned)x + 16u * (unsigned)(x >> 5), op.t[t].ci + 4 * c4, pol);
          }
          asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_addr(&full_bar[s])) : "memory");
        } else {
          // empty or direct (unit, term): nothing staged, the phase still completes
          if (lane == 0) mbar_arrive(&full_bar[s]);
          mbar_arrive(&full_bar[s]);
        }
        // A barrier phase is known by its parity only: a consumer may start to wait for a stage only once the
        // fill of THIS lap has been armed (else it would take the previous lap's completion for its own).
        __syncwarp();
        if (lane == 0) st_release_cta(&produced[t], base + j + 1);
        s += NT;
        while (s >= NS) {
          s -= NS;
          ph ^= 1u;
        }
      }
    }
  } else if (warp < NT + cfg.ncons) {
    // ------------------------------------------------------------------ consumers
    // Lane l walks row l of the unit.  Entry x (counted from the first tensor row of the stage) sits at byte
    // 16 (x + x/8) of the value region and 4 x + 16 (x/32) of the index region: the padded layout the TMA wrote.
    // Per (unit, term): wait for the stage, request the gathers of the first SB NB entries of the row (all in
    // flight at once, in registers), multiply, hand the stage back.  A warp holds one stage at a time; the
    // latency of its gathers is covered by the other consumer warps, the latency of HBM by the ring.
    constexpr int SB = 8;                           // batch of entries; NB batches are in flight per lane
    const int grp = warp - NT;
    const int NGRP = cfg.ncons;

    // this lane's row pointers of a unit, requested two units ahead (a dependent HBM round trip under load);
    // rows beyond n read rp[n]: empty rows, and lane 31 always holds the end of the unit's entry range
    int nrs[2][NT], nre[2][NT];
    auto fetch = [&](int64_t i, int slot) {
#pragma unroll
      for (int t = 0; t < NT; ++t) nrs[slot][t] = nre[slot][t] = 0;
      if (i < my_units) {
        const int64_t row = (((int64_t)blockIdx.x + i * gridDim.x) << 5) + lane;
#pragma unroll
        for (int t = 0; t < NT; ++t) {
          nrs[slot][t] = __ldg(op.t[t].rp + (row < n ? row : n));
          nre[slot][t] = __ldg(op.t[t].rp + (row + 1 < n ? row + 1 : n));
        }
      }
    };
    // stage and phase of (unit, term 0) of the warp's current unit
    int s0 = 0;
    unsigned ph0 = 0;
    {
      const int64_t q = (int64_t)grp * NT;
      s0 = (int)(q % NS);
      ph0 = (unsigned)((q / NS) & 1);
    }
    fetch(grp, 0);
    fetch(grp + (int64_t)NGRP, 1);
    for (int64_t i = grp; i < my_units; i += NGRP) {
      const int64_t r0 = ((int64_t)blockIdx.x + i * gridDim.x) << 5;
      const int64_t row = r0 + lane;
      int rs[NT], len[NT];
#pragma unroll
      for (int t = 0; t < NT; ++t) {
        rs[t] = nrs[0][t];
        len[t] = nre[0][t] - nrs[0][t];
        nrs[0][t] = nrs[1][t];
        nre[0][t] = nre[1][t];
      }
      fetch(i + 2 * (int64_t)NGRP, 1);
      cplx wi = make_double2(0.0, 0.0), pi = make_double2(0.0, 0.0);   // consumed in the epilogue of this unit
      if (row < n) {
        wi = w_in[row];
        pi = cfg.pol ? ld_hint(p + row, pol) : p[row];
      }
      cplx y = make_double2(0.0, 0.0);
      int s = s0;
      unsigned ph = ph0;
#pragma unroll
      for (int t = 0; t < NT; ++t) {
        const int b = __shfl_sync(0xffffffffu, rs[t], 0);
        const int e = __shfl_sync(0xffffffffu, rs[t] + len[t], 31);
        const bool direct = e - b > cfg.cap || e > ((int)op.t[t].nnz & ~31);   // uniform; as the producer decides
        const int maxlen = __reduce_max_sync(0xffffffffu, len[t]);
        const unsigned sa = smem_base + (unsigned)(s * sbytes);
        const int xv = rs[t] - (b & ~7), xc = rs[t] - (b & ~31);
        auto col_addr = [&](int j) {
          const int x = xc + j;
          return sa + coff + 4u * (unsigned)x + 16u * (unsigned)(x >> 5);
        };
        auto val_addr = [&](int j) {
          const int x = xv + j;
          return sa + 16u * (unsigned)(x + (x >> 3));
        };
        cplx a = make_double2(0.0, 0.0);
        while (ld_acquire_cta(&produced[t]) <= i) {
        }
        mbar_wait(&full_bar[s], ph);                   // also for empty and direct terms: the ring protocol is uniform
        if (direct) {
          for (int j = 0; j < len[t]; ++j) {           // straight from global memory
            const int q = rs[t] + j;
            cfma(a, ld_stream(op.t[t].v + q, pol), w_in[ld_stream_i32(op.t[t].ci + q, pol)]);
          }
        } else if (maxlen > 0) {
          cplx X[NB][SB];
#pragma unroll
          for (int h = 0; h < NB; ++h) {
            if (maxlen > SB * h) {
#pragma unroll
              for (int u = 0; u < SB; ++u)
                if (SB * h + u < len[t]) X[h][u] = w_in[lds_i32(col_addr(SB * h + u))];
            }
          }
#pragma unroll
          for (int h = 0; h < NB; ++h) {
            if (maxlen > SB * h) {
#pragma unroll
              for (int v = 0; v < SB; v += 4) {
                cplx m[4];
#pragma unroll
                for (int u = 0; u < 4; ++u)
                  if (SB * h + v + u < len[t]) m[u] = lds_c128(val_addr(SB * h + v + u));
#pragma unroll
                for (int u = 0; u < 4; ++u)
                  if (SB * h + v + u < len[t]) cfma(a, m[u], X[h][v + u]);
              }
            }
          }
          if (maxlen > SB * NB) {                      // rows longer than SB NB entries: plain loop
            for (int j = SB * NB; j < len[t]; ++j) cfma(a, lds_c128(val_addr(j)), w_in[lds_i32(col_addr(j))]);
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty_bar[s]);     // every read of this stage is done
        const cplx ca = cmul(op.t[t].coef, a);
        y.x += ca.x;
        y.y += ca.y;
        if (++s == NS) {
          s = 0;
          ph ^= 1u;
        }
      }
      if (row < n) {
        cplx wn;
        wn.x = inv_gamma * y.x - shift * wi.x;
        wn.y = inv_gamma * y.y - shift * wi.y;
        cfma(pi, dk, wn);
        if (cfg.pol) {
          st_hint(w_out + row, wn, pol);
          st_hint(p + row, pi, pol);
        } else {
          w_out[row] = wn;
          p[row] = pi;
        }
        sw += wn.x * wn.x + wn.y * wn.y;
        sp += pi.x * pi.x + pi.y * pi.y;
      }
      // first stage of the warp's next unit: NGRP units further on
      s0 += (NGRP * NT) % NS;
      ph0 ^= (unsigned)(((NGRP * NT) / NS) & 1);
      if (s0 >= NS) {
        s0 -= NS;
        ph0 ^= 1u;
      }
    }
  }

  // block partials (fixed tree) and the stop test in the last block of the launch
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    sw += shfl_down_d(sw, o);
    sp += shfl_down_d(sp, o);
  }
  if (lane == 0) {
    red_w[warp] = sw;
    red_p[warp] = sp;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0;
    const int nw = blockDim.x >> 5;
    for (int w = 0; w < nw; ++w) {
      a += red_w[w];
      b += red_p[w];
    }
    partials[2 * blockIdx.x] = a;
    partials[2 * blockIdx.x + 1] = b;
  }
  if (last_block_ticket(ticket)) leja_finalize_warp0(partials, gridDim.x, abs_dk, tol, false, status);   // S7
}

// ---------------------------------------------------------------------------------------------------------
// Row-block kernel with TMA staging ("rowtma"): the occupancy structure of kernels_csr_rowblock.cu -- every warp
// owns 32 consecutive rows and a private staging buffer, 12 warps per SM, no warp waits for another -- with the
// staging done by the TMA instead of 48 cp.async instructions per lane and block:
//   values          ONE tensor copy per (block, term) into the padded layout (box wider than the tensor row, see
//                   the header of this file), completion counted in bytes on the warp's own mbarrier;
//   column indices  16-byte cp.async by the 32 lanes into the matching padded layout (a 3 KB copy would cost the
//                   TMA as much as the 12 KB of values: its cost is per copy), tracked by the same mbarrier;
// and with all gathers of up to RT_NB*8 entries of a row in flight in registers before the first FMA.
// ---------------------------------------------------------------------------------------------------------
constexpr int RT_WARPS = 4;                       // warps per CTA, 3 CTAs per SM
constexpr int RT_CAP = 768;                       // entries per warp buffer (one term of one 32-row block)
constexpr int RT_VROWS = RT_CAP / 8 + 8;          // value tensor rows (8 entries each): 96 + unaligned start, 8-row boxes
constexpr int RT_CROWS = RT_CAP / 32 + 1;         // index rows (32 entries each)
constexpr int RT_BYTES_PER_WARP = (((RT_VROWS + RT_CROWS) * ST_ROW_BYTES + 127) / 128) * 128;   // TMA: 128-byte aligned
constexpr int RT_SMEM = RT_WARPS * RT_BYTES_PER_WARP;
constexpr int RT_NB = 3;                          // batches of 8 entries in flight per lane

template <int NT>
__global__ void __launch_bounds__(RT_WARPS * 32, 3)
    csr_leja_iter_rowtma_kernel(CsrOp op, const __grid_constant__ StreamMaps maps, const cplx* __restrict__ w_in,
                                cplx* __restrict__ w_out, cplx* __restrict__ p, double inv_gamma, double shift,
                                cplx dk, double abs_dk, double tol, LejaStatus* status, double* partials,
                                unsigned* ticket, int pol_on) {
  if (status->done) return;
  extern __shared__ __align__(128) unsigned char rt_smem[];
  __shared__ __align__(8) uint64_t bar[RT_WARPS];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const unsigned buf = smem_addr(rt_smem) + (unsigned)(warp * RT_BYTES_PER_WARP);
  const unsigned cbuf = buf + RT_VROWS * ST_ROW_BYTES;
  if (lane == 0) mbar_init(&bar[warp], 33);        // lane 0's arrive with the byte count + one arrive per lane
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  __syncwarp();
  unsigned phase = 0;
  const uint64_t pol = policy_evict_first();
  const int64_t n = op.n;
  const int64_t nblocks = (n + 31) >> 5;
  const int64_t total_warps = (int64_t)gridDim.x * RT_WARPS;
  double sw = 0.0, sp = 0.0;

  for (int64_t blk = (int64_t)blockIdx.x * RT_WARPS + warp; blk < nblocks; blk += total_warps) {
    const int64_t row = (blk << 5) + lane;
    const bool valid = row < n;
    int rs_t[NT], re_t[NT];
#pragma unroll
    for (int t = 0; t < NT; ++t) {
      rs_t[t] = __ldg(op.t[t].rp + (valid ? row : n));
      re_t[t] = __ldg(op.t[t].rp + (valid ? row + 1 : n));
    }
    cplx wi = make_double2(0.0, 0.0), pi = make_double2(0.0, 0.0);
    if (valid) {
      wi = w_in[row];
      pi = pol_on ? ld_hint(p + row, pol) : p[row];
    }
    cplx y = make_double2(0.0, 0.0);
#pragma unroll
    for (int t = 0; t < NT; ++t) {
      const int32_t* __restrict__ ci = op.t[t].ci;
      const cplx* __restrict__ vv = op.t[t].v;
      const int rs = rs_t[t], re = re_t[t];
      const int tail_from = (int)op.t[t].nnz & ~31;   // entries from here on are not covered by the tensor map
      cplx a = make_double2(0.0, 0.0);
      int first = 0;   // first lane (row) of the block not yet consumed
      while (first < 32) {
        const int base = __shfl_sync(0xffffffffu, rs, first);
        const bool fits = (re - base) <= RT_CAP && re <= tail_from;   // monotone in the lane: re ascends
        const unsigned nofit = ~__ballot_sync(0xffffffffu, fits || lane < first);
        const int last = nofit ? (__ffs(nofit) - 1) : 32;             // first lane whose row does not fit any more
        if (last == first) {
          // a row longer than the buffer, or in the tail of the arrays: the whole warp strides over it
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
        const int end = __shfl_sync(0xffffffffu, re, last - 1);
        if (end > base) {
          // ---- stage entries [base, end): values by the TMA, indices by cp.async
          if (lane == 0) {
            const int q0 = base >> 3;
            const int nv = ((end + 7) >> 3) - q0;
            const int iv = (nv + maps.vg - 1) / maps.vg - 1;
            mbar_arrive_expect_tx(&bar[warp], (unsigned)((iv + 1) * maps.vg * ST_ROW_BYTES));
            tma_rows_g2s(buf, &maps.v[t][iv], q0, &bar[warp], pol);
          }
          const int x0 = base & ~31;
          for (int c4 = (base >> 2) + lane; c4 < ((end + 3) >> 2); c4 += 32) {
            const int x = 4 * c4 - x0;
            cp_async16_shared(cbuf + 4u * (unsigned)x + 16u * (unsigned)(x >> 5), ci + 4 * c4, pol);
          }
          asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_addr(&bar[warp])) : "memory");
          mbar_wait(&bar[warp], phase);
          phase ^= 1u;
          // ---- lane l walks row first <= l < last out of the padded buffer
          const bool mine = lane >= first && lane < last;
          const int mylen = mine ? re - rs : 0;
          const int maxlen = __reduce_max_sync(0xffffffffu, mylen);
          const int xv = rs - (base & ~7), xc = rs - x0;
          for (int j0 = 0; j0 < maxlen; j0 += 8 * RT_NB) {
            cplx X[RT_NB][8];
#pragma unroll
            for (int h = 0; h < RT_NB; ++h) {
              if (maxlen > j0 + 8 * h) {
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                  const int j = j0 + 8 * h + u;
                  if (j < mylen) {
                    const int x = xc + j;
                    X[h][u] = w_in[lds_i32(cbuf + 4u * (unsigned)x + 16u * (unsigned)(x >> 5))];
                  }
                }
              }
            }
#pragma unroll
            for (int h = 0; h < RT_NB; ++h) {
              if (maxlen > j0 + 8 * h) {
#pragma unroll
                for (int v = 0; v < 8; v += 4) {
                  cplx m[4];
#pragma unroll
                  for (int u = 0; u < 4; ++u) {
                    const int x = xv + j0 + 8 * h + v + u;
                    if (j0 + 8 * h + v + u < mylen) m[u] = lds_c128(buf + 16u * (unsigned)(x + (x >> 3)));
                  }
#pragma unroll
                  for (int u = 0; u < 4; ++u)
                    if (j0 + 8 * h + v + u < mylen) cfma(a, m[u], X[h][v + u]);
                }
              }
            }
          }
          __syncwarp();   // everyone done reading before the buffer is refilled
        }
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
      if (pol_on) {
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
  block_reduce_sum2<RT_WARPS * 32>(sw, sp);
  if (threadIdx.x == 0) {
    partials[2 * blockIdx.x] = sw;
    partials[2 * blockIdx.x + 1] = sp;
  }
  if (last_block_ticket(ticket)) leja_finalize_warp0(partials, gridDim.x, abs_dk, tol, false, status);   // S7
}

// max over the 32-row units and the terms of the stored entries of one term in one unit
__global__ void __launch_bounds__(256) csr_unit_cap_kernel(CsrOp op, int* __restrict__ out) {
  const int64_t nunits = (op.n + 31) >> 5;
  int m = 0;
  for (int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; u < nunits; u += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r0 = u << 5, r1 = r0 + 32 < op.n ? r0 + 32 : op.n;
    for (int t = 0; t < op.nterms; ++t) m = max(m, op.t[t].rp[r1] - op.t[t].rp[r0]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(out, m);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* ptr = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)ptr;
  }
  return fn;
}

// Box heights: (i + 1) * granule, the granule the smallest multiple of 8 rows that reaches the stage size.
void box_granule(int cap, int* vg) {
  const int vr = stage_vrows(cap);
  *vg = 8;
  while (*vg * ST_NVH < vr) *vg += 8;
}

// Tensor maps of one term: rows of 128 bytes, box one 16-byte element wider than the row (zero-filled pad).
bool encode_term_maps(const CsrTerm& T, int vg, CUtensorMap* v) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  const cuuint32_t estr[2] = {1, 1};
  const cuuint64_t gstride[1] = {128};
  const cuuint64_t vrows = (cuuint64_t)(T.nnz / 8);
  if (vrows == 0) return false;
  for (int i = 0; i < ST_NVH; ++i) {
    const int vhi = (i + 1) * vg;
    if (vhi > 256) break;
    const cuuint64_t gdim[2] = {16, vrows};                      // 8 complex128 = 16 doubles per tensor row
    const cuuint32_t box[2] = {18, (cuuint32_t)vhi};           // + one complex of padding
    if (enc(&v[i], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void*)T.v, gdim, gstride, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return false;
  }
  return true;
}

// tensor maps are cached per workspace, keyed by the terms' arrays
struct MapCache {
  const void* key_v[3] = {nullptr, nullptr, nullptr};
  const void* key_c[3] = {nullptr, nullptr, nullptr};
  int64_t key_nnz[3] = {0, 0, 0};
  int key_cap = 0;
  int nterms = 0;
  StreamMaps maps;
};

// Stage capacity: the largest (unit, term) of the operator, but never so large that fewer than four stages fit
// the ring -- (unit, term)s above the capacity are read straight from global memory ("direct").
int stage_cap(const CsrOp& op) {
  int cap = (op.unit_cap + 31) & ~31;
  int cap_max = 32;
  while (ST_SMEM_BUDGET / stage_bytes_of(cap_max + 32) >= 4 && stage_vrows(cap_max + 32) <= 256) cap_max += 32;
  return cap < cap_max ? cap : cap_max;
}

}  // namespace

int csr_unit_cap(const CsrOp& op, cudaStream_t st, int* cap_out) {
  int* d = nullptr;
  if (cudaMalloc(&d, sizeof(int)) != cudaSuccess) return MAGNUS_ENOMEM;
  cudaMemsetAsync(d, 0, sizeof(int), st);
  const int64_t nunits = (op.n + 31) >> 5;
  int64_t g = (nunits + 255) / 256;
  if (g > (int64_t)device_sm_count() * 8) g = (int64_t)device_sm_count() * 8;
  csr_unit_cap_kernel<<<(int)g, 256, 0, st>>>(op, d);
  int h = 0;
  cudaMemcpyAsync(&h, d, sizeof(int), cudaMemcpyDeviceToHost, st);
  const cudaError_t e = cudaStreamSynchronize(st);
  cudaFree(d);
  if (e != cudaSuccess) return MAGNUS_ECUDA;
  *cap_out = h;
  return MAGNUS_OK;
}

void stream_maps_free(Workspace* ws) {
  delete static_cast<MapCache*>(ws->stream_maps);
  ws->stream_maps = nullptr;
}

// The TMA needs 16-byte aligned arrays and at least one full tensor row per array.
bool csr_stream_supported(const CsrOp& op) {
  if (op.unit_cap <= 0) return false;
  for (int t = 0; t < op.nterms; ++t)
    if (((uintptr_t)op.t[t].v & 15) || ((uintptr_t)op.t[t].ci & 15) || op.t[t].nnz < 32) return false;
  return encode_tiled_fn() != nullptr;
}

int launch_csr_leja_iter_stream(const CsrOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma,
                                double shift, cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st) {
  MapCache* mc = static_cast<MapCache*>(ws->stream_maps);
  if (!mc) {
    mc = new (std::nothrow) MapCache();
    if (!mc) return -1;
    ws->stream_maps = mc;
  }
  const int cap = stage_cap(op);
  bool same = mc->nterms == op.nterms && mc->key_cap == cap;
  for (int t = 0; t < op.nterms && same; ++t)
    same = mc->key_v[t] == op.t[t].v && mc->key_c[t] == op.t[t].ci && mc->key_nnz[t] == op.t[t].nnz;
  if (!same) {
    mc->nterms = 0;
    box_granule(cap, &mc->maps.vg);
    for (int t = 0; t < op.nterms; ++t) {
      if (!encode_term_maps(op.t[t], mc->maps.vg, mc->maps.v[t])) return -1;
      mc->key_v[t] = op.t[t].v;
      mc->key_c[t] = op.t[t].ci;
      mc->key_nnz[t] = op.t[t].nnz;
    }
    mc->key_cap = cap;
    mc->nterms = op.nterms;
  }

  StreamCfg cfg;
  cfg.cap = cap;
  int ns = ST_SMEM_BUDGET / stage_bytes_of(cfg.cap);
  if (ns > ST_MAX_STAGES) ns = ST_MAX_STAGES;
  // csr_kernel 3: defaults; 20000 + 1000*ncons + 10*(stages, 0 = all that fit) + pol selects a variant (tuning sweeps)
  cfg.ncons = 7;
  cfg.pfd = 0;
  cfg.pol = (int64_t)64 * op.n > (int64_t)64 * 1024 * 1024 ? 1 : 0;   // vectors beyond L2: stream p and w+
  if (ws->csr_kernel >= 20000 && ws->csr_kernel < 30000) {
    const int v = ws->csr_kernel - 20000;
    cfg.ncons = v / 1000;
    cfg.pfd = (v / 10) % 100;
    if (cfg.pfd > 31) cfg.pfd = 31;
    cfg.pol = v % 10;
    if (cfg.ncons < 1 || cfg.ncons + op.nterms > 10) return -1;
  }
  cfg.nstages = ns;
  // a consumer holds at most one stage, and never while it waits: any ring of two or more stages makes progress;
  // stages beyond the consumers' are the prefetch depth (barrier-phase aliasing is excluded by `produced`)
  if (ns < 2) return -1;
  if (cfg.ncons > ns - 1) cfg.ncons = ns - 1;
  const int smem = ns * stage_bytes_of(cfg.cap);
  const int threads = 32 * (cfg.ncons + op.nterms);
  const int64_t nunits = (op.n + 31) >> 5;
  int64_t g = device_sm_count();
  if (g > nunits) g = nunits;
  if (g > kMaxPartials) g = kMaxPartials;
#define ST_LAUNCH(NT, NB, MAXT)                                                                                    \
  do {                                                                                                             \
    auto kern = csr_leja_iter_stream_kernel<NT, NB, MAXT>;                                                         \
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return -1;   \
    kern<<<(int)g, threads, smem, st>>>(op, mc->maps, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol,           \
                                        ws->status, ws->partials, ws->tickets, cfg);                               \
  } while (0)
  cfg.pol &= 1;
  // up to 7 consumer warps run with 255 registers per thread, 8 or 9 with 168
  if (threads <= 256) {
    if (op.nterms == 1) ST_LAUNCH(1, 3, 256);
    else if (op.nterms == 2) ST_LAUNCH(2, 3, 256);
    else ST_LAUNCH(3, 3, 256);
  } else {
    if (op.nterms == 1) ST_LAUNCH(1, 3, 320);
    else if (op.nterms == 2) ST_LAUNCH(2, 3, 320);
    else ST_LAUNCH(3, 3, 320);
  }
#undef ST_LAUNCH
  ws->launches += 1;
  return (int)g;
}

// maps of the operator's terms, cached in the workspace (box granule for a buffer of `cap` entries)
static MapCache* maps_for(const CsrOp& op, int cap, Workspace* ws) {
  MapCache* mc = static_cast<MapCache*>(ws->stream_maps);
  if (!mc) {
    mc = new (std::nothrow) MapCache();
    if (!mc) return nullptr;
    ws->stream_maps = mc;
  }
  bool same = mc->nterms == op.nterms && mc->key_cap == cap;
  for (int t = 0; t < op.nterms && same; ++t)
    same = mc->key_v[t] == op.t[t].v && mc->key_c[t] == op.t[t].ci && mc->key_nnz[t] == op.t[t].nnz;
  if (!same) {
    mc->nterms = 0;
    box_granule(cap, &mc->maps.vg);
    for (int t = 0; t < op.nterms; ++t) {
      if (!encode_term_maps(op.t[t], mc->maps.vg, mc->maps.v[t])) return nullptr;
      mc->key_v[t] = op.t[t].v;
      mc->key_c[t] = op.t[t].ci;
      mc->key_nnz[t] = op.t[t].nnz;
    }
    mc->key_cap = cap;
    mc->nterms = op.nterms;
  }
  return mc;
}

bool csr_rowtma_supported(const CsrOp& op) {
  for (int t = 0; t < op.nterms; ++t)
    if (((uintptr_t)op.t[t].v & 15) || ((uintptr_t)op.t[t].ci & 15) || op.t[t].nnz < 32) return false;
  return encode_tiled_fn() != nullptr;
}

int launch_csr_leja_iter_rowtma(const CsrOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma,
                                double shift, cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st) {
  MapCache* mc = maps_for(op, RT_CAP, ws);
  if (!mc) return -1;
  const int64_t nblocks = (op.n + 31) >> 5;
  int64_t g = (nblocks + RT_WARPS - 1) / RT_WARPS;
  const int64_t cap = (int64_t)device_sm_count() * 3;
  if (g > cap) g = cap;
  const int pol_on = (int64_t)64 * op.n > (int64_t)64 * 1024 * 1024 ? 1 : 0;   // vectors beyond L2: stream p and w+
#define RT_LAUNCH(NT)                                                                                              \
  do {                                                                                                             \
    auto kern = csr_leja_iter_rowtma_kernel<NT>;                                                                   \
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, RT_SMEM) != cudaSuccess) return -1; \
    kern<<<(int)g, RT_WARPS * 32, RT_SMEM, st>>>(op, mc->maps, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol,  \
                                                 ws->status, ws->partials, ws->tickets, pol_on);                   \
  } while (0)
  if (op.nterms == 1) RT_LAUNCH(1);
  else if (op.nterms == 2) RT_LAUNCH(2);
  else RT_LAUNCH(3);
#undef RT_LAUNCH
  ws->launches += 1;
  return (int)g;
}

}  // namespace magnus
