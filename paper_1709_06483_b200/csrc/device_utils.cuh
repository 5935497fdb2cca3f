// Small device helpers: complex128 arithmetic on double2, deterministic block
// reductions (fixed shuffle tree, no atomics), cache-hinted 128-bit loads.
#ifndef MAGNUS_DEVICE_UTILS_CUH
#define MAGNUS_DEVICE_UTILS_CUH

#include <cuda_runtime.h>
#include <stdint.h>

namespace magnus {

typedef double2 cplx;

__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
// |z| for the Gershgorin radii: exact for purely real or imaginary entries (the spin-chain case),
// one fma + sqrt otherwise (no hypot scaling: |M_ij| of a Hamiltonian is far from over/underflow;
// the last-ulp difference to hypot is absorbed by the interval snapping, reading c4).
__device__ __forceinline__ double cabs_fast(cplx z) {
  if (z.y == 0.0) return fabs(z.x);
  if (z.x == 0.0) return fabs(z.y);
  return sqrt(fma(z.x, z.x, z.y * z.y));
}
// acc += a * b
__device__ __forceinline__ void cfma(cplx& acc, cplx a, cplx b) {
  acc.x = fma(a.x, b.x, acc.x);
  acc.x = fma(-a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y);
  acc.y = fma(a.y, b.x, acc.y);
}

// Streaming loads of matrix data that is read once per launch: kept out of L1
// (no_allocate) and marked evict-first in L2 through a createpolicy descriptor,
// so that the gathered vector w stays cached.  (The direct .L2::evict_first
// qualifier exists only for 256-bit loads on sm_100a; ld_stream256 uses it.)
__device__ __forceinline__ uint64_t policy_evict_first() {
  uint64_t pol;
  asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
  uint64_t pol;
  asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ cplx ld_stream(const cplx* p, uint64_t pol) {
  cplx r;
  asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;"
               : "=d"(r.x), "=d"(r.y)
               : "l"(p), "l"(pol));
  return r;
}
__device__ __forceinline__ int ld_stream_i32(const int32_t* p, uint64_t pol) {
  int r;
  asm("ld.global.nc.L1::no_allocate.L2::cache_hint.s32 %0, [%1], %2;" : "=r"(r) : "l"(p), "l"(pol));
  return r;
}
// 256-bit streaming load (two complex128), sm_100a LDG.256 with L2 evict-first.
__device__ __forceinline__ void ld_stream256(const cplx* p, cplx& a, cplx& b) {
  asm("ld.global.nc.L1::no_allocate.L2::evict_first.v4.f64 {%0, %1, %2, %3}, [%4];"
               : "=d"(a.x), "=d"(a.y), "=d"(b.x), "=d"(b.y)
               : "l"(p));
}
// 128-bit load / store carrying an L2 cache-policy descriptor (createpolicy), coherent path.
__device__ __forceinline__ cplx ld_hint(const cplx* p, uint64_t pol) {
  cplx r;
  asm volatile("ld.global.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(r.x), "=d"(r.y) : "l"(p), "l"(pol) : "memory");
  return r;
}
__device__ __forceinline__ void st_hint(cplx* p, cplx v, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}
// gather load that does not allocate an L1 line (read-only path)
__device__ __forceinline__ cplx ld_gather_na(const cplx* p) {
  cplx r;
  asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
  return r;
}
// Streaming store (written once, re-read only by the next launch).
__device__ __forceinline__ void st_stream(cplx* p, cplx v) {
  asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}

// ---- row-block staging (kernels_csr_rowblock.cu, csr_gershgorin_staged_kernel) ----
// Shared-memory slot of staged entry e: one 16-byte pad every 8 entries, so that 32 lanes reading
// at a row-length stride spread over the banks.
__device__ __forceinline__ int rb_slot(int e) { return e + (e >> 3); }

__device__ __forceinline__ void cp_async16(void* dst_smem, const void* src, uint64_t pol) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(dst_smem);
  asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(s), "l"(src), "l"(pol)
               : "memory");
}
__device__ __forceinline__ void cp_async4(void* dst_smem, const void* src, uint64_t pol) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(dst_smem);
  asm volatile("cp.async.ca.shared.global.L2::cache_hint [%0], [%1], 4, %2;" ::"r"(s), "l"(src), "l"(pol)
               : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

__device__ __forceinline__ double shfl_xor_d(double v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }
__device__ __forceinline__ double shfl_down_d(double v, int d) { return __shfl_down_sync(0xffffffffu, v, d); }

// Sum of (a, b) over the block; result valid in thread 0.  Fixed tree.
template <int THREADS>
__device__ __forceinline__ void block_reduce_sum2(double& a, double& b) {
  __shared__ double sa[THREADS / 32], sb[THREADS / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += shfl_down_d(a, o);
    b += shfl_down_d(b, o);
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0) {
    sa[warp] = a;
    sb[warp] = b;
  }
  __syncthreads();
  if (warp == 0) {
    a = lane < THREADS / 32 ? sa[lane] : 0.0;
    b = lane < THREADS / 32 ? sb[lane] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      a += shfl_down_d(a, o);
      b += shfl_down_d(b, o);
    }
  }
  __syncthreads();
}

// (min of lo, max of hi) over the block; result valid in thread 0.
template <int THREADS>
__device__ __forceinline__ void block_reduce_minmax(double& lo, double& hi) {
  __shared__ double slo[THREADS / 32], shi[THREADS / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lo = fmin(lo, shfl_down_d(lo, o));
    hi = fmax(hi, shfl_down_d(hi, o));
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0) {
    slo[warp] = lo;
    shi[warp] = hi;
  }
  __syncthreads();
  if (warp == 0) {
    lo = lane < THREADS / 32 ? slo[lane] : INFINITY;
    hi = lane < THREADS / 32 ? shi[lane] : -INFINITY;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      lo = fmin(lo, shfl_down_d(lo, o));
      hi = fmax(hi, shfl_down_d(hi, o));
    }
  }
  __syncthreads();
}

// ---- grid barrier of the persistent (cooperative, all CTAs resident) sweep kernels ----
__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

// All CTAs of the (cooperative, co-resident) grid meet here; everything written before is visible after.
__device__ __forceinline__ void grid_barrier(unsigned* counter, unsigned& generation) {
  __syncthreads();
  generation += 1;
  if (threadIdx.x == 0) {
    const unsigned target = generation * gridDim.x;
    __threadfence();
    atomicAdd(counter, 1u);
    while (ld_acquire_u32(counter) < target) {
    }
    __threadfence();
  }
  __syncthreads();
}

}  // namespace magnus
#endif
