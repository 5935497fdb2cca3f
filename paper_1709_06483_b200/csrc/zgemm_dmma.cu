// D3 -- the dense M4 commutator product P = A2 A1 (P:262 l.6-7 "A_4 = A_2 A_1")
// as a complex128 GEMM on the FP64 tensor pipe: mma.sync.m8n8k4.f64 (SASS
// DMMA.8x8x4; tcgen05 has no f64 kind, so this is the one legacy-shape MMA in
// the library).  C = A * B, all row-major n x n.
//
// Tiling: CTA 128 x 64 complex outputs, 8 warps as 4 (m) x 2 (n), warp tile
// 32 x 32 complex = 4 x 4 DMMA tiles, four real DMMAs per complex tile and k4:
//   C_re += A_re B_re + A_im (-B_im),   C_im += A_re B_im + A_im B_re.
// Operands stay interleaved (re, im) in shared memory: one LDS.128 yields both
// planes of a fragment element.  K is consumed in slabs of 16 complex through a
// 3-stage cp.async ring (16-byte copies, zero-filled outside the matrix).
// Row pitches of 20 (A) and 66 (B) double2 make the fragment loads conflict-free.
// Two instantiations: 128 x 64 tiles (8 warps, one CTA per SM) and 64 x 64 tiles (4 warps, two CTAs per SM).
// The small tile is for sizes whose 128 x 64 tile count leaves the last wave mostly empty (n = 2048: 512
// tiles on 148 SMs = 3.46 waves): with two CTAs per SM the last, partial wave has an SM to itself per CTA
// and runs at about twice the per-CTA speed, so the tail costs half a wave instead of a whole one.
#include "magnus_internal.h"
#include "device_utils.cuh"

namespace magnus {

namespace {

constexpr int BN = 64, BK = 16, STAGES = 3;
constexpr int LDA_S = BK + 4;    // double2 units
constexpr int LDB_S = BN + 2;
constexpr int B_STAGE = BK * LDB_S;
template <int BM>
constexpr int zgemm_smem() { return STAGES * (BM * LDA_S + B_STAGE) * (int)sizeof(cplx); }

__device__ __forceinline__ void cp_async16_zfill(void* dst_smem, const void* src, bool valid) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(dst_smem);
  const int bytes = valid ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

__device__ __forceinline__ void dmma8x8x4(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

template <int BM>
__global__ void __launch_bounds__(BM * 2, BM == 128 ? 1 : 2) zgemm_dmma_kernel(int64_t n, const cplx* __restrict__ A, int64_t lda,
                                                                       const cplx* __restrict__ B, int64_t ldb,
                                                                       cplx* __restrict__ C, int64_t ldc, int tiles_m,
                                                                       int tiles_n) {
  constexpr int THREADS = BM * 2;              // BM / 32 x 2 warps
  constexpr int A_STAGE = BM * LDA_S;          // double2 per stage
  extern __shared__ __align__(16) unsigned char zg_smem[];
  cplx* sA = reinterpret_cast<cplx*>(zg_smem);
  cplx* sB = sA + STAGES * A_STAGE;

  // grouped rasterisation: 8 tile-rows share their B panels through L2
  const int GROUP = 8;
  const int bid = blockIdx.x;
  const int per_group = GROUP * tiles_n;
  const int group = bid / per_group;
  const int first_m = group * GROUP;
  const int gsize = min(tiles_m - first_m, GROUP);
  const int tm = first_m + (bid % per_group) % gsize;
  const int tn = (bid % per_group) / gsize;
  const int64_t m0 = (int64_t)tm * BM, n0 = (int64_t)tn * BN;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int wm = warp >> 1, wn = warp & 1;           // BM / 32 x 2 warps
  const int g = lane >> 2, q = lane & 3;

  double cre[4][4][2], cim[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      cre[i][j][0] = cre[i][j][1] = 0.0;
      cim[i][j][0] = cim[i][j][1] = 0.0;
    }

  const int KT = (int)((n + BK - 1) / BK);

  auto load_stage = [&](int stage, int kt) {
    const int64_t k0 = (int64_t)kt * BK;
    cplx* a_dst = sA + stage * A_STAGE;
    cplx* b_dst = sB + stage * B_STAGE;
#pragma unroll
    for (int i = 0; i < (BM * BK) / THREADS; ++i) {
      const int idx = tid + i * THREADS;
      const int r = idx / BK, kk = idx % BK;
      const int64_t gr = m0 + r, gk = k0 + kk;
      const bool ok = gr < n && gk < n;
      cp_async16_zfill(a_dst + r * LDA_S + kk, A + (ok ? gr * lda + gk : 0), ok);
    }
#pragma unroll
    for (int i = 0; i < (BK * BN) / THREADS; ++i) {
      const int idx = tid + i * THREADS;
      const int kk = idx / BN, c = idx % BN;
      const int64_t gk = k0 + kk, gc = n0 + c;
      const bool ok = gk < n && gc < n;
      cp_async16_zfill(b_dst + kk * LDB_S + c, B + (ok ? gk * ldb + gc : 0), ok);
    }
  };

#pragma unroll
  for (int s = 0; s < STAGES - 1; ++s) {
    if (s < KT) load_stage(s, s);
    cp_async_commit();
  }

  for (int kt = 0; kt < KT; ++kt) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    const int nxt = kt + STAGES - 1;
    if (nxt < KT) load_stage(nxt % STAGES, nxt);
    cp_async_commit();

    const cplx* a_s = sA + (kt % STAGES) * A_STAGE + (wm * 32 + g) * LDA_S + q;
    const cplx* b_s = sB + (kt % STAGES) * B_STAGE + q * LDB_S + wn * 32 + g;
#pragma unroll
    for (int ks = 0; ks < BK / 4; ++ks) {
      cplx af[4], bf[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) af[i] = a_s[i * 8 * LDA_S + ks * 4];
#pragma unroll
      for (int j = 0; j < 4; ++j) bf[j] = b_s[ks * 4 * LDB_S + j * 8];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const double nbi = -bf[j].y;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          dmma8x8x4(cre[i][j][0], cre[i][j][1], af[i].x, bf[j].x);
          dmma8x8x4(cim[i][j][0], cim[i][j][1], af[i].x, bf[j].y);
          dmma8x8x4(cre[i][j][0], cre[i][j][1], af[i].y, nbi);
          dmma8x8x4(cim[i][j][0], cim[i][j][1], af[i].y, bf[j].x);
        }
      }
    }
  }
  cp_async_wait<0>();

  // epilogue: lane holds C[row g][cols 2q, 2q+1] of every 8x8 tile
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int64_t r = m0 + wm * 32 + i * 8 + g;
    if (r >= n) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int64_t c = n0 + wn * 32 + j * 8 + 2 * q;
      cplx* dst = C + r * ldc + c;
      if (c < n) dst[0] = make_double2(cre[i][j][0], cim[i][j][0]);
      if (c + 1 < n) dst[1] = make_double2(cre[i][j][1], cim[i][j][1]);
    }
  }
}

// ---- register-resident peak probes ------------------------------------------
__global__ void __launch_bounds__(256) dmma_peak_kernel(int iters, double* __restrict__ sink) {
  double c[16][2];
#pragma unroll
  for (int i = 0; i < 16; ++i) c[i][0] = c[i][1] = 0.0;
  double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) dmma8x8x4(c[i][0], c[i][1], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i][0] + c[i][1];
  if (s == 123.456) sink[0] = s;
}

__global__ void __launch_bounds__(256) dfma_peak_kernel(int iters, double* __restrict__ sink) {
  double c[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) c[i] = i;
  const double a = 1.0 + threadIdx.x * 1e-9, b = 1e-9;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = fma(c[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i];
  if (s == 123.456) sink[0] = s;
}

}  // namespace

int launch_zgemm(int64_t n, const cplx* A, int64_t lda, const cplx* B, int64_t ldb, cplx* C, int64_t ldc,
                 cudaStream_t st) {
  // wave efficiency of the 128 x 64 tiling: tiles / (waves * SMs); below 0.93 the 64 x 64 tiling (two CTAs per SM,
  // half-cost tail) is used
  const int sms = device_sm_count();
  const int tn = (int)((n + BN - 1) / BN);
  const int64_t t128 = (int64_t)((n + 127) / 128) * tn;
  const double eff128 = (double)t128 / (double)(((t128 + sms - 1) / sms) * sms);
  // per launch (cheap): the attribute is per device, a process-wide flag would miss a second GPU
  if (eff128 >= 0.93) {
    if (cudaFuncSetAttribute(zgemm_dmma_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, zgemm_smem<128>()) !=
        cudaSuccess)
      return MAGNUS_ECUDA;
    const int tm = (int)((n + 127) / 128);
    zgemm_dmma_kernel<128><<<tm * tn, 256, zgemm_smem<128>(), st>>>(n, A, lda, B, ldb, C, ldc, tm, tn);
  } else {
    if (cudaFuncSetAttribute(zgemm_dmma_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, zgemm_smem<64>()) !=
        cudaSuccess)
      return MAGNUS_ECUDA;
    const int tm = (int)((n + 63) / 64);
    zgemm_dmma_kernel<64><<<tm * tn, 128, zgemm_smem<64>(), st>>>(n, A, lda, B, ldb, C, ldc, tm, tn);
  }
  return cudaGetLastError() == cudaSuccess ? MAGNUS_OK : MAGNUS_ECUDA;
}

int fp64_peaks(double* dmma_tflops, double* dfma_tflops, cudaStream_t st) {
  double* sink = nullptr;
  if (cudaMalloc(&sink, sizeof(double)) != cudaSuccess) return MAGNUS_ENOMEM;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int blocks = device_sm_count() * 8, iters = 4096;
  float ms = 0.f;
  double best_mma = 0.0, best_fma = 0.0;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, st);
    dmma_peak_kernel<<<blocks, 256, 0, st>>>(iters, sink);
    cudaEventRecord(e1, st);
    cudaEventSynchronize(e1);
    cudaEventElapsedTime(&ms, e0, e1);
    // per warp and iteration: 16 DMMA of 8*8*4 FMAs = 512 flop each
    const double flop = (double)blocks * 8.0 * iters * 16.0 * 512.0;
    if (rep > 0 && ms > 0.f) best_mma = fmax(best_mma, flop / (ms * 1e-3) * 1e-12);
    cudaEventRecord(e0, st);
    dfma_peak_kernel<<<blocks, 256, 0, st>>>(iters, sink);
    cudaEventRecord(e1, st);
    cudaEventSynchronize(e1);
    cudaEventElapsedTime(&ms, e0, e1);
    const double flop2 = (double)blocks * 256.0 * iters * 16.0 * 2.0;
    if (rep > 0 && ms > 0.f) best_fma = fmax(best_fma, flop2 / (ms * 1e-3) * 1e-12);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  if (cudaGetLastError() != cudaSuccess) return MAGNUS_ECUDA;
  *dmma_tflops = best_mma;
  *dfma_tflops = best_fma;
  return MAGNUS_OK;
}

}  // namespace magnus
