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
// Two launch shapes of the same kernel.  One CTA per 128 x 64 tile, all of K -- used when the tile count fills
// its last wave (n = 16384: 221.4 waves).  SPLIT TAIL -- one persistent CTA per SM -- when it does not (n = 2048:
// 512 tiles on 148 SMs = 3.46 waves, half of the machine idle in the last one): CTA b first does the tiles
// b, b + SMs, ... of the full waves in the grouped raster order (so that concurrent tiles keep sharing their
// panels in L2), then the R = tiles mod SMs leftover tiles are each split into s = SMs / R ranges of K: the
// CTAs of the later ranges park their partial tile in a workspace, the CTA of the first range adds them in range
// order (a fixed order) and stores.  The tail then costs 1/s of a wave.
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

// STREAMK = false: grid = tiles, the CTA does tile blockIdx.x over all of K.
// STREAMK = true:  grid = SMs (cooperative: all CTAs resident); `split` = s; parked[b] / flags[b] belong to CTA b.
template <bool STREAMK>
__global__ void __launch_bounds__(256, 1) zgemm_dmma_kernel(int64_t n, const cplx* __restrict__ A, int64_t lda,
                                                             const cplx* __restrict__ B, int64_t ldb,
                                                             cplx* __restrict__ C, int64_t ldc, int tiles_m, int tiles_n,
                                                             double* parked, unsigned* flags, int split) {
  constexpr int BM = 128;
  constexpr int THREADS = BM * 2;              // BM / 32 x 2 warps
  constexpr int A_STAGE = BM * LDA_S;          // double2 per stage
  extern __shared__ __align__(16) unsigned char zg_smem[];
  cplx* sA = reinterpret_cast<cplx*>(zg_smem);
  cplx* sB = sA + STAGES * A_STAGE;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int wm = warp >> 1, wn = warp & 1;           // BM / 32 x 2 warps
  const int g = lane >> 2, q = lane & 3;
  const int KT = (int)((n + BK - 1) / BK);
  const int ntiles = tiles_m * tiles_n;
  const int full = STREAMK ? ntiles / (int)gridDim.x : 0;      // full waves
  const int nitems = STREAMK ? full + 1 : 1;                   // this CTA's tiles of the full waves, then its tail range

  for (int item = 0; item < nitems; ++item) {
  int tile, kt_begin = 0, kt_end = KT, piece = 0;
  if (!STREAMK) {
    tile = blockIdx.x;
  } else if (item < full) {
    tile = item * (int)gridDim.x + (int)blockIdx.x;
  } else {
    tile = full * (int)gridDim.x + (int)blockIdx.x / split;
    piece = (int)blockIdx.x % split;
    if (tile >= ntiles) break;                                 // CTAs beyond R * s have no tail work
    kt_begin = (int)((int64_t)KT * piece / split);
    kt_end = (int)((int64_t)KT * (piece + 1) / split);
  }
  // grouped rasterisation: 8 tile-rows share their B panels through L2
  const int GROUP = 8;
  const int per_group = GROUP * tiles_n;
  const int group = tile / per_group;
  const int first_m = group * GROUP;
  const int gsize = min(tiles_m - first_m, GROUP);
  const int tm = first_m + (tile % per_group) % gsize;
  const int tn = (tile % per_group) / gsize;
  const int64_t m0 = (int64_t)tm * BM, n0 = (int64_t)tn * BN;

  double cre[4][4][2], cim[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      cre[i][j][0] = cre[i][j][1] = 0.0;
      cim[i][j][0] = cim[i][j][1] = 0.0;
    }
  __syncthreads();                             // the previous segment's last slab is consumed before the ring is refilled

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

  const int KS = kt_end - kt_begin;            // slabs of this segment; ring slots count from the segment start
#pragma unroll
  for (int s = 0; s < STAGES - 1; ++s) {
    if (s < KS) load_stage(s, kt_begin + s);
    cp_async_commit();
  }

  for (int kt = 0; kt < KS; ++kt) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    const int nxt = kt + STAGES - 1;
    if (nxt < KS) load_stage(nxt % STAGES, kt_begin + nxt);
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

  if (STREAMK && piece > 0) {
    // a later range of a split tile: park the partial tile, raise the flag
    double* dst = parked + (size_t)blockIdx.x * 64 * THREADS + tid;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int s4 = (i * 4 + j) * 4;
        __stcg(dst + (size_t)(s4 + 0) * THREADS, cre[i][j][0]);
        __stcg(dst + (size_t)(s4 + 1) * THREADS, cre[i][j][1]);
        __stcg(dst + (size_t)(s4 + 2) * THREADS, cim[i][j][0]);
        __stcg(dst + (size_t)(s4 + 3) * THREADS, cim[i][j][1]);
      }
    __threadfence();
    __syncthreads();
    if (tid == 0) atomicExch(flags + blockIdx.x, 1u);
    continue;
  }
  if (STREAMK && item == full && split > 1) {
    // the first range of a split tile: add the parked ranges in range order
    for (int pc = 1; pc < split; ++pc) {
      if (tid == 0) {
        while (atomicAdd(flags + blockIdx.x + pc, 0u) == 0u) {
        }
        __threadfence();
      }
      __syncthreads();
      const double* src = parked + (size_t)(blockIdx.x + pc) * 64 * THREADS + tid;
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int s4 = (i * 4 + j) * 4;
          cre[i][j][0] += __ldcg(src + (size_t)(s4 + 0) * THREADS);
          cre[i][j][1] += __ldcg(src + (size_t)(s4 + 1) * THREADS);
          cim[i][j][0] += __ldcg(src + (size_t)(s4 + 2) * THREADS);
          cim[i][j][1] += __ldcg(src + (size_t)(s4 + 3) * THREADS);
        }
    }
  }

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
  }   // items of this CTA
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

int zgemm_scratch_alloc(ZgemmScratch* zs) {
  if (zs->parked) return MAGNUS_OK;
  const int sms = device_sm_count();
  if (cudaMalloc(&zs->parked, sizeof(double) * 64 * 256 * (size_t)sms) != cudaSuccess ||
      cudaMalloc(&zs->flags, sizeof(unsigned) * (size_t)sms) != cudaSuccess) {
    cudaGetLastError();
    zgemm_scratch_free(zs);
    return MAGNUS_ENOMEM;
  }
  return MAGNUS_OK;
}

void zgemm_scratch_free(ZgemmScratch* zs) {
  cudaFree(zs->parked);
  cudaFree(zs->flags);
  zs->parked = nullptr;
  zs->flags = nullptr;
}

// zs (nullable): the workspace of the split-tail form; without it one CTA per tile runs whatever the size
int launch_zgemm(int64_t n, const cplx* A, int64_t lda, const cplx* B, int64_t ldb, cplx* C, int64_t ldc,
                 cudaStream_t st, const ZgemmScratch* zs) {
  const int sms = device_sm_count();
  int tm = (int)((n + 127) / 128), tn = (int)((n + BN - 1) / BN);
  const int KT = (int)((n + BK - 1) / BK);
  const int64_t tiles = (int64_t)tm * tn;
  // wave efficiency of one CTA per tile: tiles / (waves * SMs); the split tail needs at least one full wave, a
  // leftover that can be split at least in two, and ranges of at least 8 slabs
  const double eff = (double)tiles / (double)(((tiles + sms - 1) / sms) * sms);
  const int R = (int)(tiles % sms);
  int split = R > 0 ? sms / R : 1;
  if (split > 4) split = 4;
  while (split > 1 && KT / split < 8) --split;
  const int smem = zgemm_smem<128>();
  // per launch (cheap): the attribute is per device, a process-wide flag would miss a second GPU
  if (cudaFuncSetAttribute(zgemm_dmma_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess ||
      cudaFuncSetAttribute(zgemm_dmma_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess)
    return MAGNUS_ECUDA;
  if (zs && zs->parked && eff < 0.93 && tiles >= sms && split > 1 &&
      cudaMemsetAsync(zs->flags, 0, sizeof(unsigned) * (size_t)sms, st) == cudaSuccess) {
    double* parked = zs->parked;
    unsigned* flags = zs->flags;
    void* args[] = {&n, &A, &lda, &B, &ldb, &C, &ldc, &tm, &tn, &parked, &flags, &split};
    if (cudaLaunchCooperativeKernel((const void*)zgemm_dmma_kernel<true>, dim3(sms), dim3(256), args, smem, st) == cudaSuccess)
      return MAGNUS_OK;
    cudaGetLastError();   // could not be launched cooperatively: one CTA per tile
  }
  int one = 1;
  zgemm_dmma_kernel<false><<<(unsigned)tiles, 256, smem, st>>>(n, A, lda, B, ldb, C, ldc, tm, tn, nullptr, nullptr, one);
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
