// Dense kernels: assembly of H(t) fused with the Gershgorin row bounds (rows
// S2+S3), the Omega_H assembly of M4 (row D4), and the fused dense Leja
// iteration (row S6).  Row-major complex128.
// P:n = PAPER.md line n; c1..c7 = readings in DESIGN.md section 3.
#include <cstring>

#include "magnus_internal.h"
#include "device_utils.cuh"
#include "leja_finalize.cuh"

namespace magnus {

namespace {

constexpr int DW = 8;   // warps per block; one row per warp

// ---------------------------------------------------------------------------
// S2 + S3: M = A + g B (P:256-258, P:262 l.3-4 "A_1 = H_1 + d_1 H_2"), one warp per
// row with 128-bit coalesced accesses, fused with the Gershgorin row bounds
// lo_i = Re M_ii - sum_{j != i} |M_ij|, hi_i = Re M_ii + ...  (c4).
// WRITE = false, B = nullptr: bounds of A only (leja_expmv on a dense matrix).
// ---------------------------------------------------------------------------
template <bool HAS_B, bool WRITE>
__global__ void __launch_bounds__(DW * 32) dense_assemble_kernel(int64_t n, const cplx* __restrict__ A, int64_t lda,
                                                                  const cplx* __restrict__ B, int64_t ldb, double g,
                                                                  cplx* __restrict__ M, double* out, unsigned* ticket,
                                                                  double* fin) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double lo = INFINITY, hi = -INFINITY;
  for (int64_t row = (int64_t)blockIdx.x * DW + warp; row < n; row += (int64_t)gridDim.x * DW) {
    const cplx* a = A + row * lda;
    const cplx* b = HAS_B ? B + row * ldb : nullptr;
    cplx* m = WRITE ? M + row * n : nullptr;
    double R = 0.0, d = 0.0;
#pragma unroll 4
    for (int64_t j = lane; j < n; j += 32) {
      cplx z = a[j];
      if (HAS_B) {
        const cplx y = b[j];
        z.x = fma(g, y.x, z.x);
        z.y = fma(g, y.y, z.y);
      }
      if (WRITE) m[j] = z;
      if (j == row) d = z.x; else R += hypot(z.x, z.y);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      R += shfl_xor_d(R, o);
      d += shfl_xor_d(d, o);     // exactly one lane holds the diagonal, the others 0
    }
    lo = fmin(lo, d - R);
    hi = fmax(hi, d + R);
  }
  block_reduce_minmax<DW * 32>(lo, hi);
  if (threadIdx.x == 0) {
    out[2 * blockIdx.x] = lo;
    out[2 * blockIdx.x + 1] = hi;
  }
  if (last_block_ticket(ticket)) minmax_finalize_warp0(out, gridDim.x, fin);
}

// A1 = H0 + f1 H1, A2 = H0 + f2 H1 (P:262 l.3-4), one pass over H0 and H1.
__global__ void __launch_bounds__(256) dense_assemble2_kernel(int64_t n, const cplx* __restrict__ H0, int64_t ld0,
                                                               const cplx* __restrict__ H1, int64_t ld1, double f1,
                                                               double f2, cplx* __restrict__ A1,
                                                               cplx* __restrict__ A2) {
  const int64_t total = n * n;
  for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (int64_t)gridDim.x * blockDim.x) {
    const int64_t i = q / n, j = q - i * n;
    const cplx a = H0[i * ld0 + j], b = H1[i * ld1 + j];
    A1[q] = make_double2(fma(f1, b.x, a.x), fma(f1, b.y, a.y));
    A2[q] = make_double2(fma(f2, b.x, a.x), fma(f2, b.y, a.y));
  }
}

// ---------------------------------------------------------------------------
// D4: Omega_H = (A1 + A2)/2 - i kappa (P - P^H)  (P:262 l.5, 8, 9 with A = -iH; c1),
// written over A1, fused with the Gershgorin bounds of Omega_H.  P^H is read
// through a 32x33 shared-memory tile so that both P reads are coalesced.
// Block = 32 x 8 threads, owns a strip of 32 rows.
// ---------------------------------------------------------------------------
// General form Omega = wa A1 + wb A2 - i kappa (P - P^H): M4 has wa = wb = 1/2; M6 uses it with
// A1 = H(t2), A2 = H1 and P = L R, see magnus_step.
__global__ void __launch_bounds__(256) dense_omega_kernel(int64_t n, cplx* __restrict__ A1, const cplx* __restrict__ A2,
                                                           const cplx* __restrict__ P, double wa, double wb,
                                                           double kappa, double* out, unsigned* ticket,
                                                           double* fin) {
  __shared__ cplx tile[32][33];
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  double lo = INFINITY, hi = -INFINITY;
  const int64_t nstrips = (n + 31) / 32;
  for (int64_t ib = blockIdx.x; ib < nstrips; ib += gridDim.x) {
    double R[4] = {0.0, 0.0, 0.0, 0.0}, D[4] = {0.0, 0.0, 0.0, 0.0};
    for (int64_t jb = 0; jb < nstrips; ++jb) {
      // tile[a][b] = P[jb*32 + a][ib*32 + b]
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int64_t r = jb * 32 + ty + 8 * k, c = ib * 32 + tx;
        tile[ty + 8 * k][tx] = (r < n && c < n) ? P[r * n + c] : make_double2(0.0, 0.0);
      }
      __syncthreads();
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int64_t i = ib * 32 + ty + 8 * k, j = jb * 32 + tx;
        if (i < n && j < n) {
          const cplx pij = P[i * n + j];
          const cplx pji = tile[tx][ty + 8 * k];
          const double kx = pij.x - pji.x, ky = pij.y + pji.y;      // K = P - P^H
          const cplx a1 = A1[i * n + j], a2 = A2[i * n + j];
          cplx om;
          om.x = wa * a1.x + wb * a2.x + kappa * ky;                 // -i kappa (kx + i ky) = kappa (ky - i kx)
          om.y = wa * a1.y + wb * a2.y - kappa * kx;
          A1[i * n + j] = om;
          if (i == j) D[k] = om.x; else R[k] += hypot(om.x, om.y);
        }
      }
      __syncthreads();
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      double r = R[k], d = D[k];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        r += shfl_xor_d(r, o);
        d += shfl_xor_d(d, o);
      }
      if (ib * 32 + ty + 8 * k < n) {
        lo = fmin(lo, d - r);
        hi = fmax(hi, d + r);
      }
    }
  }
  block_reduce_minmax<256>(lo, hi);
  if (threadIdx.x == 0) {
    out[2 * blockIdx.x] = lo;
    out[2 * blockIdx.x + 1] = hi;
  }
  if (last_block_ticket(ticket)) minmax_finalize_warp0(out, gridDim.x, fin);
}

// K = P + s P^H, s = -1 (K = P - P^H: the commutator of two Hermitian or two anti-Hermitian factors of P) or
// s = +1 (the commutator of a Hermitian with an anti-Hermitian factor).
__global__ void __launch_bounds__(256) dense_antiherm_kernel(int64_t n, const cplx* __restrict__ P,
                                                              cplx* __restrict__ K, double s) {
  __shared__ cplx tile[32][33];
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const int64_t ib = blockIdx.y, jb = blockIdx.x;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int64_t r = jb * 32 + ty + 8 * k, c = ib * 32 + tx;
    tile[ty + 8 * k][tx] = (r < n && c < n) ? P[r * n + c] : make_double2(0.0, 0.0);
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int64_t i = ib * 32 + ty + 8 * k, j = jb * 32 + tx;
    if (i < n && j < n) {
      const cplx pij = P[i * n + j];
      const cplx pji = tile[tx][ty + 8 * k];
      K[i * n + j] = make_double2(pij.x + s * pji.x, pij.y - s * pji.y);
    }
  }
}

// ---------------------------------------------------------------------------
// S6 dense: one warp per row.  Lanes stream the row with 128-bit loads that
// bypass L1 and are evict-first in L2 (the matrix is read once per iteration);
// w (16 n bytes) is re-read by every warp and served by L1/L2.
//   y_i = sum_j M_ij w_j;  w+_i = inv_gamma y_i - shift w_i;  p_i += d_k w+_i   (c5)
// plus the block partials of sum |w+|^2, sum |p|^2 for the stop test (S7).
// ---------------------------------------------------------------------------
constexpr int GU = 8;   // independent 128-bit loads in flight per lane

__global__ void __launch_bounds__(DW * 32) dense_leja_iter_kernel(DenseOp op, const cplx* __restrict__ w_in,
                                                                   cplx* __restrict__ w_out, cplx* __restrict__ p,
                                                                   double inv_gamma, double shift, cplx dk,
                                                                   double abs_dk, double tol, LejaStatus* status,
                                                                   double* partials, unsigned* ticket) {
  if (status->done) return;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint64_t pol = policy_evict_first();
  const int64_t n = op.n;
  double sw = 0.0, sp = 0.0;
  for (int64_t row = (int64_t)blockIdx.x * DW + warp; row < n; row += (int64_t)gridDim.x * DW) {
    const cplx* __restrict__ m = op.M + row * op.ld;
    cplx acc[2] = {make_double2(0.0, 0.0), make_double2(0.0, 0.0)};
    int64_t j = lane;
    for (; j + 32 * (GU - 1) < n; j += 32 * GU) {
      cplx mv[GU], xv[GU];
#pragma unroll
      for (int u = 0; u < GU; ++u) mv[u] = ld_stream(m + j + 32 * u, pol);
#pragma unroll
      for (int u = 0; u < GU; ++u) xv[u] = w_in[j + 32 * u];
#pragma unroll
      for (int u = 0; u < GU; ++u) cfma(acc[u & 1], mv[u], xv[u]);
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
      sw += wn.x * wn.x + wn.y * wn.y;
      sp += pi.x * pi.x + pi.y * pi.y;
    }
  }
  block_reduce_sum2<DW * 32>(sw, sp);
  if (threadIdx.x == 0) {
    partials[2 * blockIdx.x] = sw;
    partials[2 * blockIdx.x + 1] = sp;
  }
  if (last_block_ticket(ticket)) leja_finalize_warp0(partials, gridDim.x, abs_dk, tol, false, status);   // S7
}

__global__ void __launch_bounds__(256) dense_lincomb_kernel(int64_t total, cplx* __restrict__ out, LinComb lc) {
  for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (int64_t)gridDim.x * blockDim.x) {
    cplx acc = make_double2(0.0, 0.0);
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (lc.x[k]) cfma(acc, lc.c[k], lc.x[k][q]);
    out[q] = acc;
  }
}

// one warp per row
__global__ void __launch_bounds__(256) csr_to_dense_kernel(int64_t n, const int32_t* __restrict__ rp,
                                                            const int32_t* __restrict__ ci, const cplx* __restrict__ v,
                                                            cplx* __restrict__ A) {
  const int64_t row = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  if (row >= n) return;
  for (int q = rp[row] + (threadIdx.x & 31); q < rp[row + 1]; q += 32) A[row * n + ci[q]] = v[q];
}

// Sampled Hermitian check: pseudo-random (i, j) pairs, largest |M_ij - conj(M_ji)|.
__global__ void dense_hermitian_check_kernel(DenseOp op, int64_t samples, double* __restrict__ worst) {
  double bad = 0.0;
  for (int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; s < samples; s += (int64_t)gridDim.x * blockDim.x) {
    uint64_t z = (uint64_t)s * 0x9E3779B97F4A7C15ull + 0x632BE59BD9B4E019ull;
    z ^= z >> 29;
    z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 32;
    const int64_t i = (int64_t)(z % (uint64_t)op.n), j = (int64_t)((z >> 20) % (uint64_t)op.n);
    const cplx a = op.M[i * op.ld + j], b = op.M[j * op.ld + i];
    bad = fmax(bad, fmax(fabs(a.x - b.x), fabs(a.y + b.y)));
  }
  double neg = -bad, dummy = -INFINITY;
  block_reduce_minmax<256>(neg, dummy);
  if (threadIdx.x == 0) worst[blockIdx.x] = -neg;
}

// ---------------------------------------------------------------------------
// S3 for a planned batch: the Gershgorin bounds of M_e = H0 + g_e H1 for E exponentials from ONE pass over
// H0 and H1 (the bounds do not depend on psi, so a run of steps can be planned ahead).  A CTA takes a row,
// every thread keeps its entries of the row (n <= 256 * DGB_EPT) in registers and walks the g_e in chunks
// of DGB_CH; a chunk's row sums are reduced over the block and folded into keys[e] (min) / keys[E + e] (max)
// with integer atomics on an order-preserving encoding of the double -- min and max do not depend on the
// order, so the result is deterministic.  |z| = sqrt(re^2 + im^2) (cabs_fast); the last-ulp difference to
// hypot is absorbed by the interval snapping (reading c4).
// ---------------------------------------------------------------------------
constexpr int DGB_EPT = 16, DGB_CH = 8;

__device__ __forceinline__ unsigned long long ordered_key(double x) {
  const unsigned long long u = (unsigned long long)__double_as_longlong(x);
  return (u >> 63) ? ~u : (u | 0x8000000000000000ull);
}

__global__ void __launch_bounds__(256) dense_gershgorin_batch_kernel(int n, const cplx* __restrict__ H0, int64_t ld0,
                                                                      const cplx* __restrict__ H1, int64_t ld1,
                                                                      const double* __restrict__ coefs, int E,
                                                                      unsigned long long* keys) {
  __shared__ double s_part[8][DGB_CH];
  __shared__ double s_diag[2];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  for (int row = blockIdx.x; row < n; row += gridDim.x) {
    cplx a[DGB_EPT], b[DGB_EPT];
    const cplx* pa = H0 + (int64_t)row * ld0;
    const cplx* pb = H1 + (int64_t)row * ld1;
#pragma unroll
    for (int i = 0; i < DGB_EPT; ++i) {
      const int j = tid + 256 * i;
      a[i] = j < n ? ld_gather_na(pa + j) : make_double2(0.0, 0.0);
      b[i] = j < n ? ld_gather_na(pb + j) : make_double2(0.0, 0.0);
      if (j == row) {                      // the diagonal enters the centre, not the radius
        s_diag[0] = a[i].x;
        s_diag[1] = b[i].x;
        a[i] = make_double2(0.0, 0.0);
        b[i] = make_double2(0.0, 0.0);
      }
    }
    __syncthreads();
    const double da = s_diag[0], db = s_diag[1];
    for (int e0 = 0; e0 < E; e0 += DGB_CH) {
      double R[DGB_CH];
#pragma unroll
      for (int c = 0; c < DGB_CH; ++c) {
        const double g = coefs[4 * min(e0 + c, E - 1)];
        double r = 0.0;
#pragma unroll
        for (int i = 0; i < DGB_EPT; ++i) {
          const double zx = fma(g, b[i].x, a[i].x), zy = fma(g, b[i].y, a[i].y);
          r += sqrt(fma(zx, zx, zy * zy));
        }
        R[c] = r;
      }
#pragma unroll
      for (int c = 0; c < DGB_CH; ++c) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) R[c] += shfl_xor_d(R[c], o);
        if (lane == 0) s_part[warp][c] = R[c];
      }
      __syncthreads();
      if (tid < DGB_CH && e0 + tid < E) {
        double r = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) r += s_part[w][tid];
        const double d = fma(coefs[4 * (e0 + tid)], db, da);
        atomicMin(keys + e0 + tid, ordered_key(d - r));
        atomicMax(keys + E + e0 + tid, ordered_key(d + r));
      }
      __syncthreads();
    }
  }
}

int row_grid(int64_t n) {
  int64_t g = (n + DW - 1) / DW;
  if (g > kMaxPartials) g = kMaxPartials;
  return (int)g;
}

}  // namespace

int launch_dense_gershgorin(const DenseOp& op, Workspace* ws, cudaStream_t st) {
  const int g = row_grid(op.n);
  dense_assemble_kernel<false, false><<<g, DW * 32, 0, st>>>(op.n, op.M, op.ld, nullptr, 0, 0.0, nullptr, ws->gersh,
                                                             ws->tickets + 1, gersh_final(ws));
  ws->launches += 1;
  return g;
}

// keys (device, 2 E entries) come back as ordered keys: dense_gershgorin_batch_decode turns a host copy into doubles
int launch_dense_gershgorin_batch(int64_t n, const cplx* H0, int64_t ld0, const cplx* H1, int64_t ld1,
                                  const double* coefs_dev, int E, double* ab_keys_dev, Workspace* ws, cudaStream_t st) {
  if (n > 256 * DGB_EPT) return MAGNUS_EINVAL;
  unsigned long long* keys = reinterpret_cast<unsigned long long*>(ab_keys_dev);
  if (cudaMemsetAsync(keys, 0xFF, sizeof(unsigned long long) * (size_t)E, st) != cudaSuccess ||
      cudaMemsetAsync(keys + E, 0, sizeof(unsigned long long) * (size_t)E, st) != cudaSuccess)
    return MAGNUS_ECUDA;
  int64_t g = n;
  if (g > (int64_t)device_sm_count() * 8) g = (int64_t)device_sm_count() * 8;
  dense_gershgorin_batch_kernel<<<(int)g, 256, 0, st>>>((int)n, H0, ld0, H1, ld1, coefs_dev, E, keys);
  ws->launches += 1;
  return MAGNUS_OK;
}

// host: keys[e] (min), keys[E + e] (max) -> ab[2e], ab[2e + 1]
void dense_gershgorin_batch_decode(const double* keys_host, int E, double* ab) {
  auto dec = [](double kd) {
    unsigned long long k;
    memcpy(&k, &kd, sizeof k);
    const unsigned long long u = (k >> 63) ? (k & 0x7FFFFFFFFFFFFFFFull) : ~k;
    double x;
    memcpy(&x, &u, sizeof x);
    return x;
  };
  for (int e = 0; e < E; ++e) {
    ab[2 * e] = dec(keys_host[e]);
    ab[2 * e + 1] = dec(keys_host[E + e]);
  }
}

int launch_dense_assemble(int64_t n, const cplx* A, int64_t lda, const cplx* B, int64_t ldb, double g, cplx* M,
                          Workspace* ws, cudaStream_t st) {
  const int grid = row_grid(n);
  dense_assemble_kernel<true, true><<<grid, DW * 32, 0, st>>>(n, A, lda, B, ldb, g, M, ws->gersh, ws->tickets + 1,
                                                              gersh_final(ws));
  ws->launches += 1;
  return grid;
}

void launch_dense_assemble2(int64_t n, const cplx* H0, int64_t ld0, const cplx* H1, int64_t ld1, double f1, double f2,
                            cplx* A1, cplx* A2, Workspace* ws, cudaStream_t st) {
  int64_t g = (n * n + 255) / 256;
  if (g > (int64_t)device_sm_count() * 16) g = (int64_t)device_sm_count() * 16;
  dense_assemble2_kernel<<<(int)g, 256, 0, st>>>(n, H0, ld0, H1, ld1, f1, f2, A1, A2);
  ws->launches += 1;
}

int launch_dense_omega(int64_t n, cplx* A1, const cplx* A2, const cplx* P, double wa, double wb, double kappa,
                       Workspace* ws, cudaStream_t st) {
  int64_t g = (n + 31) / 32;
  if (g > kMaxPartials) g = kMaxPartials;
  dense_omega_kernel<<<(int)g, 256, 0, st>>>(n, A1, A2, P, wa, wb, kappa, ws->gersh, ws->tickets + 1, gersh_final(ws));
  ws->launches += 1;
  return (int)g;
}

void launch_dense_antiherm(int64_t n, const cplx* P, cplx* K, double s, cudaStream_t st) {
  const unsigned t = (unsigned)((n + 31) / 32);
  dense_antiherm_kernel<<<dim3(t, t), 256, 0, st>>>(n, P, K, s);
}

// out = c0 X0 + c1 X1 + c2 X2 + c3 X3, elementwise on n x n row-major matrices (null inputs are skipped)
void launch_dense_lincomb(int64_t n, cplx* out, LinComb lc, Workspace* ws, cudaStream_t st) {
  int64_t g = (n * n + 255) / 256;
  if (g > (int64_t)device_sm_count() * 16) g = (int64_t)device_sm_count() * 16;
  dense_lincomb_kernel<<<(int)g, 256, 0, st>>>(n * n, out, lc);
  ws->launches += 1;
}

// A = CSR matrix written out densely (row-major, zero-filled first)
void launch_csr_to_dense(int64_t n, const int32_t* rp, const int32_t* ci, const cplx* v, cplx* A, cudaStream_t st) {
  cudaMemsetAsync(A, 0, sizeof(cplx) * (size_t)n * (size_t)n, st);
  int64_t g = (n + 7) / 8;
  csr_to_dense_kernel<<<(int)g, 256, 0, st>>>(n, rp, ci, v, A);
}

int launch_dense_leja_iter(const DenseOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma, double shift,
                           cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st) {
  const int g = row_grid(op.n);
  dense_leja_iter_kernel<<<g, DW * 32, 0, st>>>(op, w_in, w_out, p, inv_gamma, shift, dk, abs_dk, tol, ws->status,
                                                ws->partials, ws->tickets);
  ws->launches += 1;
  return g;
}

int dense_hermitian_check(const DenseOp& op, cudaStream_t st, double* max_violation) {
  const int grid = 64;
  double* worst = nullptr;
  if (cudaMalloc(&worst, sizeof(double) * grid) != cudaSuccess) return MAGNUS_ENOMEM;
  dense_hermitian_check_kernel<<<grid, 256, 0, st>>>(op, 1 << 20, worst);
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
