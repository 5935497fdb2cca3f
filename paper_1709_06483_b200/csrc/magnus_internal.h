// Internal declarations shared by the translation units of libmagnus_b200.so.
// Not installed; the public surface is include/magnus.h.
#ifndef MAGNUS_INTERNAL_H
#define MAGNUS_INTERNAL_H

#include <complex>
#include <cstdint>

#include "../../include/magnus.h"

namespace magnus {

const int kMaxDegree = 128;   // m_max (reading c6)

// ---- host_leja.cpp -------------------------------------------------------
const double* leja_points();                                  // kMaxDegree + 1 points
void divided_differences(double theta, int m, std::complex<double>* out);
void snap_interval(double* a, double* b);
void tridiag_extreme_eigenvalues(const double* alpha, const double* beta, int k, double* lo, double* hi);
int step_coefficients(int scheme, magnus_drive_fn f, void* user, double t, double tau,
                      double* coef_h1, double* h_scale, double* kappa);

// ---- error plumbing (api.cu) ----------------------------------------------
void set_error(const char* fmt, ...);

}  // namespace magnus

#ifdef __CUDACC__
#include <cuda_runtime.h>

namespace magnus {

typedef double2 cplx;   // (x, y) = (re, im), 16-byte aligned: one LDG.128 / STG.128

// M = sum_t coef[t] * A_t, up to three CSR terms sharing n (H0, H1 and, for M4, C = [H0,H1]).
struct CsrTerm {
  const int32_t* rp;
  const int32_t* ci;
  const cplx* v;
  cplx coef;
  int64_t nnz;
};
// Slice-major copy of a CSR operator, all terms merged (kernels_csr_slice.cu); owned by a handle or a single call.
struct SliceLayout {
  int64_t n = 0, nslices = 0, nslots = 0, nent = 0;
  int nterms = 0;
  int4* meta = nullptr;          // per 32-row slice: {first slot, slots, first slot of term 1, of term 2}
  int64_t* ent_ptr = nullptr;    // [nslices + 1]
  bool offsets = false;          // offset-slot layout (csr_kernel 6): slot_rec instead of slot_mask + ci
  unsigned* slot_mask = nullptr; // [nslots] rows of the slice with an entry in the slot
  uint2* slot_rec = nullptr;     // [nslots] {row mask, column - row}: all entries of a slot share column - row
  int32_t* ci = nullptr;         // [nent] columns, slot-major
  cplx* v = nullptr;             // [nent] values, same order
  bool real_values = false;      // offset-slot layout of an operator without imaginary parts: vr instead of v
  double* vr = nullptr;          // [nent] real parts of the values
};
struct CsrOp {
  int64_t n;
  int nterms;
  int unit_cap;   // max over 32-row units and terms of one term's stored entries in one unit (0 = unknown): stream kernel
  CsrTerm t[3];
  const SliceLayout* slice = nullptr;   // host pointer; set: the slice kernel may run (its terms = t[0..] in order)
};

struct DenseOp {
  int64_t n;
  int64_t ld;
  const cplx* M;
};
// Matrix-free periodic XXZ chain (shortcut, kernels_xxz.cu): M = H0 + g H1 with the entries recomputed from the row bits
struct XxzOp {
  int nspins;
  double jz;        // diagonal jz (N - 2k)
  double apair;     // 2 jxy: amplitude of an antiparallel pair flip
  double asingle;   // g hx: amplitude of a single flip
};

// Device-resident control block of one exponential (row S7): written by the
// finalize kernel after every iteration, read by the next iteration kernel
// (early exit) and by the host at chunk boundaries.
struct LejaStatus {
  int32_t done;      // 1 once the two-term test was met
  int32_t iters;     // mat-vecs actually performed (all sub-steps)
  int32_t k;         // degree reached in the current sub-step
  int32_t pad;
  double e_prev;     // e_{k-1} = |d_{k-1}| ||w_{k-1}||
  double err_est;    // e_k + e_{k-1} at the last test
  double norm_w2;    // sum |w_k|^2
  double norm_p2;    // sum |p_k|^2
};

// Small CSR problems run a whole Leja sweep in one launch of an 8-CTA cluster (kernels_csr_small.cu).
const int kSmallSweepMaxN = 4096;
const int kMidSweepMaxN = 65536;    // CSR problems up to this n run whole sweeps in one cooperative launch (kernels_csr_mid.cu)
const int kMidSweepMinN = 1024;     // ... above this n (up to it the 8-CTA cluster kernel is faster; csr_kernel 7 forces the cooperative one)
const int kDenseSweepMaxN = 4096;   // dense problems up to this n run whole sweeps in one cooperative launch
struct SweepTable {
  cplx d[kMaxDegree + 1];     // divided differences d_k (c3)
  double l[kMaxDegree + 1];   // Leja points l_k (c2)
};

// One exponential of a planned batch (the whole-sweep kernels: kernels_csr_small.cu, kernels_dense_sweep.cu).
// The host plans a batch ahead -- the Gershgorin intervals do not depend on psi -- and uploads one job per
// exponential; the kernel runs the jobs in order and stops at the first one that does not converge.
struct SweepJob {
  cplx coef[3];          // CSR: coefficient of each term; dense: coef[1].x = g of M = H0 + g H1
  cplx phase;            // e^{-i h c} (c7)
  double inv_gamma, c_over_gamma;
  int m_max;             // degrees 1..m_max are available in d[]
  int nterms;            // CSR terms this job uses (the handle's terms in order)
  int flags;             // dense: kSweepJobAssembled = M is already in place (M4, M6), no assembly
  int pad;
  cplx d[kMaxDegree + 1];   // divided differences d_k (c3)
};
const int kSweepJobAssembled = 1;

const int kMaxPartials = 4096;   // upper bound on blocks that write partial sums
const int kJobCap = 256;             // job slots on the device (a ring of kJobRing launches of kJobsPerLaunch jobs)
const int kJobsPerLaunch = 16;
const int kJobRing = kJobCap / kJobsPerLaunch;
const int kPlanCap = 4096;           // exponentials planned ahead at once (intervals, stop-test records)

struct Workspace {
  int64_t n = 0;
  cplx* w[2] = {nullptr, nullptr};   // ping-pong (row i gathers other rows' old w)
  cplx* p = nullptr;
  double* partials = nullptr;        // [2 * kMaxPartials]: sum|w|^2, sum|p|^2 per block
  double* gersh = nullptr;           // [2 * kMaxPartials]: min / max per block, then [0..1] final
  LejaStatus* status = nullptr;      // device
  unsigned* tickets = nullptr;       // device [2]: last-block tickets of the Leja and Gershgorin kernels
  LejaStatus* status_host = nullptr; // pinned
  double* ab_host = nullptr;         // pinned [2]
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
  int csr_kernel = 0;
  int64_t launches = 0;
  double leja_ms = 0.0;
  bool time_leja = false;
  void* stream_maps = nullptr;       // stream kernel: cached TMA tensor maps of the operator's terms (host)
  // planned batches (whole-sweep kernels), allocated on first use by ensure_sweep_jobs
  SweepJob* jobs = nullptr;          // device [kJobCap]
  SweepJob* jobs_host = nullptr;     // pinned [kJobCap]
  LejaStatus* status_arr = nullptr;  // device [kPlanCap]
  LejaStatus* status_arr_host = nullptr;   // pinned [kPlanCap]
  double* ab_out = nullptr;          // set by the planner while it enqueues the interval kernels of a batch
  double* ab_arr = nullptr;          // device [2 kPlanCap]: Gershgorin bounds of the batch's exponentials
  double* ab_arr_host = nullptr;     // pinned [2 kPlanCap]
  double* coef_arr = nullptr;        // device [4 kPlanCap]: per-exponential scalars of the batched Gershgorin kernels
  double* coef_arr_host = nullptr;   // pinned
  cudaEvent_t ring_ev[2 * kJobRing] = {};   // start / end of the launch that last used a ring slot
  double* leja_l = nullptr;          // device [kMaxDegree + 1]: Leja points (c2)
  unsigned* grid_bar = nullptr;      // device: grid-barrier counter of the dense sweep kernel
  double* sweep_partials = nullptr;  // device [2][2 * kMaxPartials]: per-CTA partial norms of the dense sweep kernel
};
// where the Gershgorin kernels put their final (min, max): the slot the planner set, else the workspace's own
inline double* gersh_final(const Workspace* ws) { return ws->ab_out ? ws->ab_out : ws->gersh + 2 * kMaxPartials; }
int ensure_sweep_jobs(Workspace* ws, cudaStream_t st);   // its initialisation is enqueued on st

// cudaDevAttrMultiProcessorCount of the current device (cached per device; 148 on B200)
int device_sm_count();

int workspace_alloc(Workspace* ws, int64_t n, cudaStream_t st);   // its initialisation is enqueued on st
void workspace_free(Workspace* ws);

struct LejaParams {
  double tol;
  double theta_max;
  int m_max;
};

// ---- kernels_common.cu ------------------------------------------------------
void launch_leja_init(const cplx* v, cplx* w, cplx* p, int64_t n, cplx d0, double abs_d0, Workspace* ws,
                      cudaStream_t st);
void launch_leja_finish(const cplx* p, cplx* out, int64_t n, cplx phase, cudaStream_t st, Workspace* ws);
void launch_scale_copy(const cplx* in, cplx* out, int64_t n, cplx phase, cudaStream_t st, Workspace* ws);

// ---- kernels_csr.cu ---------------------------------------------------------
// The iteration kernels also run the stop test (S7) in their last block: abs_dk = |d_k|, tol (c6).
// returns the number of blocks that wrote partials
int launch_csr_gershgorin(const CsrOp& op, Workspace* ws, cudaStream_t st);
// cached row statistics of one term / overlap test of the terms / bounds from the cached statistics
void launch_csr_rowstats(const CsrTerm& T, int64_t n, double* r, cplx* diag, cudaStream_t st);
void launch_csr_overlap(const CsrOp& op, int* flag, cudaStream_t st);
int launch_csr_gershgorin_cached(const CsrOp& op, const double* const* r, const cplx* const* diag, Workspace* ws,
                                 cudaStream_t st);
// the bounds of E exponentials (coefficients 1, g_e, -i kappa_e; coefs_dev[4e..4e+2] = g, kappa, terms) in one launch
void launch_csr_gershgorin_cached_batch(int64_t n, const double* const* r, const cplx* const* diag, int nterms_max,
                                        const double* coefs_dev, int E, double* ab_out, Workspace* ws, cudaStream_t st);
int launch_csr_leja_iter(const CsrOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma, double shift,
                         cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st);
int csr_commutator(const magnus_matrix* A, const magnus_matrix* B, int64_t cap, int64_t* nnz_out, int32_t* rp_out,
                   int32_t* ci_out, cplx* v_out, cudaStream_t st);
// same, handing over freshly cudaMalloc'ed arrays (caller frees with cudaFree)
int csr_commutator_owned(const magnus_matrix* A, const magnus_matrix* B, int32_t** rp, int32_t** ci, cplx** v,
                         int64_t* nnz, cudaStream_t st);
int csr_hermitian_check(const magnus_matrix* A, cudaStream_t st, double* max_violation);

// ---- kernels_csr_stream.cu --------------------------------------------------
// warp-specialised kernel for large n: bulk-copy (TMA) ring + mbarriers, see the file header
int csr_unit_cap(const CsrOp& op, cudaStream_t st, int* cap_out);      // synchronises the stream
bool csr_stream_supported(const CsrOp& op);
void stream_maps_free(Workspace* ws);
// row-block structure (a private buffer per warp) with TMA staging
bool csr_rowtma_supported(const CsrOp& op);
int launch_csr_leja_iter_rowtma(const CsrOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma,
                                double shift, cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st);
int launch_csr_leja_iter_stream(const CsrOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma,
                                double shift, cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st);

// ---- kernels_csr_slice.cu ---------------------------------------------------
// slice-major copy of op's terms (coefficients ignored); an error leaves *out empty and callers keep the CSR kernels
// offsets: slots stored as {row mask, column - row} records and no column array (csr_kernel 6)
// allow_real: store only the real parts when no stored value has an imaginary part (offset-slot layout)
int slice_layout_build(const CsrOp& op, SliceLayout* out, cudaStream_t st, bool offsets, bool allow_real = false);
// which slice layout a csr_kernel option asks for: 0 none, 1 with columns (5, 5000..5999), 2 offset slots (6, 6000..6999;
// 6500..6999: real-part storage when the operator has no imaginary parts, tuning code = the option - 500)
inline int slice_layout_kind(int csr_kernel) {
  if (csr_kernel == 5 || (csr_kernel >= 5000 && csr_kernel < 6000)) return 1;
  if (csr_kernel == 6 || (csr_kernel >= 6000 && csr_kernel < 7000)) return 2;
  return 0;
}
void slice_layout_free(SliceLayout* L);
int launch_csr_leja_iter_slice(const CsrOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma, double shift,
                               cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st);

// ---- kernels_lanczos.cu (shortcut: tight spectral interval) ------------------
void launch_lanczos_start(const cplx* v, cplx* q, cplx* qprev, int64_t n, double* scal, Workspace* ws, cudaStream_t st);
void launch_lanczos_step(cplx* u, const cplx* q, cplx* qprev, int64_t n, double* scal, int j, int m, Workspace* ws,
                         cudaStream_t st);

// ---- kernels_xxz.cu ---------------------------------------------------------
int launch_xxz_leja_iter(const XxzOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma, double shift,
                         cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st);
void xxz_gershgorin(const XxzOp& op, double* a, double* b);   // host, closed form

// ---- kernels_csr_small.cu ---------------------------------------------------
// one sub-step sweep (S5-S8) in one launch; on success status->done = 1, status->k = iterations and out is
// written; if tab's m_max iterations do not meet tol, status->pad = 1 and out is left untouched
int launch_csr_leja_sweep_small(const CsrOp& op, const cplx* v, cplx* out, double inv_gamma, double c_over_gamma,
                                 double tol, int m_max, cplx phase, const SweepTable& tab, Workspace* ws,
                                 cudaStream_t st);
// a planned batch in ONE launch: psi <- exp(job[njobs-1]) ... exp(job[0]) psi; status[e] per job (zeroed by the
// caller); stops at the first job that does not converge within its m_max (status[e].pad = 1, psi = state before it)
// gate (nullable): the stop-test record of the job before jobs[0]; the launch does nothing unless that job converged
int launch_csr_leja_sweep_small_jobs(const CsrOp& op, cplx* psi, const SweepJob* jobs, int njobs, const double* leja_l,
                                      double tol, LejaStatus* status, const LejaStatus* gate, Workspace* ws,
                                      cudaStream_t st);

// ---- kernels_csr_mid.cu -----------------------------------------------------
bool csr_mid_sweep_supported(int64_t n, int csr_kernel);   // csr_kernel 0: by size; 7: forced (any n <= kMidSweepMaxN)
int launch_csr_leja_sweep_mid_jobs(const CsrOp& op, cplx* psi, const SweepJob* jobs, int njobs, double tol,
                                   LejaStatus* status, const LejaStatus* gate, Workspace* ws, cudaStream_t st);
int launch_csr_leja_sweep_mid(const CsrOp& op, const cplx* v, cplx* out, double inv_gamma, double c_over_gamma, double tol,
                              int m_max, cplx phase, const SweepTable& tab, Workspace* ws, cudaStream_t st);

// ---- kernels_dense.cu -------------------------------------------------------
int launch_dense_gershgorin(const DenseOp& op, Workspace* ws, cudaStream_t st);
// M = A + g*B (elementwise) fused with the Gershgorin row bounds of M
int launch_dense_assemble(int64_t n, const cplx* A, int64_t lda, const cplx* B, int64_t ldb, double g, cplx* M,
                          Workspace* ws, cudaStream_t st);
// A1 = H0 + f1 H1, A2 = H0 + f2 H1 in one pass
void launch_dense_assemble2(int64_t n, const cplx* H0, int64_t ld0, const cplx* H1, int64_t ld1, double f1, double f2,
                            cplx* A1, cplx* A2, Workspace* ws, cudaStream_t st);
// Om = wa A1 + wb A2 - i kappa (P - P^H), written over A1, fused with Gershgorin bounds (row D4; M4: wa = wb = 1/2)
int launch_dense_omega(int64_t n, cplx* A1, const cplx* A2, const cplx* P, double wa, double wb, double kappa,
                       Workspace* ws, cudaStream_t st);
// K = P + s P^H (s = -1: P - P^H)
void launch_dense_antiherm(int64_t n, const cplx* P, cplx* K, double s, cudaStream_t st);
struct LinComb {
  const cplx* x[4];
  cplx c[4];
};
void launch_dense_lincomb(int64_t n, cplx* out, LinComb lc, Workspace* ws, cudaStream_t st);
void launch_csr_to_dense(int64_t n, const int32_t* rp, const int32_t* ci, const cplx* v, cplx* A, cudaStream_t st);
// planned batches on medium dense problems (kernels_dense_sweep.cu, dense_gershgorin_batch_kernel)
int launch_dense_gershgorin_batch(int64_t n, const cplx* H0, int64_t ld0, const cplx* H1, int64_t ld1,
                                  const double* coefs_dev, int E, double* ab_keys_dev, Workspace* ws, cudaStream_t st);
void dense_gershgorin_batch_decode(const double* keys_host, int E, double* ab);
bool dense_sweep_supported(int64_t n);
int launch_dense_leja_sweep_jobs(int64_t n, const cplx* H0, int64_t ld0, const cplx* H1, int64_t ld1, cplx* M, cplx* psi,
                                 const SweepJob* jobs, int njobs, double tol, LejaStatus* status, const LejaStatus* gate,
                                 Workspace* ws, cudaStream_t st);
int launch_dense_leja_sweep(const DenseOp& op, const cplx* v, cplx* out, double inv_gamma, double c_over_gamma,
                            double tol, int m_max, cplx phase, const SweepTable& tab, Workspace* ws, cudaStream_t st);
int launch_dense_leja_iter(const DenseOp& op, const cplx* w_in, cplx* w_out, cplx* p, double inv_gamma, double shift,
                           cplx dk, double abs_dk, double tol, Workspace* ws, cudaStream_t st);
int dense_hermitian_check(const DenseOp& op, cudaStream_t st, double* max_violation);

// ---- zgemm_dmma.cu ----------------------------------------------------------
// workspace of the split-tail form of the GEMM (partial tiles parked by the later K ranges of a split tile, one flag each)
struct ZgemmScratch {
  double* parked = nullptr;
  unsigned* flags = nullptr;
};
int zgemm_scratch_alloc(ZgemmScratch* zs);
void zgemm_scratch_free(ZgemmScratch* zs);
int launch_zgemm(int64_t n, const cplx* A, int64_t lda, const cplx* B, int64_t ldb, cplx* C, int64_t ldc,
                 cudaStream_t st, const ZgemmScratch* zs = nullptr);
int fp64_peaks(double* dmma_tflops, double* dfma_tflops, cudaStream_t st);

}  // namespace magnus
#endif  // __CUDACC__

#endif  // MAGNUS_INTERNAL_H
