// common.cuh -- shared helpers of the CUDA library (sm_100a only).  Nothing in here is used by oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/epw_interp.h"

namespace epw {

typedef double2 c128;  // (re, im)

__host__ __device__ __forceinline__ c128 cmake(double re, double im) { return make_double2(re, im); }
__device__ __forceinline__ c128 cmul(c128 a, c128 b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
// acc += a * b
__device__ __forceinline__ void cfma(c128 &acc, c128 a, c128 b) {
  acc.x = fma(a.x, b.x, acc.x);
  acc.x = fma(-a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y);
  acc.y = fma(a.y, b.x, acc.y);
}
// acc += conj(a) * b
__device__ __forceinline__ void cfma_conj(c128 &acc, c128 a, c128 b) {
  acc.x = fma(a.x, b.x, acc.x);
  acc.x = fma(a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y);
  acc.y = fma(-a.y, b.x, acc.y);
}
__device__ __forceinline__ c128 cconj(c128 a) { return make_double2(a.x, -a.y); }
__device__ __forceinline__ double cabs2(c128 a) { return a.x * a.x + a.y * a.y; }

static inline int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }
static inline int64_t round_up(int64_t a, int64_t b) { return ceil_div(a, b) * b; }

// SM count of the CURRENT device (grid sizing of the streaming kernels); looked up once per device ordinal.
static inline int device_sm_count() {
  static int cache[64] = {0};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 148;
  if (dev >= 0 && dev < 64 && cache[dev] > 0) return cache[dev];
  int n = 0;
  if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return 148;
  if (dev >= 0 && dev < 64) cache[dev] = n;
  return n;
}
// grid of a grid-stride kernel: `blocks` CTAs, at most `per_sm` per SM of the current device
static inline unsigned grid_cap(int64_t blocks, int per_sm) {
  const int64_t cap = (int64_t)device_sm_count() * per_sm;
  return (unsigned)(blocks < cap ? blocks : cap);
}

// ---- DMMA GEMM operand packing (see zgemm_dmma.cu for the kernel and DESIGN.md "Data layout") -----------------
// Real embedding of a complex contraction C = A B:
//   A'[m][2r+a]     = (a ? Im : Re) A[m][r]
//   B'[2r+a][2n+b]  = a==0 ? (b ? Im : Re) B[r][n] : (b ? Re : -Im) B[r][n]
//   C'[m][2n+b]     = (b ? Im : Re) C[m][n]
// Tiles: BM = 128 rows, BN = 128 real columns (64 complex), BK = 16 real k (8 complex).
// Each (tile, k-block) chunk is 2048 doubles = 16 KB, contiguous, already in the per-lane order of the
// mma.m8n8k4.f64 fragments, so one 1-D bulk TMA copy brings it to shared memory and every fragment load is a
// conflict-free LDS.128.
constexpr int GEMM_BM = 128;
constexpr int GEMM_BN = 128;  // real columns per tile
constexpr int GEMM_BK = 16;   // real k per block
constexpr int GEMM_CHUNK = 2048;  // doubles per (tile, k-block) chunk of either operand

// offset (in doubles) inside an A chunk of element (row mr in [0,128), real k kc in [0,16))
__host__ __device__ __forceinline__ int apack_offset(int mr, int kc) {
  const int wm = mr >> 6, i = (mr >> 3) & 7, g = mr & 7;
  const int ks = kc >> 2, t = kc & 3;
  return ((((wm * 4 + ks) * 4 + (i >> 1)) * 32 + (g * 4 + t)) << 1) + (i & 1);
}
// offset inside a B chunk of element (real k kc in [0,16), real column nc in [0,128))
__host__ __device__ __forceinline__ int bpack_offset(int kc, int nc) {
  const int wn = nc >> 5, j = (nc >> 3) & 3, g = nc & 7;
  const int ks = kc >> 2, t = kc & 3;
  return ((((wn * 4 + ks) * 2 + (j >> 1)) * 32 + (g * 4 + t)) << 1) + (j & 1);
}

// ---- kernel launchers (one per .cu file) ------------------------------------------------------------------
// All are asynchronous on `st` and return the cudaGetLastError() of their launches.
cudaError_t launch_phase_table(const double *x, int64_t nx, const int32_t *R, const double *w, int nr, c128 *P,
                               cudaStream_t st);
// phases for x = k-points written directly as the packed A' operand (zero padded to [Mpad][Kpad'])
cudaError_t launch_phase_pack_a(const double *x, int64_t nx, const int32_t *R, const double *w, int nr, double *Apack,
                                cudaStream_t st);
cudaError_t launch_rp_to_q(const c128 *g, int64_t rows, int np, const c128 *Pq, int nq, c128 *g1, cudaStream_t st);
cudaError_t launch_rp_to_q_dst(const c128 *g, int64_t rows, int np, const c128 *Pq, int nq, c128 *g1, c128 *const *dst_tab,
                               cudaStream_t st);   // dst_tab != NULL: add the sums into dst_tab[iq] (peer memory allowed)
int rp_to_q_max_nq(int np);   // q-points per pass whose phase table fits shared memory (<= 8; 0 = unsupported Np)
cudaError_t launch_interp_operator(const c128 *OpR, int n, int nr, const c128 *P, int64_t nx, c128 *out,
                                   cudaStream_t st);
// `work` (may be NULL): device word that accumulates the number of plane rotations executed (matrix-rotations), so that
// the FP64 work of a solve can be stated (the sweep count is data dependent).
cudaError_t launch_eigh_batched(const c128 *A, int64_t stride_a, int n, int64_t batch, double *evals, c128 *V,
                                int sqrt_mode, int32_t *status, c128 *scratch_large, unsigned long long *work,
                                cudaStream_t st);
size_t eigh_large_scratch_bytes(int n, int64_t batch);
// same with an explicit kernel choice (EPW_EIGH_AUTO / _WARP / _THREAD / _COLS, include/epw_interp.h)
cudaError_t launch_eigh_batched_algo(const c128 *A, int64_t stride_a, int n, int64_t batch, double *evals, c128 *V,
                                     int sqrt_mode, int32_t *status, c128 *scratch_large, int algo,
                                     unsigned long long *work, cudaStream_t st);
// column-pair one-sided solver (eigh_cols.cu), n in 9..16
bool eigh_cols_supported(int n);
cudaError_t launch_eigh_cols(const c128 *A, int64_t stride_a, int n, int64_t batch, double *evals, c128 *V,
                             int sqrt_mode, int32_t *status, unsigned long long *work, cudaStream_t st);
// thread-per-matrix register-resident solver (eigh_thread.cu), n in 2..8
bool eigh_thread_supported(int n);
cudaError_t launch_eigh_thread(const c128 *A, int64_t stride_a, int n, int64_t batch, double *evals, c128 *V,
                               int sqrt_mode, int32_t *status, unsigned long long *work, cudaStream_t st);

// Build the packed B' operand for one q:
//   complex column c <  nm*nbb : sum_ka g1[ka][r][el] * e[ka + nm*nu] * amp[nu]     (c = nu*nbb + el)   (S4a hoisted)
//   complex column c >= nm*nbb : phase_qe[r] * H_R[r][el]                            (H(k+q) columns; only if ncols_h)
// g1 c128 [nm][ne][nbb]; e c128 column-major [nm][nm] (NULL = identity, amp = 1); omega f64 [nm];
// phase_qe c128 [ne] (NULL = 1).  Bpack doubles [NT][KB][2048].
cudaError_t launch_pack_b(const c128 *g1, const c128 *e, const double *omega, double omega_min, const c128 *H_R,
                          const c128 *phase_qe, int nbb, int nm, int ne, int ncols_g, int ncols_h, double *Bpack,
                          cudaStream_t st);
// generic packers for epw_zgemm (row-major complex A [M][K], B [K][N])
cudaError_t launch_pack_a_generic(const c128 *A, int64_t M, int K, double *Apack, cudaStream_t st);
cudaError_t launch_pack_b_generic(const c128 *B, int K, int N, double *Bpack, cudaStream_t st);

// C[m][n] (c128, row-major, ldc) for m in [0,M), n in [0,N); Apack holds m-tiles mt0.. of a table with KB k-blocks.
cudaError_t launch_zgemm_dmma(const double *Apack, const double *Bpack, c128 *C, int64_t M, int N, int KB, int64_t ldc,
                              int num_sms, cudaStream_t st);

// Large-Nb path (zgemm_strided.cu): C[row][col] = sum_r A[row][r] B[r][col] with A read in place,
//   A[row][r] at A + b*a_batch + (row / a_rb)*a_bs + (row % a_rb) + r*a_ks,
//   C[row][col] at C + b*c_batch + (row / c_rb)*c_bs + (row % c_rb)*c_rs + col*c_cs   (c128, or |.|^2 as f64 when abs2),
//   packed B' of problem b at Bpack + (b_gather ? b_gather[b] : b) * NT*KB*2048.
cudaError_t launch_zgemm_strided(const c128 *A, int64_t a_rb, int64_t a_bs, int64_t a_ks, int64_t a_batch,
                                 const double *Bpack, const int32_t *b_gather, void *C, int64_t c_rb, int64_t c_bs,
                                 int64_t c_rs, int64_t c_cs, int64_t c_batch, int abs2, int64_t M, int N, int K,
                                 int64_t batch, int num_sms, cudaStream_t st);
// packed B' from a strided complex operand: B[r][n] at B + b*batch_stride + r*sr + n*sn (conj optional; columns scaled
// by 1/sqrt(2 omega[n]) when omega != NULL).  Bpack doubles [batch][NT][KB][2048].
cudaError_t launch_pack_b_strided(const c128 *B, int64_t sr, int64_t sn, int64_t batch_stride, int64_t batch, int conj,
                                  const double *omega, double omega_min, int K, int N, double *Bpack, cudaStream_t st);

// Uniform-grid form of S2 / S3a (re_to_k_grid.cu): the B operand of the dense path scattered into the bounding box of
// the Re list (X [box][ncols], zeros where the list has no vector), one axis of the factorised phase, and the k-list
// a grid stands for.
cudaError_t launch_box_scatter(const c128 *g1, const c128 *e, const double *omega, double omega_min, const c128 *H_R,
                               const c128 *phase_qe, const double *w_e, const int32_t *box_idx, int64_t box_size, int nbb,
                               int nm, int ne, int ncols_g, int ncols_h, c128 *X, cudaStream_t st);
cudaError_t launch_grid_axis_phase(int N, int i0, int cnt, double shift, int lo, int L, c128 *P, cudaStream_t st);
// last axis pass of the grid form, S4b and |g|^2 as one kernel on the FP64 tensor path (grid_fused.cuh): the pass as a DMMA
// product over quads of i1, then the two rotation products; g~ never reaches HBM
bool grid_fused_supported(int nb, int nm, int L1);
// fold (may be NULL): the NEXT-4 consumer taken in the epilogue of the kernel (consumer.cu has the formula); with it g2 may be
// NULL.  out, eps_k, eps_kq relative to the first k of the chunk; eps_kq = eps_k of all k when kq_idx is given.
struct SelfEnergyFold {
  double *out;
  const double *eps_k, *eps_kq, *omega_q, *w_q;
  int64_t iq;
  double mu, kT, sigma;
};
cudaError_t launch_grid_fused(const c128 *T2, int64_t slab, int ncols, int L1, const c128 *P1c, int cnt, const c128 *Uk,
                              const c128 *Ukq, const int32_t *kq_idx, int nb, int nm, int num_sms, const uint8_t *mask,
                              double *g2, const SelfEnergyFold *fold, cudaStream_t st);
// the last axis pass alone as the DMMA product of that kernel (same conditions as grid_fused_supported)
cudaError_t launch_grid_pass_dmma(const c128 *T2, int64_t slab, int ncols, int L1, const c128 *P1c, int cnt, int nb, int nm,
                                  int num_sms, c128 *gt, int64_t gt_stride, int nbatch, int64_t in_bstride,
                                  int64_t out_bstride, cudaStream_t st);
bool grid_pass_dmma_supported(int nb, int L);   // L <= 18
// one axis pass as a streaming kernel (K = L_d <= 32); P c128 [K][N] row-major (unpacked phases)
bool axis_pass_supported(int K);
cudaError_t launch_axis_pass(const c128 *A, int64_t a_rb, int64_t a_bs, int64_t a_ks, int64_t M, const c128 *P, int K, int N,
                             c128 *C, int64_t c_rb, int64_t c_bs, int64_t c_cs, int num_sms, cudaStream_t st);
cudaError_t launch_axis_pass_p(const c128 *A, int64_t a_rb, int64_t a_bs, int64_t a_ks, int64_t M, const c128 *P,
                               int64_t p_rs, int64_t p_cs, int K, int N, c128 *C, int64_t c_rb, int64_t c_bs, int64_t c_cs,
                               int num_sms, cudaStream_t st);
cudaError_t launch_grid_klist(const int32_t N[3], const double s[3], double *k_list, cudaStream_t st);

// mask (may be NULL): uint8 per pair, 0 = skipped by the energy-window pre-screening -> zeros, no arithmetic
cudaError_t launch_rotate_g2(const c128 *gt, int64_t stride_gt, const c128 *Uk, const c128 *Ukq, const int32_t *kq_idx,
                             int nb, int nm, int64_t nk, const uint8_t *mask, double *g2, cudaStream_t st);
// Energy-window pre-screening (window.cu): mask[ik] = some band of eps_k[ik] AND some band of
// eps_{k+q}[ik] (= eps_kq[ik], or eps_k_all[kq_idx[ik]] when kq_idx is given) lies in [emin, emax].
cudaError_t launch_window_mask(const double *eps_k, const double *eps_kq, const double *eps_k_all, const int32_t *kq_idx,
                               int nb, int64_t nk, double emin, double emax, uint8_t *mask, cudaStream_t st);
// g2 blocks (E doubles each) of the skipped pairs <- 0 (kernel families that cannot skip: large-Nb path)
cudaError_t launch_zero_masked(const uint8_t *mask, int64_t nk, int64_t E, double *g2, cudaStream_t st);

bool rotate_g2_small_supported(int nb, int nm);  // Nb <= 16 and the T staging buffer of one pair fits shared memory

// Eq. 6, Bloch -> Wannier (bloch_to_wannier.cu)
cudaError_t launch_eq6_unrotate(const c128 *g, const c128 *Uk, const c128 *Ukq, const c128 *e, const double *omega, int nb,
                                int nm, int64_t nkc, int64_t nqc, c128 *tmp, c128 *gt, cudaStream_t st);
cudaError_t launch_wannier_from_bloch(const c128 *gt, const double *kc, int64_t nkc, const double *qc, int64_t nqc,
                                      const int32_t *Re, int ne, const int32_t *Rp, int np, int nb, int nm, double *wk,
                                      double *wq, c128 *Pk, c128 *Pq, double *BpackK, double *BpackQ, int32_t *zero_gather,
                                      c128 *g1, c128 *g_RR, int num_sms, cudaStream_t st);

// NEXT-4 consumer (consumer.cu): Im Sigma_nk += ... over the pairs (k = 0..nk-1, q = iq) of one |g|^2 slab
cudaError_t launch_selfenergy_accumulate(const double *g2q, const double *eps_k, const double *eps_kq,
                                         const double *eps_k_all, const int32_t *kq_idx, const double *omega_q,
                                         const double *w_q, int64_t iq, double mu, double kT, double sigma, int nb, int nm,
                                         int64_t nk, double *out, cudaStream_t st);

int probe_peaks(int device, double *out4);

}  // namespace epw
