// rotate_g2.cu -- S4b: band rotation and |g|^2 (Eq. 10: U_{mm'k+q} ... U*_{nn'k}; with paper-U = V^dagger,
// V the eigenvector columns, reading G4):
//     g_{mn nu}(k,q) = sum_{m'n'} conj(Ukq[m',m]) g~_{m'n' nu}(k,q) Uk[n',n],     out = |g_{mn nu}|^2.
// The mode rotation and the 1/sqrt(2 omega) amplitude were already applied to g(Re,q) (pack.cu), so g~ arrives in
// the mode basis.  Two successive small matrix products per mode ("successive multiplication"):
//     T[nu][n][m'] = sum_n' g~[nu][n'][m'] Uk[n'][n]          then      g[nu][n][m] = sum_m' conj(Ukq[m'][m]) T[nu][n][m'].
// Small-Nb kernel: one CTA per (k,q) pair, everything staged in shared memory; 2 Nb^3 Nm complex MACs per pair on
// the plain FP64 pipe; reads 16 (Nb^2 Nm + 2 Nb^2) bytes and writes 8 Nb^2 Nm bytes per pair.
#include "common.cuh"

namespace epw {

constexpr int ROT_THREADS = 128;

__global__ void __launch_bounds__(ROT_THREADS)
    rotate_g2_small_kernel(const c128 *__restrict__ gt, int64_t stride_gt, const c128 *__restrict__ Uk,
                           const c128 *__restrict__ Ukq, const int32_t *__restrict__ kq_idx, int nb, int nm,
                           int64_t nk, double *__restrict__ g2) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int nbb = nb * nb, E = nbb * nm;
  c128 *sG = reinterpret_cast<c128 *>(smem_raw);  // [nu][n'][m']
  c128 *sT = sG + E;                              // [nu][n][m']
  c128 *sUk = sT + E;                             // [n][n'] column-major: Uk[n' + nb*n]
  c128 *sUkqH = sUk + nbb;                        // conj(Ukq[m'][m]) stored at [m'][m] (m fastest)
  for (int64_t ik = blockIdx.x; ik < nk; ik += gridDim.x) {
    const c128 *src = gt + ik * stride_gt;
    for (int e = threadIdx.x; e < E; e += ROT_THREADS) sG[e] = src[e];
    const c128 *uk = Uk + ik * nbb;
    const c128 *ukq = Ukq + (kq_idx ? (int64_t)kq_idx[ik] : ik) * nbb;
    for (int e = threadIdx.x; e < nbb; e += ROT_THREADS) {
      sUk[e] = uk[e];
      const int mp = e % nb, m = e / nb;  // ukq[e] = Ukq[m' + nb*m]
      sUkqH[m + nb * mp] = cconj(ukq[e]);
    }
    __syncthreads();
    for (int e = threadIdx.x; e < E; e += ROT_THREADS) {
      const int mp = e % nb, n = (e / nb) % nb, nu = e / nbb;
      c128 acc = cmake(0.0, 0.0);
      const c128 *gcol = sG + nu * nbb + mp;
      const c128 *ucol = sUk + nb * n;
      for (int np_ = 0; np_ < nb; np_++) cfma(acc, gcol[nb * np_], ucol[np_]);
      sT[e] = acc;
    }
    __syncthreads();
    double *dst = g2 + ik * (int64_t)E;
    for (int e = threadIdx.x; e < E; e += ROT_THREADS) {
      const int m = e % nb, rest = e / nb;  // rest = n + nb*nu
      c128 acc = cmake(0.0, 0.0);
      const c128 *trow = sT + rest * nb;
      for (int mp = 0; mp < nb; mp++) cfma(acc, sUkqH[m + nb * mp], trow[mp]);
      dst[e] = acc.x * acc.x + acc.y * acc.y;
    }
    __syncthreads();
  }
}

cudaError_t launch_rotate_g2(const c128 *gt, int64_t stride_gt, const c128 *Uk, const c128 *Ukq, const int32_t *kq_idx,
                             int nb, int nm, int64_t nk, double *g2, cudaStream_t st) {
  if (nk <= 0) return cudaSuccess;
  const size_t smem = sizeof(c128) * (size_t)(2 * nb * nb * nm + 2 * nb * nb);
  if (smem > 227 * 1024) return cudaErrorInvalidConfiguration;  // large-Nb path not built yet
  if (smem > 48 * 1024) {
    cudaError_t e =
        cudaFuncSetAttribute(rotate_g2_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  const int64_t grid = nk < 148 * 64 ? nk : 148 * 64;
  rotate_g2_small_kernel<<<(unsigned)grid, ROT_THREADS, smem, st>>>(gt, stride_gt, Uk, Ukq, kq_idx, nb, nm, nk, g2);
  return cudaGetLastError();
}

}  // namespace epw
