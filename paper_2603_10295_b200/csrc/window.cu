// window.cu -- energy-window pre-screening of (k,q) pairs ("a pre-screening of k and q points is used,
// skipping the calculation of the e-ph matrix elements involving states outside a 0.3 eV energy window"; SURVEY.md 8(f)
// NEXT-3).  A pair is kept iff some band of eps_k and some band of eps_{k+q} lies in the closed window [emin, emax];
// the decision is taken on the library's own FP64 eigenvalues, right after the eigensolves, and the rotation kernels
// skip every pair whose mask byte is 0 (its |g|^2 block is reported as zeros).
#include "common.cuh"

namespace epw {

__global__ void __launch_bounds__(256)
    window_mask_kernel(const double *__restrict__ eps_k, const double *__restrict__ eps_kq,
                       const double *__restrict__ eps_k_all, const int32_t *__restrict__ kq_idx, int nb, int64_t nk,
                       double emin, double emax, uint8_t *__restrict__ mask) {
  for (int64_t ik = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; ik < nk; ik += (int64_t)gridDim.x * blockDim.x) {
    const double *e1 = eps_k + ik * nb;
    const double *e2 = kq_idx ? eps_k_all + (int64_t)kq_idx[ik] * nb : eps_kq + ik * nb;
    bool in_k = false, in_kq = false;
    for (int b = 0; b < nb; b++) {
      in_k |= e1[b] >= emin && e1[b] <= emax;
      in_kq |= e2[b] >= emin && e2[b] <= emax;
    }
    mask[ik] = (uint8_t)(in_k && in_kq);
  }
}

cudaError_t launch_window_mask(const double *eps_k, const double *eps_kq, const double *eps_k_all, const int32_t *kq_idx,
                               int nb, int64_t nk, double emin, double emax, uint8_t *mask, cudaStream_t st) {
  if (nk <= 0) return cudaSuccess;
  const int64_t blocks = ceil_div(nk, 256);
  window_mask_kernel<<<grid_cap(blocks, 8), 256, 0, st>>>(eps_k, eps_kq, eps_k_all, kq_idx, nb, nk,
                                                                                   emin, emax, mask);
  return cudaGetLastError();
}

__global__ void __launch_bounds__(256)
    zero_masked_kernel(const uint8_t *__restrict__ mask, int64_t nk, int64_t E, double *__restrict__ g2) {
  for (int64_t ik = blockIdx.x; ik < nk; ik += gridDim.x) {
    if (mask[ik]) continue;
    double *dst = g2 + ik * E;
    for (int64_t i = threadIdx.x; i < E; i += blockDim.x) dst[i] = 0.0;
  }
}

cudaError_t launch_zero_masked(const uint8_t *mask, int64_t nk, int64_t E, double *g2, cudaStream_t st) {
  if (nk <= 0) return cudaSuccess;
  zero_masked_kernel<<<grid_cap(nk, 16), 256, 0, st>>>(mask, nk, E, g2);
  return cudaGetLastError();
}

}  // namespace epw
