// phase.cu -- S0: Fourier phase tables  w(R) exp(2 pi i x.R)  (Eq. 9, L114 Eq. 10; the "x" vector
// of Fig. 13, which the paper builds on the host once per q).
//
// The argument is reduced exactly before the trigonometric evaluation: each product x_d * R_d (R_d a small
// integer) is rounded once, its nearest integer is removed, the three remainders are summed and reduced again,
// so the angle handed to sincospi() lies in [-1, 1] with an absolute error of a few ulp(1).
#include "common.cuh"

namespace epw {

__device__ __forceinline__ double reduced_turns(double x0, double x1, double x2, int r0, int r1, int r2) {
  double t0 = x0 * (double)r0, t1 = x1 * (double)r1, t2 = x2 * (double)r2;
  t0 -= rint(t0);
  t1 -= rint(t1);
  t2 -= rint(t2);
  double t = t0 + t1 + t2;
  t -= rint(t);
  return t;  // in [-0.5, 0.5]
}

__device__ __forceinline__ c128 phase_factor(double x0, double x1, double x2, int r0, int r1, int r2, double w) {
  double s, c;
  sincospi(2.0 * reduced_turns(x0, x1, x2, r0, r1, r2), &s, &c);
  return cmake(w * c, w * s);
}

// P[ix][ir], row-major.  One thread per element; R and w are tiny and L1/L2 resident.
__global__ void __launch_bounds__(256) phase_table_kernel(const double *__restrict__ x, int64_t nx,
                                                          const int32_t *__restrict__ R,
                                                          const double *__restrict__ w, int nr,
                                                          c128 *__restrict__ P) {
  const int64_t total = nx * nr;
  for (int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; idx < total;
       idx += (int64_t)gridDim.x * blockDim.x) {
    const int64_t ix = idx / nr;
    const int ir = (int)(idx - ix * nr);
    P[idx] = phase_factor(x[3 * ix], x[3 * ix + 1], x[3 * ix + 2], R[3 * ir], R[3 * ir + 1], R[3 * ir + 2], w[ir]);
  }
}

// The same table written as the packed A' operand of the DMMA contraction: one CTA per (m-tile, k-block) chunk
// of 128 k-points x 8 lattice vectors; the chunk is assembled in shared memory in fragment order and written
// out as 16 KB of fully coalesced stores.  Rows >= nx and lattice vectors >= nr are zero padding.
__global__ void __launch_bounds__(256) phase_pack_a_kernel(const double *__restrict__ x, int64_t nx,
                                                           const int32_t *__restrict__ R,
                                                           const double *__restrict__ w, int nr, int KB,
                                                           double *__restrict__ Apack) {
  __shared__ double chunk[GEMM_CHUNK];
  const int64_t mt = blockIdx.x / KB;
  const int kb = (int)(blockIdx.x - mt * KB);
  for (int e = threadIdx.x; e < GEMM_BM * (GEMM_BK / 2); e += blockDim.x) {
    const int mr = e & (GEMM_BM - 1);
    const int rc = e >> 7;  // 0..7: lattice vector inside the k-block
    const int64_t ix = mt * GEMM_BM + mr;
    const int ir = kb * (GEMM_BK / 2) + rc;
    c128 p = cmake(0.0, 0.0);
    if (ix < nx && ir < nr)
      p = phase_factor(x[3 * ix], x[3 * ix + 1], x[3 * ix + 2], R[3 * ir], R[3 * ir + 1], R[3 * ir + 2], w[ir]);
    chunk[apack_offset(mr, 2 * rc)] = p.x;
    chunk[apack_offset(mr, 2 * rc + 1)] = p.y;
  }
  __syncthreads();
  double2 *dst = reinterpret_cast<double2 *>(Apack + (int64_t)blockIdx.x * GEMM_CHUNK);
  const double2 *src = reinterpret_cast<const double2 *>(chunk);
  for (int e = threadIdx.x; e < GEMM_CHUNK / 2; e += blockDim.x) dst[e] = src[e];
}

cudaError_t launch_phase_table(const double *x, int64_t nx, const int32_t *R, const double *w, int nr, c128 *P,
                               cudaStream_t st) {
  if (nx <= 0 || nr <= 0) return cudaSuccess;
  const int64_t total = nx * nr;
  const int grid = grid_cap(ceil_div(total, 256), 16);
  phase_table_kernel<<<grid, 256, 0, st>>>(x, nx, R, w, nr, P);
  return cudaGetLastError();
}

cudaError_t launch_phase_pack_a(const double *x, int64_t nx, const int32_t *R, const double *w, int nr, double *Apack,
                                cudaStream_t st) {
  if (nx <= 0 || nr <= 0) return cudaSuccess;
  const int KB = (int)ceil_div(2 * (int64_t)nr, GEMM_BK);
  const int64_t MT = ceil_div(nx, GEMM_BM);
  phase_pack_a_kernel<<<(unsigned)(MT * KB), 256, 0, st>>>(x, nx, R, w, nr, KB, Apack);
  return cudaGetLastError();
}

}  // namespace epw
