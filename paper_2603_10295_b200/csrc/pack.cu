// pack.cu -- operator interpolation (S3a) and the builders of the packed B' operand of the DMMA contraction,
// including the hoisted mode rotation S4a.
//
// S4a hoist: g_{..nu} = sum_ka g_{..ka} e_{q,ka,nu}/sqrt(2 omega_q,nu) (u_{ka,nu}(q); amplitude:
// BASELINE.json north_star stage 4) is linear and depends on q only, so it commutes with the Re -> k Fourier sum.
// Applying it to g(Re,q) costs Nb^2 Nm^2 Ne per q instead of the paper's Nb^2 Nm^2 per (k,q) pair
// (PAPER.md:L102, L118-122), a factor Nk/Ne fewer multiplications ("What differs from the paper").
#include "common.cuh"

namespace epw {

// S3a:  out[ix][e] = sum_ir P[ix][ir] OpR[ir][e],  e over the n*n entries (column-major layout is preserved).
__global__ void __launch_bounds__(256) interp_operator_kernel(const c128 *__restrict__ OpR, int nn, int nr,
                                                              const c128 *__restrict__ P, int64_t nx,
                                                              c128 *__restrict__ out) {
  const int64_t total = nx * nn;
  for (int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; idx < total;
       idx += (int64_t)gridDim.x * blockDim.x) {
    const int64_t ix = idx / nn;
    const int e = (int)(idx - ix * nn);
    c128 acc = cmake(0.0, 0.0);
    const c128 *p = P + ix * nr;
    for (int ir = 0; ir < nr; ir++) cfma(acc, p[ir], OpR[(int64_t)ir * nn + e]);
    out[idx] = acc;
  }
}

cudaError_t launch_interp_operator(const c128 *OpR, int n, int nr, const c128 *P, int64_t nx, c128 *out,
                                   cudaStream_t st) {
  if (nx <= 0) return cudaSuccess;
  const int64_t total = nx * n * n;
  const int64_t blocks = ceil_div(total, 256);
  interp_operator_kernel<<<grid_cap(blocks, 32), 256, 0, st>>>(OpR, n * n, nr, P, nx, out);
  return cudaGetLastError();
}

// Write one complex B element (row r, column c inside the chunk) as its 2x2 real block.
__device__ __forceinline__ void put_b(double *chunk, int rc, int cc, c128 v) {
  chunk[bpack_offset(2 * rc, 2 * cc)] = v.x;
  chunk[bpack_offset(2 * rc, 2 * cc + 1)] = v.y;
  chunk[bpack_offset(2 * rc + 1, 2 * cc)] = -v.y;
  chunk[bpack_offset(2 * rc + 1, 2 * cc + 1)] = v.x;
}

// One CTA per (n-tile, k-block) chunk: 8 lattice vectors x 64 complex columns.
__global__ void __launch_bounds__(256) pack_b_kernel(const c128 *__restrict__ g1, const c128 *__restrict__ e,
                                                     const double *__restrict__ omega, double omega_min,
                                                     const c128 *__restrict__ H_R, const c128 *__restrict__ phase_qe,
                                                     int nbb, int nm, int ne, int ncols_g, int ncols_h, int KB,
                                                     double *__restrict__ Bpack) {
  __shared__ double chunk[GEMM_CHUNK];
  const int nt = blockIdx.x / KB;
  const int kb = blockIdx.x - nt * KB;
  for (int el = threadIdx.x; el < 8 * 64; el += blockDim.x) {
    const int cc = el & 63, rc = el >> 6;
    const int c = nt * 64 + cc;
    const int r = kb * 8 + rc;
    c128 v = cmake(0.0, 0.0);
    if (r < ne) {
      if (c < ncols_g) {
        const int nu = c / nbb, x = c - nu * nbb;
        if (e != nullptr) {
          const double om = omega[nu];
          if (om > omega_min) {
            for (int ka = 0; ka < nm; ka++) cfma(v, g1[((int64_t)ka * ne + r) * nbb + x], e[ka + nm * nu]);
            const double amp = 1.0 / sqrt(2.0 * om);
            v.x *= amp;
            v.y *= amp;
          }
        } else {
          v = g1[((int64_t)nu * ne + r) * nbb + x];
        }
      } else if (c < ncols_g + ncols_h) {
        const int x = c - ncols_g;
        const c128 h = H_R[(int64_t)r * nbb + x];
        v = phase_qe ? cmul(phase_qe[r], h) : h;
      }
    }
    put_b(chunk, rc, cc, v);
  }
  __syncthreads();
  double2 *dst = reinterpret_cast<double2 *>(Bpack + (int64_t)blockIdx.x * GEMM_CHUNK);
  const double2 *src = reinterpret_cast<const double2 *>(chunk);
  for (int i = threadIdx.x; i < GEMM_CHUNK / 2; i += blockDim.x) dst[i] = src[i];
}

cudaError_t launch_pack_b(const c128 *g1, const c128 *e, const double *omega, double omega_min, const c128 *H_R,
                          const c128 *phase_qe, int nbb, int nm, int ne, int ncols_g, int ncols_h, double *Bpack,
                          cudaStream_t st) {
  const int KB = (int)ceil_div(2 * (int64_t)ne, GEMM_BK);
  const int NT = (int)ceil_div(2 * (int64_t)(ncols_g + ncols_h), GEMM_BN);
  pack_b_kernel<<<(unsigned)(NT * KB), 256, 0, st>>>(g1, e, omega, omega_min, H_R, phase_qe, nbb, nm, ne, ncols_g,
                                                     ncols_h, KB, Bpack);
  return cudaGetLastError();
}

// ---- generic packers (row-major complex inputs), used by epw_zgemm -----------------------------------------
__global__ void __launch_bounds__(256) pack_a_generic_kernel(const c128 *__restrict__ A, int64_t M, int K, int KB,
                                                             double *__restrict__ Apack) {
  __shared__ double chunk[GEMM_CHUNK];
  const int64_t mt = blockIdx.x / KB;
  const int kb = (int)(blockIdx.x - mt * KB);
  for (int e = threadIdx.x; e < GEMM_BM * 8; e += blockDim.x) {
    const int rc = e & 7, mr = e >> 3;
    const int64_t m = mt * GEMM_BM + mr;
    const int r = kb * 8 + rc;
    c128 v = cmake(0.0, 0.0);
    if (m < M && r < K) v = A[m * K + r];
    chunk[apack_offset(mr, 2 * rc)] = v.x;
    chunk[apack_offset(mr, 2 * rc + 1)] = v.y;
  }
  __syncthreads();
  double2 *dst = reinterpret_cast<double2 *>(Apack + (int64_t)blockIdx.x * GEMM_CHUNK);
  const double2 *src = reinterpret_cast<const double2 *>(chunk);
  for (int i = threadIdx.x; i < GEMM_CHUNK / 2; i += blockDim.x) dst[i] = src[i];
}

__global__ void __launch_bounds__(256) pack_b_generic_kernel(const c128 *__restrict__ B, int K, int N, int KB,
                                                             double *__restrict__ Bpack) {
  __shared__ double chunk[GEMM_CHUNK];
  const int nt = blockIdx.x / KB;
  const int kb = blockIdx.x - nt * KB;
  for (int el = threadIdx.x; el < 8 * 64; el += blockDim.x) {
    const int cc = el & 63, rc = el >> 6;
    const int c = nt * 64 + cc, r = kb * 8 + rc;
    c128 v = cmake(0.0, 0.0);
    if (r < K && c < N) v = B[(int64_t)r * N + c];
    put_b(chunk, rc, cc, v);
  }
  __syncthreads();
  double2 *dst = reinterpret_cast<double2 *>(Bpack + (int64_t)blockIdx.x * GEMM_CHUNK);
  const double2 *src = reinterpret_cast<const double2 *>(chunk);
  for (int i = threadIdx.x; i < GEMM_CHUNK / 2; i += blockDim.x) dst[i] = src[i];
}

// Strided / batched B' builder of the large-Nb path: complex B[r][n] read at  B + b*batch_stride + r*sr + n*sn,
// optionally conjugated, optionally scaled per column n by the zero-point amplitude 1/sqrt(2 omega[n]) (0 when
// omega[n] <= omega_min: BASELINE.json north_star stage 4; reading G12).  One CTA per 16 KB chunk.
__global__ void __launch_bounds__(256) pack_b_strided_kernel(const c128 *__restrict__ B, int64_t sr, int64_t sn,
                                                             int64_t batch_stride, int conj,
                                                             const double *__restrict__ omega, double omega_min, int K,
                                                             int N, int KB, int NT, double *__restrict__ Bpack) {
  __shared__ double chunk[GEMM_CHUNK];
  const int64_t b = blockIdx.x / (NT * KB);
  const int rem = (int)(blockIdx.x - b * (NT * KB));
  const int nt = rem / KB;
  const int kb = rem - nt * KB;
  const c128 *src = B + b * batch_stride;
  for (int el = threadIdx.x; el < 8 * 64; el += blockDim.x) {
    // r fastest when the operand is r-contiguous (sr == 1), n fastest otherwise: coalesced either way
    const int rc = sr == 1 ? (el & 7) : (el >> 6);
    const int cc = sr == 1 ? (el >> 3) : (el & 63);
    const int c = nt * 64 + cc, r = kb * 8 + rc;
    c128 v = cmake(0.0, 0.0);
    if (r < K && c < N) {
      v = src[(int64_t)r * sr + (int64_t)c * sn];
      if (conj) v.y = -v.y;
      if (omega != nullptr) {
        const double om = omega[c];
        const double amp = om > omega_min ? 1.0 / sqrt(2.0 * om) : 0.0;
        v.x *= amp;
        v.y *= amp;
      }
    }
    put_b(chunk, rc, cc, v);
  }
  __syncthreads();
  double2 *dst = reinterpret_cast<double2 *>(Bpack + (int64_t)blockIdx.x * GEMM_CHUNK);
  const double2 *s2 = reinterpret_cast<const double2 *>(chunk);
  for (int i = threadIdx.x; i < GEMM_CHUNK / 2; i += blockDim.x) dst[i] = s2[i];
}

cudaError_t launch_pack_b_strided(const c128 *B, int64_t sr, int64_t sn, int64_t batch_stride, int64_t batch, int conj,
                                  const double *omega, double omega_min, int K, int N, double *Bpack, cudaStream_t st) {
  if (batch <= 0) return cudaSuccess;
  const int KB = (int)ceil_div(2 * (int64_t)K, GEMM_BK);
  const int NT = (int)ceil_div(2 * (int64_t)N, GEMM_BN);
  pack_b_strided_kernel<<<(unsigned)(batch * NT * KB), 256, 0, st>>>(B, sr, sn, batch_stride, conj, omega, omega_min, K,
                                                                    N, KB, NT, Bpack);
  return cudaGetLastError();
}

cudaError_t launch_pack_a_generic(const c128 *A, int64_t M, int K, double *Apack, cudaStream_t st) {
  const int KB = (int)ceil_div(2 * (int64_t)K, GEMM_BK);
  pack_a_generic_kernel<<<(unsigned)(ceil_div(M, GEMM_BM) * KB), 256, 0, st>>>(A, M, K, KB, Apack);
  return cudaGetLastError();
}
cudaError_t launch_pack_b_generic(const c128 *B, int K, int N, double *Bpack, cudaStream_t st) {
  const int KB = (int)ceil_div(2 * (int64_t)K, GEMM_BK);
  const int NT = (int)ceil_div(2 * (int64_t)N, GEMM_BN);
  pack_b_generic_kernel<<<(unsigned)(NT * KB), 256, 0, st>>>(B, K, N, KB, Bpack);
  return cudaGetLastError();
}

}  // namespace epw
