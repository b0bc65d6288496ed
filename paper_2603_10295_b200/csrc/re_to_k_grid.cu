// re_to_k_grid.cu -- S2 (and the H(k), H(k+q) part of S3a) when the k-points form a UNIFORM GRID
//     k = ((i1 + s1)/N1, (i2 + s2)/N2, (i3 + s3)/N3),   i3 fastest                       (epw_interp_interpolate_grid).
// The phase of the Re -> k Fourier sum (Eq. 10, "FT w.r.t. Re") then factorises,
//     e^{2 pi i k.Re} = e^{2 pi i (i1+s1) n1/N1} e^{2 pi i (i2+s2) n2/N2} e^{2 pi i (i3+s3) n3/N3},     Re = (n1,n2,n3),
// so the sum over the Ne lattice vectors can be taken one crystal axis at a time (the row-column scheme of a
// multi-dimensional DFT, here with L_d << N_d inputs per axis):
//     T1[n1][n2][i3][c] = sum_n3 X [n1][n2][n3][c] e^{2 pi i (i3+s3) n3/N3}        L1 L2 N3 L3       multiplies per column
//     T2[n1][i2][i3][c] = sum_n2 T1[n1][n2][i3][c] e^{2 pi i (i2+s2) n2/N2}        L1 N2 N3 L2
//     C [i1][i2][i3][c] = sum_n1 T2[n1][i2][i3][c] e^{2 pi i (i1+s1) n1/N1}        N1 N2 N3 L1
// instead of Nk Ne per column for the dense contraction: 40x fewer multiplications for BASELINE.json configs[1]
// (7^3 vectors, 40^3 grid).  X is the B operand of the dense path, B_q[Re][c] = w_e(Re) [ g^(Re,q) | e^{2 pi i q.Re} H(Re) ],
// scattered into the bounding box [L1][L2][L3] of the Re list (zeros where the list has no vector); the result C is
// the same [k][c] array the dense kernel writes, so the eigensolver and the rotation that follow are unchanged.
// Each pass is one launch of the streaming kernel at the end of this file (or, for box extents above 32, of the in-place
// FP64 tensor-path contraction of zgemm_strided.cu); a pass is bound by writing its output to HBM, not by arithmetic.
// The result equals the plain definition up to rounding order (sums re-associated axis by axis).
#include "common.cuh"

namespace epw {

// X[box_idx[ie]][c] for c < ncols_g:  w_e sum_ka g1[ka][ie][x] e[ka][nu] / sqrt(2 omega_nu)   (S4a hoisted; c = nu*nbb + x)
//                   for c >= ncols_g: w_e phase_qe[ie] H_R[ie][x]                               (H(k+q) columns)
// e == NULL: no mode rotation (identity, amplitude 1).  g1 == NULL: only the H columns exist (ncols_g = 0).
__global__ void __launch_bounds__(256)
    box_scatter_kernel(const c128 *__restrict__ g1, const c128 *__restrict__ e, const double *__restrict__ omega,
                       double omega_min, const c128 *__restrict__ H_R, const c128 *__restrict__ phase_qe,
                       const double *__restrict__ w_e, const int32_t *__restrict__ box_idx, int nbb, int nm, int ne,
                       int ncols_g, int ncols_h, c128 *__restrict__ X) {
  const int ncols = ncols_g + ncols_h;
  const int64_t total = (int64_t)ne * ncols;
  for (int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; idx < total;
       idx += (int64_t)gridDim.x * blockDim.x) {
    const int r = (int)(idx / ncols);
    const int c = (int)(idx - (int64_t)r * ncols);
    c128 v = cmake(0.0, 0.0);
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
    } else {
      const c128 hh = H_R[(int64_t)r * nbb + (c - ncols_g)];
      v = phase_qe ? cmul(phase_qe[r], hh) : hh;
    }
    const double w = w_e[r];
    X[(int64_t)box_idx[r] * ncols + c] = cmake(w * v.x, w * v.y);
  }
}

cudaError_t launch_box_scatter(const c128 *g1, const c128 *e, const double *omega, double omega_min, const c128 *H_R,
                               const c128 *phase_qe, const double *w_e, const int32_t *box_idx, int64_t box_size, int nbb,
                               int nm, int ne, int ncols_g, int ncols_h, c128 *X, cudaStream_t st) {
  const int ncols = ncols_g + ncols_h;
  if (ncols <= 0 || ne <= 0) return cudaSuccess;
  if (box_size != ne) {  // lattice vectors missing from the bounding box contribute zero
    cudaError_t e0 = cudaMemsetAsync(X, 0, sizeof(c128) * (size_t)box_size * ncols, st);
    if (e0 != cudaSuccess) return e0;
  }
  const int64_t blocks = ceil_div((int64_t)ne * ncols, 256);
  box_scatter_kernel<<<grid_cap(blocks, 16), 256, 0, st>>>(
      g1, e, omega, omega_min, H_R, phase_qe, w_e, box_idx, nbb, nm, ne, ncols_g, ncols_h, X);
  return cudaGetLastError();
}

// One axis of the factorised phase: P[n][i] = exp(2 pi i frac((lo + n) x_i)), x_i = (i0 + i + shift)/N, n < L, i < cnt.
// Same exact argument reduction as phase.cu (the product of x with the small integer is rounded once, its nearest
// integer removed); x_i is formed exactly as a caller would form the k-list entry, (i + shift)/N in FP64.
__global__ void __launch_bounds__(256) grid_axis_phase_kernel(int N, int i0, int cnt, double shift, int lo, int L,
                                                              c128 *__restrict__ P) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= L * cnt) return;
  const int n = idx / cnt, i = idx - n * cnt;
  const double x = ((double)(i0 + i) + shift) / (double)N;
  double t = x * (double)(lo + n);
  t -= rint(t);
  double s, c;
  sincospi(2.0 * t, &s, &c);
  P[idx] = cmake(c, s);
}

cudaError_t launch_grid_axis_phase(int N, int i0, int cnt, double shift, int lo, int L, c128 *P, cudaStream_t st) {
  if (L <= 0 || cnt <= 0) return cudaSuccess;
  grid_axis_phase_kernel<<<(unsigned)ceil_div((int64_t)L * cnt, 256), 256, 0, st>>>(N, i0, cnt, shift, lo, L, P);
  return cudaGetLastError();
}

// k_list[(i1*N2 + i2)*N3 + i3] = ((i1+s1)/N1, (i2+s2)/N2, (i3+s3)/N3): the list the grid entry point stands for
// (used when a kernel family has no factorised form, e.g. the large-Nb path whose grids are one-dimensional).
__global__ void __launch_bounds__(256) grid_klist_kernel(int N1, int N2, int N3, double s1, double s2, double s3,
                                                         double *__restrict__ k_list) {
  const int64_t nk = (int64_t)N1 * N2 * N3;
  for (int64_t ik = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; ik < nk; ik += (int64_t)gridDim.x * blockDim.x) {
    const int i3 = (int)(ik % N3);
    const int64_t t = ik / N3;
    const int i2 = (int)(t % N2), i1 = (int)(t / N2);
    k_list[3 * ik] = ((double)i1 + s1) / (double)N1;
    k_list[3 * ik + 1] = ((double)i2 + s2) / (double)N2;
    k_list[3 * ik + 2] = ((double)i3 + s3) / (double)N3;
  }
}

cudaError_t launch_grid_klist(const int32_t N[3], const double s[3], double *k_list, cudaStream_t st) {
  const int64_t nk = (int64_t)N[0] * N[1] * N[2];
  const int64_t blocks = ceil_div(nk, 256);
  grid_klist_kernel<<<grid_cap(blocks, 8), 256, 0, st>>>(N[0], N[1], N[2], s[0], s[1], s[2],
                                                                                    k_list);
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------------
// One axis pass as a streaming kernel:  C[blk][col][off] = sum_{r < K} A[blk][r][off] * P[r][col]
//   A element (row, r) at  A + (row / a_rb) * a_bs + (row % a_rb) + r * a_ks      (rows contiguous for fixed r)
//   C element (row, col) at C + (row / c_rb) * c_bs + (row % c_rb) + col * c_cs
// K = L_d is 7..13 here: the pass reads each input once, writes N_d outputs per input and does 4 K DFMA per output --
// it is bound by the write stream, and a tensor-core tile pipeline (load -> DMMA -> epilogue per tile, one CTA per SM)
// only adds latency (43 us against a 14 us memory time for the axis-2 pass of configs[1]).  Here a thread keeps the K
// inputs of its row in registers (R rows per thread is a template parameter; one row measured best: more threads in
// flight beat fewer phase loads per FMA), takes the phases by broadcast from shared memory and streams the columns out
// with fully coalesced 16-byte stores; blockIdx.y splits the columns so that small passes still fill the GPU.
// ---------------------------------------------------------------------------------------------------------------
template <int KMAX, int R>
__global__ void __launch_bounds__(256)
    axis_pass_kernel(const c128 *__restrict__ A, int64_t a_rb, int64_t a_bs, int64_t a_ks, int64_t M,
                     const c128 *__restrict__ P, int64_t p_rs, int64_t p_cs, int K, int N, int cols_per_y,
                     c128 *__restrict__ C, int64_t c_rb, int64_t c_bs, int64_t c_cs) {
  extern __shared__ double2 sPh[];  // [K][ncol] of this column group
  const int col0 = blockIdx.y * cols_per_y;
  const int ncol = N - col0 < cols_per_y ? N - col0 : cols_per_y;
  for (int e = threadIdx.x; e < K * ncol; e += blockDim.x) {
    const int r = e / ncol, c = e - r * ncol;
    sPh[e] = P[(int64_t)r * p_rs + (int64_t)(col0 + c) * p_cs];
  }
  __syncthreads();
  const int64_t row0 = R * (blockIdx.x * (int64_t)blockDim.x + threadIdx.x);
  if (row0 >= M) return;
  c128 x[R][KMAX];
  c128 *dst[R];
  bool have[R];
#pragma unroll
  for (int i = 0; i < R; i++) {
    have[i] = row0 + i < M;
    const int64_t row = have[i] ? row0 + i : row0;
    const int64_t b = row / a_rb;
    const c128 *src = A + b * a_bs + (row - b * a_rb);
#pragma unroll
    for (int r = 0; r < KMAX; r++) x[i][r] = r < K ? src[(int64_t)r * a_ks] : cmake(0.0, 0.0);
    const int64_t d = row / c_rb;
    dst[i] = C + d * c_bs + (row - d * c_rb) + (int64_t)col0 * c_cs;
  }
  for (int c = 0; c < ncol; c++) {
    c128 y[R];
#pragma unroll
    for (int i = 0; i < R; i++) y[i] = cmake(0.0, 0.0);
#pragma unroll
    for (int r = 0; r < KMAX; r++) {
      if (r < K) {
        const c128 ph = sPh[r * ncol + c];
#pragma unroll
        for (int i = 0; i < R; i++) cfma(y[i], x[i][r], ph);
      }
    }
#pragma unroll
    for (int i = 0; i < R; i++)
      if (have[i]) dst[i][(int64_t)c * c_cs] = y[i];
  }
}

bool axis_pass_supported(int K) { return K >= 1 && K <= 32; }

// P element (r, col) at P + r * p_rs + col * p_cs (c128 elements)
cudaError_t launch_axis_pass_p(const c128 *A, int64_t a_rb, int64_t a_bs, int64_t a_ks, int64_t M, const c128 *P,
                               int64_t p_rs, int64_t p_cs, int K, int N, c128 *C, int64_t c_rb, int64_t c_bs, int64_t c_cs,
                               int num_sms, cudaStream_t st) {
  if (M <= 0 || N <= 0 || K <= 0) return cudaSuccess;
  if (K > 32) return cudaErrorInvalidValue;
  const int R = 1;   // rows per thread (see the kernel comment)
  const int64_t bx = ceil_div(ceil_div(M, R), 256);
  // split the columns while the row blocks alone would not give every SM a few CTAs
  int ny = 1;
  while (bx * ny < 4 * (int64_t)num_sms && ny < N && N / (ny + 1) >= 8) ny++;
  const int cols_per_y = (int)ceil_div(N, ny);
  ny = (int)ceil_div(N, cols_per_y);
  const size_t smem = sizeof(double2) * (size_t)K * cols_per_y;
  dim3 grid((unsigned)bx, (unsigned)ny);
#define EPW_AXIS_LAUNCH(KM, RR)                                                                                       \
  do {                                                                                                               \
    if (smem > 48 * 1024) {                                                                                          \
      cudaError_t e =                                                                                                \
          cudaFuncSetAttribute(axis_pass_kernel<KM, RR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);    \
      if (e != cudaSuccess) return e;                                                                                \
    }                                                                                                                \
    axis_pass_kernel<KM, RR><<<grid, 256, smem, st>>>(A, a_rb, a_bs, a_ks, M, P, p_rs, p_cs, K, N, cols_per_y, C, c_rb, \
                                                      c_bs, c_cs);                                                   \
  } while (0)
  if (K <= 8) EPW_AXIS_LAUNCH(8, 1);
  else if (K <= 16) EPW_AXIS_LAUNCH(16, 1);
  else EPW_AXIS_LAUNCH(32, 1);
#undef EPW_AXIS_LAUNCH
  return cudaGetLastError();
}

cudaError_t launch_axis_pass(const c128 *A, int64_t a_rb, int64_t a_bs, int64_t a_ks, int64_t M, const c128 *P, int K, int N,
                             c128 *C, int64_t c_rb, int64_t c_bs, int64_t c_cs, int num_sms, cudaStream_t st) {
  return launch_axis_pass_p(A, a_rb, a_bs, a_ks, M, P, N, 1, K, N, C, c_rb, c_bs, c_cs, num_sms, st);
}

}  // namespace epw
