// eigh_jacobi.cu -- S3b: batched complex-Hermitian eigensolver, A = V diag(lambda) V^dagger, lambda ascending
// (BASELINE.json north_star stage 3: "batched small Hermitian eigensolve (one warp or CTA per matrix, Jacobi in
// shared memory)"; PAPER.md:L72 U_k, L54 u(q) are the paper's only mention of these quantities).
//
// Parallel-order (round-robin tournament) Jacobi: a sweep is N-1 rounds of N/2 disjoint rotations (N = n rounded
// up to even), all N/2 rotations of a round are applied together:
//   phase 1  one lane per pair (p,q): a_pq = r e^{i phi}, tau = (a_qq-a_pp)/(2r), t = sgn(tau)/(|tau|+sqrt(1+tau^2)),
//            c = 1/sqrt(1+t^2), s = t c,  J = [[c, s e^{i phi}], [-s e^{-i phi}, c]]   (rows/cols p,q)
//   phase 2  A <- A J and V <- V J     (column pairs; one task per (row, pair))
//   phase 3  A <- J^dagger A           (row pairs;    one task per (column, pair)); a_pq := 0, diagonal real
// n <= 32: one warp per matrix, A and V in shared memory (leading dimension padded to an odd number of 16-byte
// words so both the column and the row pass are bank-conflict free), __syncwarp between phases.
// n  > 32: one CTA per matrix, A and V in an L2-resident global scratch (a 288 x 288 complex matrix is 1.3 MB and
// cannot live in the 227 KB of shared memory), __syncthreads between phases.
// Convergence: off-diagonal Frobenius norm^2 <= 1e-30 * ||A||_F^2, checked once per sweep, at most MAX_SWEEPS.
// These run on the plain FP64 pipe (DFMA/DMUL, DADD, MUFU.RSQ64H-seeded sqrt/div), not on the tensor path.
#include "common.cuh"

namespace epw {

constexpr int EIGH_MAX_SWEEPS = 40;
constexpr int EIGH_SMALL_MAX_N = 32;
constexpr int EIGH_WARPS_PER_CTA = 4;

// pair (p<q) handled by slot s in round r of the round-robin schedule over N (even) players
__device__ __forceinline__ void rr_pair(int N, int r, int s, int &p, int &q) {
  int a, b;
  if (s == 0) {
    a = N - 1;
    b = r;
  } else {
    a = r + s;
    if (a >= N - 1) a -= N - 1;
    b = r - s;
    if (b < 0) b += N - 1;
  }
  p = a < b ? a : b;
  q = a < b ? b : a;
}

struct Rot {
  double c, sr, si, pad;  // J_pq = sr + i si = s e^{i phi}
};

__device__ __forceinline__ Rot make_rot(double app, double aqq, c128 apq) {
  Rot R;
  const double r2 = apq.x * apq.x + apq.y * apq.y;
  if (r2 == 0.0) {
    R.c = 1.0; R.sr = 0.0; R.si = 0.0; R.pad = 0.0;
    return R;
  }
  const double r = sqrt(r2);
  const double tau = (aqq - app) / (2.0 * r);
  const double t = copysign(1.0, tau) / (fabs(tau) + sqrt(1.0 + tau * tau));
  const double c = rsqrt(1.0 + t * t);
  const double s_over_r = t * c / r;
  R.c = c;
  R.sr = s_over_r * apq.x;
  R.si = s_over_r * apq.y;
  R.pad = 0.0;
  return R;
}

// (x_p, x_q) <- (x_p, x_q) J  for a row vector pair:  x_p' = c x_p - conj(S) x_q ;  x_q' = S x_p + c x_q
__device__ __forceinline__ void apply_cols(c128 &xp, c128 &xq, const Rot &R) {
  const c128 a = xp, b = xq;
  xp.x = R.c * a.x - (R.sr * b.x + R.si * b.y);
  xp.y = R.c * a.y - (R.sr * b.y - R.si * b.x);
  xq.x = R.c * b.x + (R.sr * a.x - R.si * a.y);
  xq.y = R.c * b.y + (R.sr * a.y + R.si * a.x);
}
// (y_p; y_q) <- J^dagger (y_p; y_q) for a column vector pair:  y_p' = c y_p - S y_q ;  y_q' = conj(S) y_p + c y_q
__device__ __forceinline__ void apply_rows(c128 &yp, c128 &yq, const Rot &R) {
  const c128 a = yp, b = yq;
  yp.x = R.c * a.x - (R.sr * b.x - R.si * b.y);
  yp.y = R.c * a.y - (R.sr * b.y + R.si * b.x);
  yq.x = R.c * b.x + (R.sr * a.x + R.si * a.y);
  yq.y = R.c * b.y + (R.sr * a.y - R.si * a.x);
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ------------------------------------------------------------------------------------------------------
// n <= 32: warp per matrix, shared memory.
// ------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(EIGH_WARPS_PER_CTA * 32)
    eigh_small_kernel(const c128 *__restrict__ Ain, int64_t stride_a, int n, int64_t batch, double *__restrict__ evals,
                      c128 *__restrict__ Vout, int sqrt_mode, int32_t *__restrict__ status) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t b = (int64_t)blockIdx.x * EIGH_WARPS_PER_CTA + warp;
  if (b >= batch) return;
  const int ld = n | 1;
  const int N = n + (n & 1);
  const int half = N >> 1;
  const size_t per_warp = (size_t)(2 * ld * n) * sizeof(c128) + (size_t)half * sizeof(Rot) + (size_t)n * sizeof(double);
  unsigned char *base = smem_raw + (size_t)warp * ((per_warp + 15) & ~(size_t)15);
  c128 *A = reinterpret_cast<c128 *>(base);
  c128 *V = A + ld * n;
  Rot *rot = reinterpret_cast<Rot *>(V + ld * n);
  double *lam = reinterpret_cast<double *>(rot + half);

  // load the Hermitian part (A + A^dagger)/2, V = I
  const c128 *src = Ain + b * stride_a;
  double fro2 = 0.0;
  for (int e = lane; e < n * n; e += 32) {
    const int i = e % n, j = e / n;
    const c128 x = src[i + n * j], y = src[j + n * i];
    const c128 v = cmake(0.5 * (x.x + y.x), i == j ? 0.0 : 0.5 * (x.y - y.y));
    A[i + ld * j] = v;
    V[i + ld * j] = cmake(i == j ? 1.0 : 0.0, 0.0);
    fro2 += cabs2(v);
  }
  fro2 = warp_sum(fro2);
  const double thresh2 = 1e-30 * fro2;
  __syncwarp();

  bool converged = false;
  for (int sweep = 0; sweep <= EIGH_MAX_SWEEPS; sweep++) {
    double off2 = 0.0;
    for (int e = lane; e < n * n; e += 32) {
      const int i = e % n, j = e / n;
      if (i != j) off2 += cabs2(A[i + ld * j]);
    }
    off2 = warp_sum(off2);
    if (off2 <= thresh2) { converged = true; break; }
    if (sweep == EIGH_MAX_SWEEPS) break;
    for (int r = 0; r < N - 1; r++) {
      // phase 1: rotation parameters
      if (lane < half) {
        int p, q;
        rr_pair(N, r, lane, p, q);
        Rot R;
        if (q < n) R = make_rot(A[p + ld * p].x, A[q + ld * q].x, A[p + ld * q]);
        else { R.c = 1.0; R.sr = 0.0; R.si = 0.0; R.pad = 0.0; }
        rot[lane] = R;
      }
      __syncwarp();
      // phase 2: columns of A and V
      for (int e = lane; e < n * half; e += 32) {
        const int i = e % n, s = e / n;
        int p, q;
        rr_pair(N, r, s, p, q);
        if (q >= n) continue;
        const Rot R = rot[s];
        c128 xp = A[i + ld * p], xq = A[i + ld * q];
        apply_cols(xp, xq, R);
        A[i + ld * p] = xp;
        A[i + ld * q] = xq;
        c128 vp = V[i + ld * p], vq = V[i + ld * q];
        apply_cols(vp, vq, R);
        V[i + ld * p] = vp;
        V[i + ld * q] = vq;
      }
      __syncwarp();
      // phase 3: rows of A
      for (int e = lane; e < n * half; e += 32) {
        const int j = e % n, s = e / n;
        int p, q;
        rr_pair(N, r, s, p, q);
        if (q >= n) continue;
        const Rot R = rot[s];
        c128 yp = A[p + ld * j], yq = A[q + ld * j];
        apply_rows(yp, yq, R);
        A[p + ld * j] = yp;
        A[q + ld * j] = yq;
      }
      __syncwarp();
      if (lane < half) {
        int p, q;
        rr_pair(N, r, lane, p, q);
        if (q < n && (rot[lane].sr != 0.0 || rot[lane].si != 0.0)) {
          A[p + ld * q] = cmake(0.0, 0.0);
          A[q + ld * p] = cmake(0.0, 0.0);
          A[p + ld * p].y = 0.0;
          A[q + ld * q].y = 0.0;
        }
      }
      __syncwarp();
    }
  }
  if (!converged && status != nullptr && lane == 0) atomicExch(status, 1);

  // ascending order by rank counting (ties broken by index), write eigenvalues and permuted eigenvectors
  for (int j = lane; j < n; j += 32) lam[j] = A[j + ld * j].x;
  __syncwarp();
  for (int j = lane; j < n; j += 32) {
    const double lj = lam[j];
    int rank = 0;
    for (int i = 0; i < n; i++) rank += (lam[i] < lj) || (lam[i] == lj && i < j);
    double out = lj;
    if (sqrt_mode) out = lj > 0.0 ? sqrt(lj) : -sqrt(-lj);
    evals[b * n + rank] = out;
    A[j + ld * j].y = (double)rank;  // stash the destination column
  }
  __syncwarp();
  c128 *dst = Vout + b * (int64_t)n * n;
  for (int e = lane; e < n * n; e += 32) {
    const int i = e % n, j = e / n;
    const int rank = (int)A[j + ld * j].y;
    dst[i + n * rank] = V[i + ld * j];
  }
}

// ------------------------------------------------------------------------------------------------------
// n > 32: CTA per matrix, working copies of A and V in global scratch (L2 resident).
// ------------------------------------------------------------------------------------------------------
constexpr int EIGH_LARGE_THREADS = 512;

__device__ __forceinline__ double block_sum(double v, double *red) {
  v = warp_sum(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  double tot = 0.0;
  for (int w = 0; w < EIGH_LARGE_THREADS / 32; w++) tot += red[w];
  return tot;
}

__global__ void __launch_bounds__(EIGH_LARGE_THREADS)
    eigh_large_kernel(const c128 *__restrict__ Ain, int64_t stride_a, int n, int64_t batch, double *__restrict__ evals,
                      c128 *__restrict__ Vout, int sqrt_mode, int32_t *__restrict__ status,
                      c128 *__restrict__ scratch) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int N = n + (n & 1);
  const int half = N >> 1;
  Rot *rot = reinterpret_cast<Rot *>(smem_raw);
  double *lam = reinterpret_cast<double *>(rot + half);
  int *rank_of = reinterpret_cast<int *>(lam + n);
  __shared__ double red[EIGH_LARGE_THREADS / 32];
  const int tid = threadIdx.x;
  for (int64_t b = blockIdx.x; b < batch; b += gridDim.x) {
    c128 *A = scratch + (int64_t)blockIdx.x * 2 * n * n;
    c128 *V = A + (int64_t)n * n;
    const c128 *src = Ain + b * stride_a;
    double fro2 = 0.0;
    for (int e = tid; e < n * n; e += EIGH_LARGE_THREADS) {
      const int i = e % n, j = e / n;
      const c128 x = src[i + (int64_t)n * j], y = src[j + (int64_t)n * i];
      const c128 v = cmake(0.5 * (x.x + y.x), i == j ? 0.0 : 0.5 * (x.y - y.y));
      A[e] = v;
      V[e] = cmake(i == j ? 1.0 : 0.0, 0.0);
      fro2 += cabs2(v);
    }
    fro2 = block_sum(fro2, red);
    const double thresh2 = 1e-30 * fro2;
    bool converged = false;
    for (int sweep = 0; sweep <= EIGH_MAX_SWEEPS; sweep++) {
      double off2 = 0.0;
      for (int e = tid; e < n * n; e += EIGH_LARGE_THREADS) {
        const int i = e % n, j = e / n;
        if (i != j) off2 += cabs2(A[e]);
      }
      off2 = block_sum(off2, red);
      if (off2 <= thresh2) { converged = true; break; }
      if (sweep == EIGH_MAX_SWEEPS) break;
      for (int r = 0; r < N - 1; r++) {
        for (int s = tid; s < half; s += EIGH_LARGE_THREADS) {
          int p, q;
          rr_pair(N, r, s, p, q);
          Rot R;
          if (q < n) R = make_rot(A[p + (int64_t)n * p].x, A[q + (int64_t)n * q].x, A[p + (int64_t)n * q]);
          else { R.c = 1.0; R.sr = 0.0; R.si = 0.0; R.pad = 0.0; }
          rot[s] = R;
        }
        __syncthreads();
        for (int e = tid; e < n * half; e += EIGH_LARGE_THREADS) {
          const int i = e % n, s = e / n;
          int p, q;
          rr_pair(N, r, s, p, q);
          if (q >= n) continue;
          const Rot R = rot[s];
          c128 xp = A[i + (int64_t)n * p], xq = A[i + (int64_t)n * q];
          apply_cols(xp, xq, R);
          A[i + (int64_t)n * p] = xp;
          A[i + (int64_t)n * q] = xq;
          c128 vp = V[i + (int64_t)n * p], vq = V[i + (int64_t)n * q];
          apply_cols(vp, vq, R);
          V[i + (int64_t)n * p] = vp;
          V[i + (int64_t)n * q] = vq;
        }
        __syncthreads();
        for (int e = tid; e < n * half; e += EIGH_LARGE_THREADS) {
          const int j = e % n, s = e / n;
          int p, q;
          rr_pair(N, r, s, p, q);
          if (q >= n) continue;
          const Rot R = rot[s];
          c128 yp = A[p + (int64_t)n * j], yq = A[q + (int64_t)n * j];
          apply_rows(yp, yq, R);
          A[p + (int64_t)n * j] = yp;
          A[q + (int64_t)n * j] = yq;
        }
        __syncthreads();
        for (int s = tid; s < half; s += EIGH_LARGE_THREADS) {
          int p, q;
          rr_pair(N, r, s, p, q);
          if (q < n && (rot[s].sr != 0.0 || rot[s].si != 0.0)) {
            A[p + (int64_t)n * q] = cmake(0.0, 0.0);
            A[q + (int64_t)n * p] = cmake(0.0, 0.0);
            A[p + (int64_t)n * p].y = 0.0;
            A[q + (int64_t)n * q].y = 0.0;
          }
        }
        __syncthreads();
      }
    }
    if (!converged && status != nullptr && tid == 0) atomicExch(status, 1);
    for (int j = tid; j < n; j += EIGH_LARGE_THREADS) lam[j] = A[j + (int64_t)n * j].x;
    __syncthreads();
    for (int j = tid; j < n; j += EIGH_LARGE_THREADS) {
      const double lj = lam[j];
      int rank = 0;
      for (int i = 0; i < n; i++) rank += (lam[i] < lj) || (lam[i] == lj && i < j);
      double out = lj;
      if (sqrt_mode) out = lj > 0.0 ? sqrt(lj) : -sqrt(-lj);
      evals[b * n + rank] = out;
      rank_of[j] = rank;
    }
    __syncthreads();
    c128 *dst = Vout + b * (int64_t)n * n;
    for (int e = tid; e < n * n; e += EIGH_LARGE_THREADS) {
      const int i = e % n, j = e / n;
      dst[i + (int64_t)n * rank_of[j]] = V[e];
    }
    __syncthreads();
  }
}

static int eigh_large_grid(int64_t batch) { return (int)(batch < 148 ? batch : 148); }

size_t eigh_large_scratch_bytes(int n, int64_t batch) {
  if (n <= EIGH_SMALL_MAX_N) return 0;
  return (size_t)eigh_large_grid(batch) * 2 * (size_t)n * n * sizeof(c128);
}

cudaError_t launch_eigh_batched(const c128 *A, int64_t stride_a, int n, int64_t batch, double *evals, c128 *V,
                                int sqrt_mode, int32_t *status, c128 *scratch_large, cudaStream_t st) {
  if (batch <= 0) return cudaSuccess;
  if (n <= EIGH_SMALL_MAX_N) {
    const int ld = n | 1, half = (n + (n & 1)) >> 1;
    size_t per_warp = (size_t)(2 * ld * n) * sizeof(c128) + (size_t)half * sizeof(Rot) + (size_t)n * sizeof(double);
    per_warp = (per_warp + 15) & ~(size_t)15;
    const size_t smem = per_warp * EIGH_WARPS_PER_CTA;
    if (smem > 48 * 1024) {
      cudaError_t e = cudaFuncSetAttribute(eigh_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      if (e != cudaSuccess) return e;
    }
    eigh_small_kernel<<<(unsigned)ceil_div(batch, EIGH_WARPS_PER_CTA), EIGH_WARPS_PER_CTA * 32, smem, st>>>(
        A, stride_a, n, batch, evals, V, sqrt_mode, status);
  } else {
    if (scratch_large == nullptr) return cudaErrorInvalidValue;
    const int half = (n + (n & 1)) >> 1;
    const size_t smem = (size_t)half * sizeof(Rot) + (size_t)n * sizeof(double) + (size_t)n * sizeof(int);
    eigh_large_kernel<<<eigh_large_grid(batch), EIGH_LARGE_THREADS, smem, st>>>(A, stride_a, n, batch, evals, V,
                                                                                sqrt_mode, status, scratch_large);
  }
  return cudaGetLastError();
}

}  // namespace epw
