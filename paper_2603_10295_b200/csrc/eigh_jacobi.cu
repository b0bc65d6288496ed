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
#include <cooperative_groups.h>

#include <algorithm>

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

// ------------------------------------------------------------------------------------------------------
// n > 32, matrix too large for one warp: ONE-SIDED (Hestenes) parallel-order Jacobi on a thread-block CLUSTER.
//
// The two-sided kernel above needs the whole matrix twice per round (column pass and row pass) and the accumulated
// eigenvectors once; at n = 192..288 (configs[4]: H(k) 192 x 192, D(q) 288 x 288; 0.6 / 1.3 MB) that lives in L2 and
// every one of the (n-1) x sweeps rounds pays L2 latency.  Here the matrix is made positive definite by a shift,
// G = A + sigma I with sigma = ||A - mu I||_F - mu, mu = tr(A)/n, and its COLUMNS are orthogonalised by plane rotations from the right:
//   round:  alpha = ||g_p||^2, beta = ||g_q||^2, gamma = g_p^dagger g_q  for the N/2 disjoint pairs of the round
//           J_pq = the rotation that diagonalises [[alpha, gamma], [conj gamma, beta]]   (same formula as make_rot)
//           (g_p, g_q) <- (g_p, g_q) J_pq
// At convergence G = (A + sigma I) V with orthogonal columns, so v_j = g_j / ||g_j||: no eigenvector accumulation and
// no row pass.  Rows of G are distributed over the CTAs of the cluster and stay in SHARED MEMORY for the whole solve
// (n = 288 on 8 CTAs: 36 rows = 166 KB each); the only communication per round is the reduction of the N/2 partial
// (alpha, beta, gamma) triples to the pair's owner CTA and the broadcast of the rotation, both through distributed
// shared memory, with two cluster barriers.  Eigenvalues are the Rayleigh quotients v_j^dagger A v_j with the ORIGINAL
// matrix (||g_j|| - sigma would lose digits to the shift).  Convergence: |gamma| <= sqrt(n) eps sqrt(alpha beta) for
// every pair of a sweep.
// ------------------------------------------------------------------------------------------------------
namespace cg = cooperative_groups;

constexpr int EC_THREADS = 512;
constexpr int EC_MAX_SWEEPS = 40;
constexpr int EC_RQ_COLS = 4;

struct __align__(32) RotB {
  double c, sr, si, act;
};

__global__ void __launch_bounds__(EC_THREADS, 1)
    eigh_cluster_kernel(const c128 *__restrict__ Ain, int64_t stride_a, int n, int64_t batch,
                        double *__restrict__ evals, c128 *__restrict__ Vout, int sqrt_mode, int32_t *__restrict__ status,
                        c128 *__restrict__ scratch, int nr, unsigned long long *__restrict__ work) {
  cg::cluster_group cluster = cg::this_cluster();
  unsigned long long my_rot = 0;   // plane rotations this thread built as the owner of a pair (work counter)
  const int csize = (int)cluster.num_blocks(), crank = (int)cluster.block_rank();
  const int cluster_id = blockIdx.x / csize, num_clusters = gridDim.x / csize;
  extern __shared__ __align__(32) unsigned char smem_raw[];
  __shared__ double red[EC_THREADS / 32];
  const int N = n + (n & 1), half = N >> 1;
  const int hp = (half + csize - 1) / csize;  // pairs owned per CTA
  c128 *G = reinterpret_cast<c128 *>(smem_raw);                      // [n columns][nr local rows]
  double4 *part = reinterpret_cast<double4 *>(smem_raw + ((sizeof(c128) * (size_t)n * nr + 31) & ~(size_t)31));  // [csize sources][hp]
  RotB *rot = reinterpret_cast<RotB *>(part + (size_t)csize * hp);   // [half]
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int r0 = crank * nr;
  const int nloc = n - r0 < nr ? (n - r0 > 0 ? n - r0 : 0) : nr;
  c128 *Vtmp = scratch + (int64_t)cluster_id * 2 * n * n;
  double *lam = reinterpret_cast<double *>(Vtmp + (int64_t)n * n);
  double *nrm2 = lam + n;  // [csize][n]
  const double tol2 = (double)n * 1.2325951644078309e-32;  // (sqrt(n) * 2^-53)^2

  for (int64_t b = cluster_id; b < batch; b += num_clusters) {
    const c128 *src = Ain + b * stride_a;
    // ---- centre the spectrum, mu = tr(A)/n, then sigma = ||A_h - mu I||_F >= rho(A_h - mu I)  (A_h = Hermitian part);
    //      without the centring a nearly scalar matrix (D(q) = big diagonal + small couplings) would get a shift
    //      sqrt(n) times its own size and lose that factor in eigenvector accuracy.  Computed identically by every CTA.
    double tr = 0.0;
    for (int i = tid; i < n; i += EC_THREADS) tr += src[i + (int64_t)n * i].x;
    tr = warp_sum(tr);
    __syncthreads();
    if (lane == 0) red[warp] = tr;
    __syncthreads();
    tr = 0.0;
    for (int w2 = 0; w2 < EC_THREADS / 32; w2++) tr += red[w2];
    const double mu = tr / n;
    double fro2 = 0.0;
    for (int e = tid; e < n * n; e += EC_THREADS) {
      const int i = e % n, j = e / n;
      const c128 x = src[i + (int64_t)n * j], y = src[j + (int64_t)n * i];
      const double re = 0.5 * (x.x + y.x) - (i == j ? mu : 0.0), im = i == j ? 0.0 : 0.5 * (x.y - y.y);
      fro2 += re * re + im * im;
    }
    fro2 = warp_sum(fro2);
    __syncthreads();
    if (lane == 0) red[warp] = fro2;
    __syncthreads();
    fro2 = 0.0;
    for (int w2 = 0; w2 < EC_THREADS / 32; w2++) fro2 += red[w2];
    const double sigma = (fro2 > 0.0 ? sqrt(fro2) : 1.0) - mu;   // G = A_h + sigma I = (A_h - mu I) + ||.||_F I
    // ---- local rows of G ----
    for (int e = tid; e < n * nloc; e += EC_THREADS) {
      const int il = e % nloc, j = e / nloc;
      const int i = r0 + il;
      const c128 x = src[i + (int64_t)n * j], y = src[j + (int64_t)n * i];
      G[il + (size_t)nr * j] = cmake(0.5 * (x.x + y.x) + (i == j ? sigma : 0.0), i == j ? 0.0 : 0.5 * (x.y - y.y));
    }
    __syncthreads();

    bool converged = false;
    for (int sweep = 0; sweep < EC_MAX_SWEEPS && !converged; sweep++) {
      int any_act = 0;
      for (int r = 0; r < N - 1; r++) {
        // ---- step 1: partial (alpha, beta, gamma) over the local rows; 4 lanes per pair, 8 pairs per warp ----
        for (int sb = warp * 8; sb < half; sb += (EC_THREADS / 32) * 8) {  // warp-uniform trip count (shuffles inside)
          const int s = sb + (lane >> 2);
          int p = 0, q = n;
          if (s < half) rr_pair(N, r, s, p, q);
          double al = 0.0, be = 0.0, gr = 0.0, gi = 0.0;
          if (q < n) {
            const c128 *gp = G + (size_t)nr * p, *gq = G + (size_t)nr * q;
            for (int il = lane & 3; il < nloc; il += 4) {
              const c128 x = gp[il], y = gq[il];
              al = fma(x.x, x.x, fma(x.y, x.y, al));
              be = fma(y.x, y.x, fma(y.y, y.y, be));
              gr = fma(x.x, y.x, fma(x.y, y.y, gr));   // conj(x) * y
              gi = fma(x.x, y.y, fma(-x.y, y.x, gi));
            }
          }
          al += __shfl_xor_sync(0xffffffffu, al, 1); be += __shfl_xor_sync(0xffffffffu, be, 1);
          gr += __shfl_xor_sync(0xffffffffu, gr, 1); gi += __shfl_xor_sync(0xffffffffu, gi, 1);
          al += __shfl_xor_sync(0xffffffffu, al, 2); be += __shfl_xor_sync(0xffffffffu, be, 2);
          gr += __shfl_xor_sync(0xffffffffu, gr, 2); gi += __shfl_xor_sync(0xffffffffu, gi, 2);
          if (q < n && (lane & 3) == 0) {
            double4 *dst = cluster.map_shared_rank(part, s % csize);
            dst[(size_t)crank * hp + s / csize] = make_double4(al, be, gr, gi);
          }
        }
        cluster.sync();
        // ---- step 2: the owner reduces over the CTAs, builds the rotation and broadcasts it ----
        if (tid < hp) {
          const int s = crank + csize * tid;
          if (s < half) {
            int p, q;
            rr_pair(N, r, s, p, q);
            RotB R;
            R.c = 1.0; R.sr = 0.0; R.si = 0.0; R.act = 0.0;
            if (q < n) {
              double al = 0.0, be = 0.0, gr = 0.0, gi = 0.0;
              for (int c2 = 0; c2 < csize; c2++) {
                const double4 v = part[(size_t)c2 * hp + tid];
                al += v.x; be += v.y; gr += v.z; gi += v.w;
              }
              if (gr * gr + gi * gi > tol2 * al * be) {
                const Rot J = make_rot(al, be, cmake(gr, gi));
                R.c = J.c; R.sr = J.sr; R.si = J.si; R.act = 1.0;
                my_rot++;
              }
            }
            for (int c2 = 0; c2 < csize; c2++) cluster.map_shared_rank(rot, c2)[s] = R;
          }
        }
        cluster.sync();
        // ---- step 3: rotate the local rows of every column pair ----
        for (int e = tid; e < half * nloc; e += EC_THREADS) {
          const int il = e % nloc, s = e / nloc;
          const RotB R = rot[s];
          if (R.act != 0.0) {
            any_act = 1;
            int p, q;
            rr_pair(N, r, s, p, q);
            Rot J;
            J.c = R.c; J.sr = R.sr; J.si = R.si; J.pad = 0.0;
            c128 xp = G[il + (size_t)nr * p], xq = G[il + (size_t)nr * q];
            apply_cols(xp, xq, J);
            G[il + (size_t)nr * p] = xp;
            G[il + (size_t)nr * q] = xq;
          }
        }
        __syncthreads();
      }
      // every CTA sees every rotation of the sweep (nloc > 0 for all CTAs), so the decision is uniform in the cluster
      converged = __syncthreads_or(any_act) == 0;
    }
    if (!converged && status != nullptr && tid == 0 && crank == 0) atomicExch(status, 1);

    // ---- eigenvectors: normalised columns of G ----
    for (int j = warp; j < n; j += EC_THREADS / 32) {
      double a2 = 0.0;
      for (int il = lane; il < nloc; il += 32) a2 += cabs2(G[il + (size_t)nr * j]);
      a2 = warp_sum(a2);
      if (lane == 0) nrm2[(size_t)crank * n + j] = a2;
    }
    __threadfence();
    cluster.sync();
    for (int e = tid; e < n * nloc; e += EC_THREADS) {
      const int il = e % nloc, j = e / nloc;
      double a2 = 0.0;
      for (int c2 = 0; c2 < csize; c2++) a2 += nrm2[(size_t)c2 * n + j];
      const double inv = rsqrt(a2);
      const c128 g = G[il + (size_t)nr * j];
      Vtmp[(r0 + il) + (int64_t)n * j] = cmake(g.x * inv, g.y * inv);
    }
    __threadfence();
    cluster.sync();
    // ---- eigenvalues: Rayleigh quotients Re(v_j^dagger A v_j) with the original matrix, EC_RQ_COLS columns per warp ----
    const int nblk = (n + EC_RQ_COLS - 1) / EC_RQ_COLS;
    for (int jb = crank * (EC_THREADS / 32) + warp; jb < nblk; jb += csize * (EC_THREADS / 32)) {
      const int j0 = jb * EC_RQ_COLS;
      double acc[EC_RQ_COLS];
#pragma unroll
      for (int jj = 0; jj < EC_RQ_COLS; jj++) acc[jj] = 0.0;
      for (int i = lane; i < n; i += 32) {
        c128 wv[EC_RQ_COLS];
#pragma unroll
        for (int jj = 0; jj < EC_RQ_COLS; jj++) wv[jj] = cmake(0.0, 0.0);
        for (int l = 0; l < n; l++) {
          const c128 a = src[i + (int64_t)n * l];
#pragma unroll
          for (int jj = 0; jj < EC_RQ_COLS; jj++) {
            const int j = j0 + jj < n ? j0 + jj : n - 1;
            cfma(wv[jj], a, Vtmp[l + (int64_t)n * j]);
          }
        }
#pragma unroll
        for (int jj = 0; jj < EC_RQ_COLS; jj++) {
          const int j = j0 + jj < n ? j0 + jj : n - 1;
          const c128 v = Vtmp[i + (int64_t)n * j];
          acc[jj] += v.x * wv[jj].x + v.y * wv[jj].y;
        }
      }
#pragma unroll
      for (int jj = 0; jj < EC_RQ_COLS; jj++) {
        const double t = warp_sum(acc[jj]);
        if (lane == 0 && j0 + jj < n) lam[j0 + jj] = t;
      }
    }
    __threadfence();
    cluster.sync();
    // ---- ascending order by rank counting, permuted store of the local rows ----
    int *rank_of = reinterpret_cast<int *>(rot);
    for (int j = tid; j < n; j += EC_THREADS) {
      const double lj = lam[j];
      int rank = 0;
      for (int i = 0; i < n; i++) {
        const double li = lam[i];
        rank += (li < lj) || (li == lj && i < j);
      }
      rank_of[j] = rank;
      if (crank == 0) {
        double out = lj;
        if (sqrt_mode) out = lj > 0.0 ? sqrt(lj) : -sqrt(-lj);
        evals[b * n + rank] = out;
      }
    }
    __syncthreads();
    c128 *dst = Vout + b * (int64_t)n * n;
    for (int e = tid; e < n * nloc; e += EC_THREADS) {
      const int il = e % nloc, j = e / nloc;
      dst[(r0 + il) + (int64_t)n * rank_of[j]] = Vtmp[(r0 + il) + (int64_t)n * j];
    }
    cluster.sync();  // scratch, rot and part are reused by the next matrix
  }
  if (work != nullptr && my_rot) atomicAdd(work, my_rot);
}

// cluster size (1, 2, 4, 8) and rows per CTA for an n x n solve, 0 if it does not fit in distributed shared memory
static int eigh_cluster_plan(int n, int64_t batch, int *nr_out, size_t *smem_out) {
  const int half = (n + (n & 1)) >> 1;
  int best = 0;
  for (int cs = 1; cs <= 8; cs *= 2) {
    const int nr = (n + cs - 1) / cs;
    if ((int64_t)nr * (cs - 1) >= n) continue;  // every CTA must own at least one row
    const int hp = (half + cs - 1) / cs;
    const size_t smem = ((sizeof(c128) * (size_t)n * nr + 31) & ~(size_t)31) + sizeof(double4) * (size_t)cs * hp +
                        sizeof(RotB) * (size_t)half;
    if (smem > (size_t)220 * 1024) continue;
    if (best == 0) best = cs;                      // smallest cluster that fits: best throughput for large batches
    if (batch * cs <= device_sm_count()) best = cs;              // few matrices: spread each one over more SMs
  }
  if (best) {
    const int nr = (n + best - 1) / best, hp = (half + best - 1) / best;
    *nr_out = nr;
    *smem_out = ((sizeof(c128) * (size_t)n * nr + 31) & ~(size_t)31) + sizeof(double4) * (size_t)best * hp +
                sizeof(RotB) * (size_t)half;
  }
  return best;
}

static int eigh_large_grid(int64_t batch) {
  const int nsm = device_sm_count();
  return (int)(batch < nsm ? batch : nsm);
}

size_t eigh_large_scratch_bytes(int n, int64_t batch) {
  if (n <= EIGH_SMALL_MAX_N) return 0;
  return (size_t)eigh_large_grid(batch) * 2 * (size_t)n * n * sizeof(c128);
}

cudaError_t launch_eigh_batched(const c128 *A, int64_t stride_a, int n, int64_t batch, double *evals, c128 *V,
                                int sqrt_mode, int32_t *status, c128 *scratch_large, unsigned long long *work,
                                cudaStream_t st) {
  return launch_eigh_batched_algo(A, stride_a, n, batch, evals, V, sqrt_mode, status, scratch_large, EPW_EIGH_AUTO, work, st);
}

// Kernel choice: the thread-per-matrix solver needs tens of thousands of matrices to fill the GPU (32 matrices per
// 64-thread CTA) and is the throughput kernel of the per-pair H(k+q) solves; small batches (H(k) of a tiny grid, D(q)
// of a q-batch) finish sooner on the warp-per-matrix kernel, which spreads one matrix over 32 lanes.
cudaError_t launch_eigh_batched_algo(const c128 *A, int64_t stride_a, int n, int64_t batch, double *evals, c128 *V,
                                     int sqrt_mode, int32_t *status, c128 *scratch_large, int algo,
                                     unsigned long long *work, cudaStream_t st) {
  if (batch <= 0) return cudaSuccess;
  if (algo == EPW_EIGH_THREAD && !eigh_thread_supported(n)) return cudaErrorInvalidValue;
  if (algo == EPW_EIGH_THREAD || (algo == EPW_EIGH_AUTO && eigh_thread_supported(n) && batch >= 2048))
    return launch_eigh_thread(A, stride_a, n, batch, evals, V, sqrt_mode, status, work, st);
  if (algo == EPW_EIGH_COLS && !eigh_cols_supported(n)) return cudaErrorInvalidValue;
  if (algo == EPW_EIGH_COLS || (algo == EPW_EIGH_AUTO && eigh_cols_supported(n) && batch >= 2048))
    return launch_eigh_cols(A, stride_a, n, batch, evals, V, sqrt_mode, status, work, st);
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
    int nr = 0;
    size_t csmem = 0;
    const int cs = eigh_cluster_plan(n, batch, &nr, &csmem);
    if (cs > 0) {
      cudaError_t e = cudaFuncSetAttribute(eigh_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)csmem);
      if (e != cudaSuccess) return e;
      cudaLaunchConfig_t cfg = {};
      cudaLaunchAttribute attr[1];
      attr[0].id = cudaLaunchAttributeClusterDimension;
      attr[0].val.clusterDim.x = cs;
      attr[0].val.clusterDim.y = 1;
      attr[0].val.clusterDim.z = 1;
      cfg.attrs = attr;
      cfg.numAttrs = 1;
      cfg.blockDim = dim3(EC_THREADS);
      cfg.dynamicSmemBytes = csmem;
      cfg.stream = st;
      cfg.gridDim = dim3(cs);
      int max_clusters = 0;
      e = cudaOccupancyMaxActiveClusters(&max_clusters, eigh_cluster_kernel, &cfg);
      if (e != cudaSuccess) return e;
      if (max_clusters > 0) {
        const int64_t cap = std::min<int64_t>(max_clusters, eigh_large_grid(batch));
        cfg.gridDim = dim3((unsigned)(std::min<int64_t>(batch, cap) * cs));
        return cudaLaunchKernelEx(&cfg, eigh_cluster_kernel, A, stride_a, n, batch, evals, V, sqrt_mode, status,
                                  scratch_large, nr, work);
      }
    }
    const int half = (n + (n & 1)) >> 1;
    const size_t smem = (size_t)half * sizeof(Rot) + (size_t)n * sizeof(double) + (size_t)n * sizeof(int);
    eigh_large_kernel<<<eigh_large_grid(batch), EIGH_LARGE_THREADS, smem, st>>>(A, stride_a, n, batch, evals, V,
                                                                                sqrt_mode, status, scratch_large);
  }
  return cudaGetLastError();
}

}  // namespace epw
