// eigh_cols.cu -- S3b for 9 <= n <= 16 and large batches (BASELINE.json configs[2], MoS2-like: Nk*Nq solves of 11 x 11;
// north_star stage 3): ONE-SIDED (Hestenes) Jacobi with the matrix distributed BY COLUMN PAIRS over the warps of a CTA,
// lane = matrix, columns in registers.
//
// Method (the one of the cluster kernel in eigh_jacobi.cu, at register scale).  With mu = tr(A)/n and
// sigma = ||A_h - mu I||_F - mu (A_h = Hermitian part), G = A_h + sigma I is Hermitian positive definite.  Plane rotations
// from the right orthogonalise its columns:
//     alpha = ||g_p||^2, beta = ||g_q||^2, gamma = g_p^dagger g_q,   J = rotation diagonalising [[alpha, gamma], [conj gamma, beta]]
//     (g_p, g_q) <- (g_p, g_q) J            (formulas of jacobi_packed.cuh / eigh_jacobi.cu make_rot)
// At convergence G V = V Sigma, so v_j = g_j / ||g_j||: no eigenvector accumulation and no row pass -- one rotation costs
// 20 n + 60 FP64 instructions.  Eigenvalues are the Rayleigh quotients v_j^dagger A_h v_j of the ORIGINAL matrix.
//
// Distribution.  N = n rounded up to even (an odd n gets a zero pad column, which never rotates), L = N / 2 warps;
// lane l of every warp works on matrix 32 * blockIdx + l.  Warp s holds the two columns at positions (2 s, 2 s + 1) of a
// linear array as (lo, hi).  ODD-EVEN ordering: N steps per sweep alternate the pairings (0,1)(2,3).. and (1,2)(3,4)..,
// and the two columns of a pair swap positions after every rotation, so that every pair of columns meets exactly once
// per sweep (the odd-even transposition network).  In terms of the warps: after a step of the first kind warp s keeps
// its rotated lo (now at position 2s+1), sends its rotated hi (now at 2s) to warp s-1 and receives its new hi from warp
// s+1; after a step of the second kind it keeps hi, sends lo to warp s+1 and receives its new lo from warp s-1; the
// columns at the two ends sit out one step and turn around.  A moving column goes through shared memory
// ([slot][row][lane], 16-byte accesses, conflict free), one __syncthreads per step.
// Convergence: |gamma|^2 <= n eps^2 alpha beta for every pair of a sweep and every matrix of the CTA.
#include "common.cuh"
#include "jacobi_packed.cuh"

namespace epw {

constexpr int EC2_MAX_SWEEPS = 40;

template <int NN>
struct ColsCfg {
  static constexpr int N = NN + (NN & 1);
  static constexpr int L = N / 2;
  static constexpr int THREADS = 32 * L;
  static constexpr size_t COL_BYTES = sizeof(c128) * NN * 32;          // one column of 32 matrices
  static constexpr size_t BUF_BYTES = COL_BYTES * L;                   // one transition buffer
  static constexpr size_t RED_BYTES = sizeof(double) * 2 * L * 32;     // (trace | norm) partials
  static constexpr size_t LAM_BYTES = sizeof(double) * N * 32;
  static constexpr size_t SMEM = 2 * BUF_BYTES + RED_BYTES + LAM_BYTES;
};

template <int NN>
__device__ __forceinline__ bool hestenes_rotate(c128 (&lo)[NN], c128 (&hi)[NN], double tol2) {
  double al = 0.0, be = 0.0, gr = 0.0, gi = 0.0;
#pragma unroll
  for (int i = 0; i < NN; i++) {
    al = fma(lo[i].x, lo[i].x, fma(lo[i].y, lo[i].y, al));
    be = fma(hi[i].x, hi[i].x, fma(hi[i].y, hi[i].y, be));
    gr = fma(lo[i].x, hi[i].x, fma(lo[i].y, hi[i].y, gr));   // gamma = conj(lo) . hi
    gi = fma(lo[i].x, hi[i].y, fma(-lo[i].y, hi[i].x, gi));
  }
  const double r2 = fma(gr, gr, gi * gi);
  const bool live = r2 > tol2 * al * be && r2 >= 1e-280;
  if (!__any_sync(0xffffffffu, live)) return false;
  // half-angle form (jacobi_packed.cuh): two dependent rsqrt, no subtraction
  const double a = 0.5 * (be - al);
  const double h = rsqrt(live ? fma(a, a, r2) : 1.0);
  const double x = fma(0.5 * fabs(a), h, 0.5);
  const double rc = rsqrt(x);
  const double sor = copysign(0.5 * h * rc, a);
  PlaneRot R;
  R.c = live ? x * rc : 1.0;
  R.sr = live ? sor * gr : 0.0;
  R.si = live ? sor * gi : 0.0;
#pragma unroll
  for (int i = 0; i < NN; i++) jacobi_apply_v(lo[i], hi[i], R);
  return true;
}

template <int NN>
__global__ void __launch_bounds__(ColsCfg<NN>::THREADS, (NN <= 12 ? 2 : 1))
    eigh_cols_kernel(const c128 *__restrict__ Ain, int64_t stride_a, int64_t batch, double *__restrict__ evals,
                     c128 *__restrict__ Vout, int sqrt_mode, int32_t *__restrict__ status,
                     unsigned long long *__restrict__ work) {
  typedef ColsCfg<NN> Cfg;
  constexpr int N = Cfg::N, L = Cfg::L;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128 *bufA = reinterpret_cast<c128 *>(smem_raw);                       // lo columns in flight (second-kind steps)
  c128 *bufB = reinterpret_cast<c128 *>(smem_raw + Cfg::BUF_BYTES);      // hi columns in flight (first-kind steps)
  double *red = reinterpret_cast<double *>(smem_raw + 2 * Cfg::BUF_BYTES);
  double *lam = reinterpret_cast<double *>(smem_raw + 2 * Cfg::BUF_BYTES + Cfg::RED_BYTES);
  const int s = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t bm = (int64_t)blockIdx.x * 32 + lane;
  const bool have = bm < batch;
  const c128 *src = Ain + (have ? bm : 0) * stride_a;

  // ---- centre and shift: mu = tr/n, G = (A_h - mu I) + ||A_h - mu I||_F I ----
  const int ja = 2 * s, jb = 2 * s + 1;   // jb == NN: the zero pad column of an odd n
  double tr = 0.0;
  if (have) {
    tr = src[ja + NN * ja].x;
    if (jb < NN) tr += src[jb + NN * jb].x;
  }
  red[s * 32 + lane] = tr;
  __syncthreads();
  tr = 0.0;
#pragma unroll
  for (int w = 0; w < L; w++) tr += red[w * 32 + lane];
  const double mu = tr / NN;
  c128 lo[NN], hi[NN];
  double fro2 = 0.0;
#pragma unroll
  for (int i = 0; i < NN; i++) {
    c128 va = make_double2(0.0, 0.0), vb = make_double2(0.0, 0.0);
    if (have) {
      const c128 x = src[i + NN * ja], y = src[ja + NN * i];
      va = make_double2(0.5 * (x.x + y.x) - (i == ja ? mu : 0.0), i == ja ? 0.0 : 0.5 * (x.y - y.y));
      if (jb < NN) {
        const c128 x2 = src[i + NN * jb], y2 = src[jb + NN * i];
        vb = make_double2(0.5 * (x2.x + y2.x) - (i == jb ? mu : 0.0), i == jb ? 0.0 : 0.5 * (x2.y - y2.y));
      }
    }
    lo[i] = va;
    hi[i] = vb;
    fro2 = fma(va.x, va.x, fma(va.y, va.y, fma(vb.x, vb.x, fma(vb.y, vb.y, fro2))));
  }
  red[(L + s) * 32 + lane] = fro2;
  __syncthreads();
  fro2 = 0.0;
#pragma unroll
  for (int w = 0; w < L; w++) fro2 += red[(L + w) * 32 + lane];
  const double shift = fro2 > 0.0 ? sqrt(fro2) : 1.0;
  if (have) {
#pragma unroll
    for (int i = 0; i < NN; i++) {
      if (i == ja) lo[i].x += shift;
      if (i == jb) hi[i].x += shift;
    }
  }
  const double tol2 = (double)NN * 1.2325951644078309e-32;  // (sqrt(n) 2^-53)^2

  c128 *outA = bufA + ((size_t)s * NN) * 32 + lane, *outB = bufB + ((size_t)s * NN) * 32 + lane;
  const c128 *inB = bufB + ((size_t)(s + 1) * NN) * 32 + lane;                               // hi from warp s+1
  const c128 *inA = s > 0 ? bufA + ((size_t)(s - 1) * NN) * 32 + lane : bufB + lane;          // lo from warp s-1 / parked
  bool converged = false;
  int nrot = 0;  // rotations this warp executed (for the optional work counter)
  for (int sweep = 0; sweep < EC2_MAX_SWEEPS && !converged; sweep++) {
    int any_act = 0;
    for (int step2 = 0; step2 < L; step2++) {
      // ---- first kind: pairs (2s, 2s+1) ----
      { const bool a = hestenes_rotate<NN>(lo, hi, tol2); any_act |= a ? 1 : 0; nrot += a ? 1 : 0; }
#pragma unroll
      for (int i = 0; i < NN; i++) outB[(size_t)i * 32] = hi[i];
      __syncthreads();
      if (s < L - 1) {
#pragma unroll
        for (int i = 0; i < NN; i++) hi[i] = inB[(size_t)i * 32];
        // ---- second kind: pairs (2s+1, 2s+2); the last warp sits out ----
        { const bool a = hestenes_rotate<NN>(lo, hi, tol2); any_act |= a ? 1 : 0; nrot += a ? 1 : 0; }
#pragma unroll
        for (int i = 0; i < NN; i++) outA[(size_t)i * 32] = lo[i];
      } else {
#pragma unroll
        for (int i = 0; i < NN; i++) hi[i] = lo[i];   // its lo (position N-1) turns around and becomes hi
      }
      __syncthreads();
#pragma unroll
      for (int i = 0; i < NN; i++) lo[i] = inA[(size_t)i * 32];
    }
    converged = __syncthreads_or(any_act) == 0;
  }
  if (!converged && status != nullptr && threadIdx.x == 0) atomicExch(status, 1);
  if (work != nullptr) {
    const unsigned m = __ballot_sync(0xffffffffu, have);
    if (lane == 0) atomicAdd(work, (unsigned long long)nrot * __popc(m));
  }

  // ---- eigenvectors = normalised columns; eigenvalues = Rayleigh quotients with the original Hermitian part ----
  double na = 0.0, nb2 = 0.0;
#pragma unroll
  for (int i = 0; i < NN; i++) {
    na = fma(lo[i].x, lo[i].x, fma(lo[i].y, lo[i].y, na));
    nb2 = fma(hi[i].x, hi[i].x, fma(hi[i].y, hi[i].y, nb2));
  }
  const bool pad_a = !(na > 0.0), pad_b = !(nb2 > 0.0);  // the zero pad column of an odd n (G is positive definite)
  const double ia = pad_a ? 0.0 : rsqrt(na), ib = pad_b ? 0.0 : rsqrt(nb2);
#pragma unroll
  for (int i = 0; i < NN; i++) {
    lo[i].x *= ia; lo[i].y *= ia;
    hi[i].x *= ib; hi[i].y *= ib;
  }
  double la = 0.0, lb = 0.0;
  if (have) {
#pragma unroll
    for (int i = 0; i < NN; i++) {
      const double dii = src[i + NN * i].x;
      la = fma(dii, fma(lo[i].x, lo[i].x, lo[i].y * lo[i].y), la);
      lb = fma(dii, fma(hi[i].x, hi[i].x, hi[i].y * hi[i].y), lb);
#pragma unroll
      for (int l = i + 1; l < NN; l++) {
        const c128 x = src[i + NN * l], y = src[l + NN * i];
        const c128 h = make_double2(0.5 * (x.x + y.x), 0.5 * (x.y - y.y));   // A_h[i][l]
        // 2 Re( conj(v_i) h v_l )
        c128 pa = make_double2(0.0, 0.0), pb = make_double2(0.0, 0.0);
        cfma_conj(pa, lo[i], lo[l]);
        cfma_conj(pb, hi[i], hi[l]);
        la = fma(2.0, h.x * pa.x - h.y * pa.y, la);
        lb = fma(2.0, h.x * pb.x - h.y * pb.y, lb);
      }
    }
  }
  const double big = __longlong_as_double(0x7ff0000000000000LL);
  lam[(2 * s) * 32 + lane] = pad_a ? big : la;
  lam[(2 * s + 1) * 32 + lane] = pad_b ? big : lb;
  __syncthreads();
  if (have) {
    int ra = 0, rb = 0;
#pragma unroll
    for (int j = 0; j < N; j++) {
      const double lj = lam[j * 32 + lane];
      ra += (lj < la) || (lj == la && j < 2 * s);
      rb += (lj < lb) || (lj == lb && j < 2 * s + 1);
    }
    c128 *dst = Vout + bm * (int64_t)(NN * NN);
    if (!pad_a) {
      double out = la;
      if (sqrt_mode) out = out > 0.0 ? sqrt(out) : -sqrt(-out);
      evals[bm * NN + ra] = out;
#pragma unroll
      for (int i = 0; i < NN; i++) dst[i + NN * ra] = lo[i];
    }
    if (!pad_b) {
      double out = lb;
      if (sqrt_mode) out = out > 0.0 ? sqrt(out) : -sqrt(-out);
      evals[bm * NN + rb] = out;
#pragma unroll
      for (int i = 0; i < NN; i++) dst[i + NN * rb] = hi[i];
    }
  }
}

template <int NN>
static cudaError_t launch_cols_n(const c128 *A, int64_t stride_a, int64_t batch, double *evals, c128 *V, int sqrt_mode,
                                 int32_t *status, unsigned long long *work, cudaStream_t st) {
  typedef ColsCfg<NN> Cfg;
  cudaError_t e = cudaFuncSetAttribute(eigh_cols_kernel<NN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
  if (e != cudaSuccess) return e;
  eigh_cols_kernel<NN><<<(unsigned)ceil_div(batch, 32), Cfg::THREADS, Cfg::SMEM, st>>>(A, stride_a, batch, evals, V,
                                                                                      sqrt_mode, status, work);
  return cudaGetLastError();
}

bool eigh_cols_supported(int n) { return n >= 9 && n <= 16; }

cudaError_t launch_eigh_cols(const c128 *A, int64_t stride_a, int n, int64_t batch, double *evals, c128 *V,
                             int sqrt_mode, int32_t *status, unsigned long long *work, cudaStream_t st) {
  if (batch <= 0) return cudaSuccess;
  switch (n) {
    case 9: return launch_cols_n<9>(A, stride_a, batch, evals, V, sqrt_mode, status, work, st);
    case 10: return launch_cols_n<10>(A, stride_a, batch, evals, V, sqrt_mode, status, work, st);
    case 11: return launch_cols_n<11>(A, stride_a, batch, evals, V, sqrt_mode, status, work, st);
    case 12: return launch_cols_n<12>(A, stride_a, batch, evals, V, sqrt_mode, status, work, st);
    case 13: return launch_cols_n<13>(A, stride_a, batch, evals, V, sqrt_mode, status, work, st);
    case 14: return launch_cols_n<14>(A, stride_a, batch, evals, V, sqrt_mode, status, work, st);
    case 15: return launch_cols_n<15>(A, stride_a, batch, evals, V, sqrt_mode, status, work, st);
    case 16: return launch_cols_n<16>(A, stride_a, batch, evals, V, sqrt_mode, status, work, st);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace epw
