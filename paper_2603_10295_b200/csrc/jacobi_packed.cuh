// jacobi_packed.cuh -- the arithmetic of the thread-per-matrix Hermitian Jacobi eigensolver (eigh_thread.cu), S3b of the
// path (BASELINE.json north_star stage 3; PAPER.md:L72 U_k, L54 u(q) are the paper's only mention of these quantities).
//
// Two-sided cyclic Jacobi, A <- J^dagger A J, V <- V J, on a Hermitian matrix held in PACKED form: the real diagonal
// d[i] and the strict upper triangle u[i][j] = a_ij (i < j); a_ji = conj(a_ij) is implied, so one plane rotation costs
// (n-2) column-pair updates for A instead of the 2n of the full row + column pass, plus n for the rows of V.
//   a_pq = r e^{i phi}, tau = (a_qq - a_pp)/(2r), t = sgn(tau)/(|tau| + sqrt(1 + tau^2)), c = 1/sqrt(1 + t^2), s = t c
//   (evaluated in the equivalent half-angle form, see jacobi_rotate_packed),
//   S = s e^{i phi},  J = [[c, S], [-conj(S), c]] on rows/columns (p, q)           (same convention as eigh_jacobi.cu)
//   a_pp <- a_pp - t r,  a_qq <- a_qq + t r,  a_pq <- 0,
//   (a_jp, a_jq) <- (c a_jp - conj(S) a_jq,  S a_jp + c a_jq)   for every j not in {p, q},
//   (v_ip, v_iq) <- (c v_ip - conj(S) v_iq,  S v_ip + c v_iq)   for every row i of V.
// Pairs follow the round-robin tournament over NE = n rounded up to even players (NE - 1 rounds of NE/2 disjoint pairs);
// every index below is a compile-time constant once the loops over (round, slot) are unrolled, so d, u and V live in
// registers.  The functions are __host__ __device__ so that the same arithmetic can be exercised on a CPU.
#pragma once
#include <math.h>

#include "common.cuh"

namespace epw {

template <int N>
struct RoundRobin {
  static constexpr int NE = N + (N & 1);
  static constexpr int ROUNDS = NE - 1;
  static constexpr int HALF = NE / 2;
  __host__ __device__ static constexpr int first(int r, int s) { return s == 0 ? NE - 1 : (r + s) % (NE - 1); }
  __host__ __device__ static constexpr int second(int r, int s) { return s == 0 ? r : (r - s + (NE - 1)) % (NE - 1); }
  __host__ __device__ static constexpr int p(int r, int s) { return first(r, s) < second(r, s) ? first(r, s) : second(r, s); }
  __host__ __device__ static constexpr int q(int r, int s) { return first(r, s) < second(r, s) ? second(r, s) : first(r, s); }
};

struct PlaneRot {
  double c, sr, si;  // S = sr + i si
};

__host__ __device__ __forceinline__ double jp_rsqrt(double x) {
#ifdef __CUDA_ARCH__
  return rsqrt(x);
#else
  return 1.0 / sqrt(x);
#endif
}

// Hermitian matrix element a_ij from the packed form (i != j)
template <int N>
__host__ __device__ __forceinline__ c128 herm_get(const c128 (&u)[N][N], int i, int j) {
  return i < j ? u[i][j] : make_double2(u[j][i].x, -u[j][i].y);
}
template <int N>
__host__ __device__ __forceinline__ void herm_set(c128 (&u)[N][N], int i, int j, c128 v) {
  if (i < j) u[i][j] = v;
  else u[j][i] = make_double2(v.x, -v.y);
}

// One plane rotation (p < q) on the packed matrix; returns the rotation for the eigenvector update.
// Off-diagonal elements with |a_pq|^2 < 1e-280 are treated as already zero (identity rotation).
template <int N>
__host__ __device__ __forceinline__ PlaneRot jacobi_rotate_packed(double (&d)[N], c128 (&u)[N][N], int p, int q) {
  const c128 apq = u[p][q];
  const double r2 = fma(apq.x, apq.x, apq.y * apq.y);
  const bool live = r2 >= 1e-280;
  // half-angle form of the same rotation (tan 2 theta = r / a, |theta| <= pi/4): two dependent rsqrt instead of
  // rsqrt -> sqrt -> divide -> rsqrt, and no subtraction anywhere (cos 2 theta in [0,1], x in [1/2, 1]):
  //   h = 1/sqrt(a^2 + r^2), cos 2theta = |a| h, c = sqrt(x), x = (1 + cos 2theta)/2, S = sgn(a) a_pq h / (2c), t r = sgn(a) r^2 h / (2x)
  const double a = 0.5 * (d[q] - d[p]);
  const double h = jp_rsqrt(live ? fma(a, a, r2) : 1.0);
  const double x = fma(0.5 * fabs(a), h, 0.5);
  const double rc = jp_rsqrt(x);
  const double sor = copysign(0.5 * h * rc, a);
  PlaneRot R;
  R.c = live ? x * rc : 1.0;
  R.sr = live ? sor * apq.x : 0.0;
  R.si = live ? sor * apq.y : 0.0;
  const double tr = live ? copysign(0.5 * r2 * h * (rc * rc), a) : 0.0;
  d[p] -= tr;
  d[q] += tr;
  if (live) u[p][q] = make_double2(0.0, 0.0);
#pragma unroll
  for (int j = 0; j < N; j++) {
    if (j == p || j == q) continue;
    const c128 xp = herm_get<N>(u, j, p), xq = herm_get<N>(u, j, q);
    c128 yp, yq;
    yp.x = R.c * xp.x - (R.sr * xq.x + R.si * xq.y);
    yp.y = R.c * xp.y - (R.sr * xq.y - R.si * xq.x);
    yq.x = R.c * xq.x + (R.sr * xp.x - R.si * xp.y);
    yq.y = R.c * xq.y + (R.sr * xp.y + R.si * xp.x);
    herm_set<N>(u, j, p, yp);
    herm_set<N>(u, j, q, yq);
  }
  return R;
}

// (v_p, v_q) <- (v_p, v_q) J for one row of V
__host__ __device__ __forceinline__ void jacobi_apply_v(c128 &vp, c128 &vq, const PlaneRot &R) {
  const c128 a = vp, b = vq;
  vp.x = R.c * a.x - (R.sr * b.x + R.si * b.y);
  vp.y = R.c * a.y - (R.sr * b.y - R.si * b.x);
  vq.x = R.c * b.x + (R.sr * a.x - R.si * a.y);
  vq.y = R.c * b.y + (R.sr * a.y + R.si * a.x);
}

// squared Frobenius norm of the strict off-diagonal part
template <int N>
__host__ __device__ __forceinline__ double herm_off2(const c128 (&u)[N][N]) {
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < N; i++)
#pragma unroll
    for (int j = i + 1; j < N; j++) s = fma(u[i][j].x, u[i][j].x, fma(u[i][j].y, u[i][j].y, s));
  return 2.0 * s;
}

}  // namespace epw
