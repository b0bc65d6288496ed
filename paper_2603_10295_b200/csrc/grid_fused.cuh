// grid_fused.cuh -- uniform-grid path, Nb <= 16: the LAST axis pass of S2, S4b and |g|^2 in ONE kernel, all three products
// on the FP64 tensor path (mma.sync.m8n8k4.f64, SASS DMMA), so that g~(k,q) never goes to HBM.
//
//   g~_{m'n' nu}(k,q) = sum_{n1} e^{2 pi i (i1+s1) n1 / N1} T2[n1][(i2,i3)][nu,n',m']      (last axis of the factorised
//                                                         Re -> k sum, re_to_k_grid.cu; Eq. 10)
//   g_{mn nu}(k,q)    = sum_{m'n'} conj(U_{k+q}[m',m]) g~_{m'n' nu} U_k[n',n],   out = |g_{mn nu}|^2   (
//                                                         BASELINE.json north_star stage 4; reading G4)
// In the two-kernel grid path the last pass writes g~ (16 Nb^2 Nm bytes per pair) and rotate_g2.cu reads it back: 852 of
// the 1,371 MB moved per q on configs[1].  Here the L1 rows T2[.][cell][mode group] of one (i2,i3) cell of the grid come
// into shared memory by bulk TMA, and a warp takes a QUAD of four consecutive i1 of that cell:
//   pass       C[c][(j,re/im)] = sum_{(n1,re/im)} T2[n1][c] (x) p[n1][j]     one DMMA tile = 8 columns c x 4 pairs j:
//              A' fragments = re/im of T2 straight from shared memory (one LDS.64 per DMMA), B' fragments = the 2x2 real
//              embedding of the four pairs' phases, held in registers; K = 2 L1 real.  The tile lands as one complex
//              g~_j[c] per lane and goes to a per-warp staging buffer [pair][c] (the rotation wants all of ONE pair in a
//              fragment, the pass produces four pairs side by side: the exchange has to cross lanes);
//   product 1  T[m'][n]  = sum_n' g~[n'][m'] Uk[n'][n]        A' from the staging buffer, B' = embedding of U_k;
//   product 2  |sum_m' T[m'][n] conj(Ukq[m'][m])|^2           T through a second staging buffer, B'' = conj(U_{k+q});
// the U fragments of the four pairs stay in registers over all modes when Nb <= 8.
// HBM traffic per pair: 32 Nb^2 (the two U) + 8 Nb^2 Nm (output) bytes; T2 (16 Nb^2 Nm L1 N2 N3 bytes per q) is L2-resident.
// FP64 work per pair: 8 L1 Nb^2 Nm (pass) + 16 Nb^3 Nm (rotation) flops, all of it DMMA.
#pragma once
#include <type_traits>

#include "common.cuh"
#include "dmma_pipe.cuh"

namespace epw {

template <int NB>
struct GF {
  static constexpr int NBB = NB * NB;
  static constexpr int KS = (2 * NB + 3) / 4;   // k-steps of 4 real of the two rotation products
  static constexpr int NT = (2 * NB + 7) / 8;   // column tiles of 8 real
  static constexpr int MTR = (NB + 7) / 8;      // row tiles of the rotation products per mode
  static constexpr int MTP = (NBB + 7) / 8;     // row tiles (columns c of g~) of the pass per mode
  static constexpr int NBP = NB + ((12 - (NB & 7)) & 7);     // row (n') pitch of the g~ staging buffer: = 4 (mod 8) complex
  static constexpr int PST = NB * NBP + ((10 - ((NB * NBP) & 7)) & 7);   // pair stride of that buffer: = 2 (mod 8) complex
  static constexpr int SP = NB + ((6 - (NB & 3)) & 3);       // row pitch of the T staging buffer: = 2 (mod 4) complex
  static constexpr int TROWS = MTR * 8;
  static constexpr bool UREG = NB <= 8;         // U fragments of the four pairs of a quad resident over all modes
  static_assert(2 * KS <= SP, "T pitch must cover the padded K range");
};

// row pitch of the T2 rows in shared memory: = 4 (mod 8) complex, so that the two rows (n1 = 2 ks, 2 ks + 1) a pass fragment
// reads fall into different halves of the 32 banks
__host__ __device__ constexpr int gf_row_pitch(int cols) { return cols + ((12 - (cols & 7)) & 7); }

constexpr int GF_MAX_KSP = 8;   // k-steps of the pass: 2 L1 real <= 32, i.e. L1 <= 16
constexpr int GF_MAX_KSP_PASS = 9;   // ... of the pass-only variant: L1 <= 18 (the 17 lattice vectors of a ribbon)
constexpr int GF_WARPS = 8;     // warps of the one persistent CTA per SM (one warp per quad)
// Warps per quad.  With 2, each of two warps takes half of the pass tiles and rotates two of the four pairs: the U
// fragments of a warp are then those of two pairs (64 registers) and twelve warps fit the register file (152 per thread)
// where one warp per quad allows eight; the two meet at a named barrier twice per mode.  Measured: no gain -- 18.4 vs
// 18.3 ms per 96 q on configs[1], 40.6 vs 38.4 ms per 13 q on configs[3], FP64 tensor pipe 70 % busy either way (the
// short DMMA bursts between the staging steps limit it, not the number of warps) -- so one warp per quad stays.
constexpr int GF_WPQ = 1;
constexpr int GF_WARPS_PAIRED = 12;
constexpr int GF_WARPS_PASS = 16;   // ... of the pass-only variant (no U fragments: 128 registers per thread are plenty)
constexpr int GF_MAX_BUF = 4;   // depth of the T2 tile ring

struct GridFusedParams {
  const c128 *T2;        // [L1][slab][ncols], g columns first
  int64_t slab;
  int ncols, L1, cnt;    // cnt: i1 planes of this chunk
  const c128 *P1c;       // [L1][cnt]
  int nquads, ngroups, nbuf;   // quads of four i1 in the chunk, mode groups per cell, depth of the T2 tile ring
  const c128 *Uk, *Ukq;  // relative to the first k of the chunk (k = j*slab + cell)
  const int32_t *kq_idx;
  int nm, nug;           // modes, modes per CTA
  const uint8_t *mask;
  double *g2;            // NULL allowed when the consumer is on: |g|^2 then never leaves the SM
  c128 *gt;              // pass-only variant: g~ [k][gt_stride] relative to the chunk (the g columns first)
  int64_t gt_stride;
  // pass-only variant: nbatch independent problems of this shape, input b at T2 + b * in_bstride ([L1][slab][ncols]),
  // output b at gt + b * out_bstride ([cnt][slab][gt_stride]); "cells" then run over nbatch * slab
  int nbatch;
  int64_t in_bstride, out_bstride;
  // NEXT-4 consumer folded into the epilogue of product 2 (consumer.cu has the formula, reading G18):
  //   Im Sigma_nk += pi w_q / (s sqrt(pi)) sum_{m,nu} |g_mn nu|^2 [(n_nu + f_m) e^{-((e_n - e_m + w_nu)/s)^2} + (n_nu + 1 - f_m) e^{-((e_n - e_m - w_nu)/s)^2}]
  double *cons_out;      // [k][Nb] relative to the chunk, NULL = consumer off
  const double *eps_k;   // [k][Nb] relative to the chunk
  const double *eps_kq;  // [k][Nb] relative to the chunk, or (kq_idx given) eps_k of ALL k, indexed through kq_idx
  const double *omega_q; // [nm] of this q
  const double *w_q;     // weights of the call's q-points or NULL (= 1)
  int64_t iq;
  double mu, kT, sigma;
};

// (per-warp scratch of the consumer: e_n, e_m, f_m of the warp's pairs [pairs][3][NB], then (omega, bose) of the tile's modes)

// embedding entry of a complex number z for fragment coordinates (a = real sub-row, b = real sub-column):
//   [[re, im], [-im, re]]
__device__ __forceinline__ double embed(c128 z, int a, int b) { return a == 0 ? (b ? z.y : z.x) : (b ? z.x : -z.y); }

// Fragments of the embedding of U (or conj U) for the lane (g, t): entry (ks, nt) is +-(one component of U[r][c]),
// r = 2 ks + t/2, c = 4 nt + g/2.  Component and sign depend on the lane only (a = t & 1, b = g & 1):
//   U:       [[re, im], [-im, re]]   component a ^ b, negative where a = 1, b = 0
//   conj U:  [[re, -im], [im, re]]   component a ^ b, negative where a = 0, b = 1
// The loads come first and the sign is applied later (u_frag_sign: an integer XOR on the high word), so that nothing has
// to wait for the loads before the first pass of an item has been issued.
template <int NB>
__device__ __forceinline__ void load_u_frag_raw(const c128 *__restrict__ u, int g, int t,
                                                double (&b)[GF<NB>::KS][GF<NB>::NT]) {
  typedef GF<NB> C;
  const double *ud = reinterpret_cast<const double *>(u) + ((t & 1) ^ (g & 1));
#pragma unroll
  for (int ks = 0; ks < C::KS; ks++)
#pragma unroll
    for (int nt = 0; nt < C::NT; nt++) {
      const int r = 2 * ks + (t >> 1), c = 4 * nt + (g >> 1);
      b[ks][nt] = (r < NB && c < NB) ? ud[(r + NB * c) * 2] : 0.0;
    }
}
template <int NB>
__device__ __forceinline__ void u_frag_sign(bool conj, int g, int t, double (&b)[GF<NB>::KS][GF<NB>::NT]) {
  typedef GF<NB> C;
  const int a = t & 1, bb = g & 1;
  const int flip = (conj ? (a == 0 && bb == 1) : (a == 1 && bb == 0)) ? (int)0x80000000 : 0;
#pragma unroll
  for (int ks = 0; ks < C::KS; ks++)
#pragma unroll
    for (int nt = 0; nt < C::NT; nt++)
      b[ks][nt] = __hiloint2double(__double2hiint(b[ks][nt]) ^ flip, __double2loint(b[ks][nt]));
}
template <int NB>
__device__ __forceinline__ void load_u_frag(const c128 *__restrict__ u, bool conj, int g, int t,
                                            double (&b)[GF<NB>::KS][GF<NB>::NT]) {
  load_u_frag_raw<NB>(u, g, t, b);
  u_frag_sign<NB>(conj, g, t, b);
}

// e^-y for 0 <= y < 64 without the range checks of the library routine: y = k ln 2 + r (Cody-Waite, |r| <= ln 2 / 2),
// e^-r by its Taylor polynomial of degree 12 (remainder 2e-16), 2^-k through the exponent field.
__device__ __forceinline__ double exp_neg(double y) {
  const double k = rint(y * 1.4426950408889634);
  double r = fma(-k, 6.93147180369123816490e-01, y);
  r = -fma(-k, 1.90821492927058770002e-10, r);   // r <- -(y - k ln 2)
  double p = 1.0 / 479001600.0;
  p = fma(p, r, 1.0 / 39916800.0);
  p = fma(p, r, 1.0 / 3628800.0);
  p = fma(p, r, 1.0 / 362880.0);
  p = fma(p, r, 1.0 / 40320.0);
  p = fma(p, r, 1.0 / 5040.0);
  p = fma(p, r, 1.0 / 720.0);
  p = fma(p, r, 1.0 / 120.0);
  p = fma(p, r, 1.0 / 24.0);
  p = fma(p, r, 1.0 / 6.0);
  p = fma(p, r, 0.5);
  p = fma(p, r, 1.0);
  p = fma(p, r, 1.0);
  return p * __hiloint2double((1023 - (int)k) << 20, 0);
}

// The two rotation products of ONE pair and ONE mode.  sG: this pair's g~ of the mode in the staging buffer [c = n' NB + m'],
// sT: this pair's T buffer [n][m'] (pitch SP, padding rows / columns stay zero).
template <int NB>
__device__ __forceinline__ void product1(const double *__restrict__ sG, double *__restrict__ sT, int g, int t,
                                         const double (&b1)[GF<NB>::KS][GF<NB>::NT]) {
  typedef GF<NB> C;
#pragma unroll
  for (int mtr = 0; mtr < C::MTR; mtr++) {
    const int mp = 8 * mtr + g;
    double a[C::KS];
#pragma unroll
    for (int ks = 0; ks < C::KS; ks++) {
      const int np_ = 2 * ks + (t >> 1);
      a[ks] = (mp < NB && np_ < NB) ? sG[(np_ * C::NBP + mp) * 2 + (t & 1)] : 0.0;
    }
    double acc[C::NT][2];
#pragma unroll
    for (int nt = 0; nt < C::NT; nt++) acc[nt][0] = acc[nt][1] = 0.0;
#pragma unroll
    for (int ks = 0; ks < C::KS; ks++)
#pragma unroll
      for (int nt = 0; nt < C::NT; nt++) dmma884(acc[nt][0], acc[nt][1], a[ks], b1[ks][nt]);
    // lane owns T[m' = mp][n = 4 nt + t]  ->  sT[n][m']
    if (mp < NB) {
#pragma unroll
      for (int nt = 0; nt < C::NT; nt++) {
        const int n = 4 * nt + t;
        if (n < NB) *reinterpret_cast<double2 *>(sT + ((size_t)n * C::SP + mp) * 2) = make_double2(acc[nt][0], acc[nt][1]);
      }
    }
  }
}

// cons (may be NULL): this pair's e_n [NB], e_m [NB], f_m [NB]; wb: (omega, bose) of this mode; the contribution of the
// pair and mode to Im Sigma_n is reduced over the four lanes that share a row n and added to cdst[n] by one of them
// (plain read-modify-write: the (pair, n) entries of a tile belong to this warp; atomic when modes are split over tiles)
template <int NB>
__device__ __forceinline__ void product2(const double *__restrict__ sT, double *__restrict__ dst, int g, int t,
                                         const double (&b2)[GF<NB>::KS][GF<NB>::NT], bool store,
                                         const double *__restrict__ cons = nullptr, const double *__restrict__ wb = nullptr,
                                         double *__restrict__ cdst = nullptr, double inv_s = 0.0, double pref = 0.0,
                                         bool atomic = false) {
  typedef GF<NB> C;
#pragma unroll
  for (int mtr = 0; mtr < C::MTR; mtr++) {
    const int n = 8 * mtr + g;
    const double *arow = sT + (size_t)n * C::SP * 2 + t;
    double acc[C::NT][2];
#pragma unroll
    for (int nt = 0; nt < C::NT; nt++) acc[nt][0] = acc[nt][1] = 0.0;
#pragma unroll
    for (int ks = 0; ks < C::KS; ks++) {
      const double a = arow[4 * ks];
#pragma unroll
      for (int nt = 0; nt < C::NT; nt++) dmma884(acc[nt][0], acc[nt][1], a, b2[ks][nt]);
    }
    if (store && dst != nullptr && n < NB) {
#pragma unroll
      for (int nt = 0; nt < C::NT; nt++) {
        const int m = 4 * nt + t;
        if (m < NB) dst[n * NB + m] = acc[nt][0] * acc[nt][0] + acc[nt][1] * acc[nt][1];
      }
    }
    if (cons != nullptr) {
      // Every lane has 2 NT candidate terms (absorption and emission peak of each of its elements); a Gaussian below e^-50
      // of its peak cannot reach the last bit of the sum (same cut as consumer.cu), and few survive.  The exponentials
      // share the FP64 pipe with the DMMAs, so the warp evaluates them one ROUND at a time -- each lane its next surviving
      // candidate -- and stops when no lane has one left (1-2 rounds where a fixed order would take 2 NT).
      const double w = wb[0], bose = wb[1];
      double y[2 * C::NT], cf[2 * C::NT];
      unsigned pend = 0;
#pragma unroll
      for (int nt = 0; nt < C::NT; nt++) {
        const int m = 4 * nt + t;
        const bool on = store && n < NB && m < NB && w > 0.0;
        const int mm = m < NB ? m : 0, nn = n < NB ? n : 0;
        const double de_ = cons[nn] - cons[NB + mm], f = cons[2 * NB + mm];
        const double xa = (de_ + w) * inv_s, xe = (de_ - w) * inv_s;
        const double v = acc[nt][0] * acc[nt][0] + acc[nt][1] * acc[nt][1];
        y[2 * nt] = xa * xa;
        y[2 * nt + 1] = xe * xe;
        cf[2 * nt] = v * (bose + f);
        cf[2 * nt + 1] = v * (bose + 1.0 - f);
        if (on && y[2 * nt] < 50.0) pend |= 1u << (2 * nt);
        if (on && y[2 * nt + 1] < 50.0) pend |= 1u << (2 * nt + 1);
      }
      double sum = 0.0;
      while (__any_sync(0xffffffffu, pend != 0)) {
        const int b = __ffs(pend) - 1;   // -1: this lane has nothing left
        double yy = 0.0, cc = 0.0;
#pragma unroll
        for (int i = 0; i < 2 * C::NT; i++)
          if (b == i) { yy = y[i]; cc = cf[i]; }
        sum = fma(cc, exp_neg(yy), sum);
        pend &= pend - 1;
      }
      sum += __shfl_xor_sync(0xffffffffu, sum, 1);
      sum += __shfl_xor_sync(0xffffffffu, sum, 2);
      if (t == 0 && n < NB && sum != 0.0) {
        if (atomic) atomicAdd(cdst + n, pref * sum);
        else cdst[n] += pref * sum;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// The kernel is PERSISTENT: one CTA of GF_WARPS warps per SM (255 registers per thread: the U fragments of a quad take
// 128).  Work item = (cell, mode group, quad); the items are numbered with the quad fastest, every CTA takes one
// contiguous range of them (equal to within one item) and deals it round-robin to its warps.  The T2 rows of a
// (cell, mode group) tile arrive by bulk TMA in a ring of shared-memory buffers: full[buf] is an mbarrier the copies
// complete on; a buffer is handed back by the last warp that leaves it (shared-memory counter), and that warp issues the
// copies of the tile NBUF places further on.  So the T2 loads, the launch and the tail of a cell overlap the DMMAs of
// the warps that are still at work, which a one-CTA-per-cell grid could not do (half the FP64 pipe idle at ten quads
// per cell).
// KSPMAX: k-steps of the pass the phase fragments are sized for (4: L1 <= 8, 8: L1 <= 16)
// ---------------------------------------------------------------------------------------------------------------
// VAR: 0 = pass + rotation + |g|^2;  1 = the same with the NEXT-4 consumer in the epilogue;  2 = the pass alone, g~ written
// to global memory for rotate_g2.cu (the two-kernel form of 9 <= Nb <= 16: the streaming axis pass spends 4 L1 DFMA per
// output element on the plain FP64 pipe and is bound by it at L1 = 13, the DMMA product is not)
template <int NB, int VAR>
struct GFShape {
  static constexpr bool PASS_ONLY = VAR == 2;
  static constexpr int WPQ = (GF<NB>::UREG && !PASS_ONLY) ? GF_WPQ : 1;       // warps per quad
  static constexpr int NW = PASS_ONLY ? GF_WARPS_PASS : (WPQ == 2 ? GF_WARPS_PAIRED : GF_WARPS);
  static constexpr int PPW = GF<NB>::UREG ? 4 / WPQ : 1;                      // pairs whose U fragments a warp holds
  static constexpr int CPW = GF<NB>::UREG ? PPW : 4;                          // pairs in a warp's consumer table
  // shared memory of one quad group (WPQ warps): g~ staging of the four pairs, then per warp its T buffers
  static constexpr size_t t_bytes = sizeof(c128) * (size_t)PPW * GF<NB>::TROWS * GF<NB>::SP;
  static constexpr size_t g_bytes = sizeof(c128) * 4 * (size_t)GF<NB>::PST;
  __host__ __device__ static constexpr size_t cons_bytes(int nug) { return sizeof(double) * (size_t)((3 * CPW * NB + 2 * nug + 1) & ~1); }
  __host__ __device__ static constexpr size_t group_bytes(int nug) {
    return PASS_ONLY ? 0 : g_bytes + WPQ * (t_bytes + (VAR == 1 ? cons_bytes(nug) : 0));
  }
};

template <int NB, int KSPMAX, int VAR>
__global__ void __launch_bounds__(GFShape<NB, VAR>::NW * 32, 1) grid_fused_kernel(const GridFusedParams p) {
  typedef GF<NB> C;
  typedef GFShape<NB, VAR> S;
  constexpr bool CONS = VAR == 1, PASS_ONLY = VAR == 2;
  constexpr int NW = S::NW, WPQ = S::WPQ, PPW = S::PPW, NQG = NW / WPQ;
  constexpr int NBB = C::NBB;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = lane >> 2, t = lane & 3;
  const int L1 = p.L1, ksp = (L1 + 1) >> 1, L1e = 2 * ksp;
  const int RP = gf_row_pitch(p.nug * NBB);                    // row pitch of a T2 buffer (complex)
  const size_t buf_elems = (size_t)L1e * RP + 8;                // (+ 8 so that the ragged last pass tile stays inside)
  const int64_t E = (int64_t)p.nm * NBB;
  c128 *sT2 = reinterpret_cast<c128 *>(smem_raw);               // [nbuf][L1e][RP]
  unsigned char *wbase = smem_raw + sizeof(c128) * buf_elems * p.nbuf;
  const int qgroup = warp / WPQ, half = warp - qgroup * WPQ;   // quad group of this warp, and which of its WPQ warps it is
  const size_t gstride = S::group_bytes(p.nug);
  const size_t wpart = S::t_bytes + (CONS ? S::cons_bytes(p.nug) : 0);
  double *sG = reinterpret_cast<double *>(wbase + (size_t)qgroup * gstride);       // [4 pairs][PST] complex, shared by the group
  double *sT = reinterpret_cast<double *>(wbase + (size_t)qgroup * gstride + S::g_bytes + (size_t)half * wpart);  // [PPW][TROWS][SP]
  double *sC = sT + PPW * C::TROWS * C::SP * 2;                                    // consumer scratch (CONS only)
  uint64_t *full = reinterpret_cast<uint64_t *>(wbase + (size_t)NQG * gstride);   // [nbuf]
  // the warps of a quad group meet here (a warp alone: __syncwarp)
  auto group_sync = [&]() {
    if (WPQ == 1) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(1 + qgroup), "n"(WPQ * 32) : "memory");
  };
  const double c_inv_s = CONS ? 1.0 / p.sigma : 0.0;
  const double c_pref = CONS ? 3.14159265358979323846 * (p.w_q ? p.w_q[p.iq] : 1.0) * c_inv_s * 0.56418958354775628695 : 0.0;
  const bool c_atomic = p.ngroups > 1;
  int *cnt = reinterpret_cast<int *>(full + GF_MAX_BUF);                                      // [nbuf]

  // ---- this CTA's items and tiles ----
  const int64_t total = p.slab * p.nbatch * p.ngroups * p.nquads;
  const int64_t lo = total * blockIdx.x / gridDim.x, hi = total * (blockIdx.x + 1) / gridDim.x;
  if (lo >= hi) return;
  const int64_t tile_lo = lo / p.nquads;
  const int ntiles = (int)((hi - 1) / p.nquads - tile_lo) + 1;

  auto issue_tile = [&](int tr) {   // one thread: the L1 row copies of tile tile_lo + tr into its ring buffer
    const int64_t tile = tile_lo + tr;
    const int64_t cell = tile / p.ngroups;
    const int nu0 = (int)(tile - cell * p.ngroups) * p.nug;
    const int nuc = p.nm - nu0 < p.nug ? p.nm - nu0 : p.nug;
    const int b = tr % p.nbuf;
    const uint32_t bar = smem_u32(full + b);
    const uint32_t row_bytes = (uint32_t)(sizeof(c128) * nuc * NBB);
    mbar_expect_tx(bar, row_bytes * (uint32_t)L1);
    c128 *dst = sT2 + buf_elems * b;
    for (int n1 = 0; n1 < L1; n1++)
      tma_bulk_g2s(smem_u32(dst + (size_t)n1 * RP),
                   p.T2 + (cell / p.slab) * p.in_bstride + ((int64_t)n1 * p.slab + cell % p.slab) * p.ncols + (int64_t)nu0 * NBB,
                   row_bytes, bar);
  };

  if (threadIdx.x == 0) {
    for (int b = 0; b < p.nbuf; b++) {
      mbar_init(smem_u32(full + b), 1);
      cnt[b] = 0;
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // zero what the copies never write: the padding row n1 = L1 (odd L1) and the tail of every buffer; the T buffers
  for (int b = 0; b < p.nbuf; b++) {
    c128 *dst = sT2 + buf_elems * b;
    for (int i = threadIdx.x; i < RP + 8; i += blockDim.x) {
      if (L1e > L1 && i < RP) dst[(size_t)L1 * RP + i] = make_double2(0.0, 0.0);
      if (i >= RP) dst[(size_t)L1e * RP + (i - RP)] = make_double2(0.0, 0.0);
    }
  }
  if (!PASS_ONLY)
    for (int i = lane; i < PPW * C::TROWS * C::SP * 2; i += 32) sT[i] = 0.0;
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  __syncthreads();
  if (threadIdx.x == 0)
    for (int tr = 0; tr < p.nbuf && tr < ntiles; tr++) issue_tile(tr);

  int held = -1;   // tile (relative) whose buffer this warp is reading
  auto acquire = [&](int tr) { mbar_wait(smem_u32(full + tr % p.nbuf), (uint32_t)((tr / p.nbuf) & 1)); };
  auto release = [&](int tr) {
    __syncwarp();
    if (lane == 0) {
      __threadfence_block();
      const int b = tr % p.nbuf;
      if (atomicAdd(cnt + b, 1) == NW - 1) {   // last warp out: the buffer is free for the tile nbuf places on
        atomicExch(cnt + b, 0);
        if (tr + p.nbuf < ntiles) {
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic reads above, async-proxy writes below
          issue_tile(tr + p.nbuf);
        }
      }
    }
  };
  auto advance_to = [&](int tr) {
    while (held < tr) {
      if (held >= 0) release(held);
      held++;
      acquire(held);
    }
  };
  // pair index of pair jj of an item, and the L2 prefetch of the two U matrices of the four pairs of the NEXT item
  auto prefetch_u = [&](int64_t item) {
    const int64_t tile = item / p.nquads;
    const int quad = (int)(item - tile * p.nquads);
    const int64_t cell = tile / p.ngroups;
    const int jj = lane >> 3, line = lane & 7;    // 4 pairs x 8 lines of 128 bytes cover an 8 x 8 matrix; more lines below
    const int j = 4 * quad + jj;
    if (j < p.cnt) {
      const int64_t k = (int64_t)j * p.slab + cell;
      const char *a = reinterpret_cast<const char *>(p.Uk + k * NBB);
      const char *b = reinterpret_cast<const char *>(p.Ukq + (p.kq_idx ? (int64_t)p.kq_idx[k] : k) * NBB);
      for (int off = line * 128; off < (int)(sizeof(c128) * NBB); off += 8 * 128) {
        asm volatile("prefetch.global.L2 [%0];" ::"l"(a + off));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(b + off));
      }
    }
  };

  // Items have equal length and the two warps that share a scheduler (warp and warp + 4) would walk through them in step:
  // both in the set-up, the staging steps and the epilogue at the same time, the FP64 pipe idle.  The upper four warps
  // start half an item late (about half of the DMMA issue time of an item shared by two warps).
  if (!PASS_ONLY && warp >= 4) {
    const long long wait = (long long)p.nug * (C::MTP * ksp + 8 * C::MTR * C::KS * C::NT) * 16;
    const long long t0 = clock64();
    while (clock64() - t0 < wait) {}
  }
  for (int64_t item = lo + qgroup; item < hi; item += NQG) {
    const int64_t tile = item / p.nquads;
    const int quad = (int)(item - tile * p.nquads);
    const int64_t cell = tile / p.ngroups;
    const int nu0 = (int)(tile - cell * p.ngroups) * p.nug;
    const int nuc = p.nm - nu0 < p.nug ? p.nm - nu0 : p.nug;
    const int j0 = 4 * quad;
    if (!PASS_ONLY && half == 0 && item + NQG < hi) prefetch_u(item + NQG);
    // ---- per pair of the quad: index, validity, energy-window decision ----
    int64_t kc[4];
    bool live[4];
    bool any = false;
#pragma unroll
    for (int jj = 0; jj < 4; jj++) {
      const bool valid = j0 + jj < p.cnt;
      kc[jj] = (int64_t)(valid ? j0 + jj : j0) * p.slab + cell;
      live[jj] = valid && (PASS_ONLY || p.mask == nullptr || p.mask[kc[jj]] != 0);
      if (valid && !live[jj] && p.g2 != nullptr && jj / (4 / WPQ) == half) {   // a skipped pair reports zeros
        double *dz = p.g2 + kc[jj] * E + (int64_t)nu0 * NBB;
        for (int i = lane; i < nuc * NBB; i += 32) dz[i] = 0.0;
      }
      any |= live[jj];
    }
    if (!any) continue;   // (a quad with some pairs skipped is computed whole; only its stores are predicated)
    // the pairs this warp rotates: jj = half * PPW + jo
    int64_t kcw[PPW];
    bool livew[PPW];
#pragma unroll
    for (int jo = 0; jo < PPW; jo++) {
      kcw[jo] = kc[jo];
      livew[jo] = live[jo];
#pragma unroll
      for (int hh = 1; hh < WPQ; hh++)
        if (half == hh) { kcw[jo] = kc[(hh * PPW + jo) & 3]; livew[jo] = live[(hh * PPW + jo) & 3]; }
    }
    if (CONS) {
      // e_n(k), e_m(k+q) and the Fermi factor of the final states for this warp's pairs; (omega, Bose factor) of the modes
      for (int idx = lane; idx < S::CPW * NB; idx += 32) {
        const int jo = idx / NB, i = idx - jo * NB, jj = C::UREG ? half * PPW + jo : jo;
        const int64_t k = (int64_t)(j0 + jj < p.cnt ? j0 + jj : j0) * p.slab + cell;
        const double e2 = (p.kq_idx ? p.eps_kq + (int64_t)p.kq_idx[k] * NB : p.eps_kq + k * NB)[i];
        sC[jo * 3 * NB + i] = p.eps_k[k * NB + i];
        sC[jo * 3 * NB + NB + i] = e2;
        sC[jo * 3 * NB + 2 * NB + i] = 1.0 / (exp((e2 - p.mu) / p.kT) + 1.0);
      }
      for (int nl = lane; nl < nuc; nl += 32) {
        const double w = p.omega_q[nu0 + nl];
        sC[3 * S::CPW * NB + 2 * nl] = w;
        sC[3 * S::CPW * NB + 2 * nl + 1] = w > 0.0 ? 1.0 / expm1(w / p.kT) : 0.0;
      }
    }
    // ---- B' of the pass: 2x2 embedding of the phases p[n1][j] of the four pairs; fragment ks: k-row 4 ks + t, column g ----
    double bp[KSPMAX];
#pragma unroll
    for (int ks = 0; ks < KSPMAX; ks++) {
      const int n1 = 2 * ks + (t >> 1), j = j0 + (g >> 1);
      c128 ph = make_double2(0.0, 0.0);
      if (n1 < L1 && j < p.cnt) ph = p.P1c[(int64_t)n1 * p.cnt + j];
      bp[ks] = embed(ph, t & 1, g & 1);
    }
    // ---- U fragments ----
    double b1[PPW][C::KS][C::NT], b2[PPW][C::KS][C::NT];
    if (C::UREG && !PASS_ONLY) {
#pragma unroll
      for (int jo = 0; jo < PPW; jo++) {
        load_u_frag_raw<NB>(p.Uk + kcw[jo] * NBB, g, t, b1[jo]);
        load_u_frag_raw<NB>(p.Ukq + (p.kq_idx ? (int64_t)p.kq_idx[kcw[jo]] : kcw[jo]) * NBB, g, t, b2[jo]);
      }
    }
    advance_to((int)(tile - tile_lo));
    const c128 *sT2b = sT2 + buf_elems * (held % p.nbuf);
    // ---- pass: g~_j[c] for the four pairs and the NBB columns c of mode nul -> staging buffer [pair][n'][m'] ----
    // (the column tiles of a mode are split between the WPQ warps of the group: warp `half` takes tiles
    //  half * MTW .. half * MTW + MTW - 1)
    constexpr int MTW = (C::MTP + WPQ - 1) / WPQ;
    auto pass = [&](int nul, auto exact) {
      const double *tsrc = reinterpret_cast<const double *>(sT2b + (size_t)(t >> 1) * RP + nul * NBB + g) + (t & 1);
#pragma unroll
      for (int mt0 = 0; mt0 < MTW; mt0 += 8) {
        const int mtb = half * MTW + mt0;   // first tile of this block of (up to) eight
        double acc[8][2];
#pragma unroll
        for (int i = 0; i < 8; i++) acc[i][0] = acc[i][1] = 0.0;
#pragma unroll
        for (int ks = 0; ks < KSPMAX; ks++) {
          if (decltype(exact)::value || ks < ksp) {
#pragma unroll
            for (int i = 0; i < 8; i++) {
              if (mt0 + i < MTW && (WPQ == 1 || mtb + i < C::MTP)) {
                const double a = tsrc[((size_t)2 * ks * RP + 8 * (mtb + i)) * 2];
                dmma884(acc[i][0], acc[i][1], a, bp[ks]);
              }
            }
          }
        }
#pragma unroll
        for (int i = 0; i < 8; i++) {
          const int cl = 8 * (mtb + i) + g;
          if (mt0 + i < MTW && mtb + i < C::MTP && cl < NBB) {
            if (PASS_ONLY) {   // lane (g, t): g~ of pair t, column cl -- eight lanes write 128 contiguous bytes
              if (j0 + t < p.cnt)
                p.gt[(cell / p.slab) * p.out_bstride + ((int64_t)(j0 + t) * p.slab + cell % p.slab) * p.gt_stride +
                     (int64_t)(nu0 + nul) * NBB + cl] = make_double2(acc[i][0], acc[i][1]);
            } else {
              *reinterpret_cast<double2 *>(sG + ((size_t)t * C::PST + (cl / NB) * C::NBP + cl % NB) * 2) =
                  make_double2(acc[i][0], acc[i][1]);
            }
          }
        }
      }
    };
    if (PASS_ONLY) {
      for (int nul = 0; nul < nuc; nul++) {
        if (ksp == KSPMAX) pass(nul, std::true_type());
        else pass(nul, std::false_type());
      }
      continue;
    }
    const bool exact = ksp == KSPMAX;   // no k-step to skip: the common case, without the branches
    if (exact) pass(0, std::true_type());
    else pass(0, std::false_type());
    if (C::UREG) {
      // the first pass is on its way: now wait for the U loads and give the fragments their signs
#pragma unroll
      for (int jo = 0; jo < PPW; jo++) {
        u_frag_sign<NB>(false, g, t, b1[jo]);
        u_frag_sign<NB>(true, g, t, b2[jo]);
      }
    }
    group_sync();   // g~ of mode 0 is complete (all tiles, from every warp of the group)
    for (int nul = 0; nul < nuc; nul++) {
      if (C::UREG) {
        // ---- product 1 of this warp's pairs (no branch inside: independent DMMA chains) ----
#pragma unroll
        for (int jo = 0; jo < PPW; jo++)
          product1<NB>(sG + (size_t)(half * PPW + jo) * C::PST * 2, sT + (size_t)jo * C::TROWS * C::SP * 2, g, t, b1[jo]);
        group_sync();   // T is written; every warp of the group has read g~ of this mode
        // ---- product 2 and |.|^2 of this mode, and in the same stretch of code the pass of the NEXT mode: the staging
        //      buffer of g~ is free once product 1 has read it, and the two are independent DMMA chains ----
#pragma unroll
        for (int jo = 0; jo < PPW; jo++)
          product2<NB>(sT + (size_t)jo * C::TROWS * C::SP * 2,
                       p.g2 ? p.g2 + kcw[jo] * E + (int64_t)(nu0 + nul) * NBB : nullptr, g, t, b2[jo], livew[jo],
                       CONS ? sC + jo * 3 * NB : nullptr, sC + 3 * S::CPW * NB + 2 * nul,
                       CONS ? p.cons_out + kcw[jo] * NB : nullptr, c_inv_s, c_pref, c_atomic);
        if (nul + 1 < nuc) {
          if (exact) pass(nul + 1, std::true_type());
          else pass(nul + 1, std::false_type());
        }
        group_sync();
      } else {
        // Nb > 8: the fragments of one U matrix at a time (36 registers at Nb = 11), pair by pair
#pragma unroll 1
        for (int jj = 0; jj < 4; jj++) {
          if (j0 + jj >= p.cnt) break;
          const int64_t k = (int64_t)(j0 + jj) * p.slab + cell;
          if (p.mask != nullptr && p.mask[k] == 0) continue;
          load_u_frag<NB>(p.Uk + k * NBB, false, g, t, b1[0]);
          product1<NB>(sG + (size_t)jj * C::PST * 2, sT, g, t, b1[0]);
          __syncwarp();
          load_u_frag<NB>(p.Ukq + (p.kq_idx ? (int64_t)p.kq_idx[k] : k) * NBB, true, g, t, b2[0]);
          product2<NB>(sT, p.g2 ? p.g2 + k * E + (int64_t)(nu0 + nul) * NBB : nullptr, g, t, b2[0], true,
                       CONS ? sC + jj * 3 * NB : nullptr, sC + 12 * NB + 2 * nul, CONS ? p.cons_out + k * NB : nullptr, c_inv_s,
                       c_pref, c_atomic);
          __syncwarp();
        }
        if (nul + 1 < nuc) {
          if (exact) pass(nul + 1, std::true_type());
          else pass(nul + 1, std::false_type());
        }
        __syncwarp();
      }
    }
  }
  // hand back every remaining tile of the CTA (a warp may have had no item in the last ones)
  advance_to(ntiles - 1);
  release(held);
}

// Modes per tile, ring depth and shared memory: all modes in one tile when a ring of two such tiles fits beside the
// staging buffers (the U fragments are then loaded once per pair), else the largest mode group that does.
template <int NB>
static bool gf_plan(int nm, int L1, int var, int *nug_out, int *nbuf_out, size_t *smem_out) {
  typedef GF<NB> C;
  if (L1 < 1 || L1 > 2 * (var == 2 ? GF_MAX_KSP_PASS : GF_MAX_KSP) || nm < 1) return false;
  const int L1e = 2 * ((L1 + 1) / 2);
  const size_t limit = (size_t)225 * 1024;
  // bytes of the shared-memory plan with n modes per group: (everything but the T2 ring, one T2 buffer).  Both grow with n
  // (gf_row_pitch is the next number = 4 mod 8), so the largest n that fits is found by bisection -- nm is E / 64 = 166,000
  // on configs[4]'s pass-only launches, and this runs on every launch.
  auto bytes_of = [&](int n, size_t *fixed_out) {
    const size_t groups_bytes = var == 2 ? 0
                                : var == 1 ? (GFShape<NB, 1>::NW / GFShape<NB, 1>::WPQ) * GFShape<NB, 1>::group_bytes(n)
                                           : (GFShape<NB, 0>::NW / GFShape<NB, 0>::WPQ) * GFShape<NB, 0>::group_bytes(n);
    *fixed_out = groups_bytes + GF_MAX_BUF * (sizeof(uint64_t) + sizeof(int)) + 16;
    return sizeof(c128) * ((size_t)L1e * gf_row_pitch(n * C::NBB) + 8);
  };
  for (int want_buf = 2; want_buf >= 1; want_buf--) {
    auto fits = [&](int n) {
      size_t fixed = 0;
      const size_t per_buf = bytes_of(n, &fixed);
      return fixed + want_buf * per_buf <= limit;
    };
    if (!fits(1)) continue;
    int lo = 1, hi = nm;   // largest n in [1, nm] that fits
    while (lo < hi) {
      const int mid = lo + (hi - lo + 1) / 2;
      if (fits(mid)) lo = mid;
      else hi = mid - 1;
    }
    {
      int n = lo;
      size_t fixed = 0;
      bytes_of(n, &fixed);
      // equal mode groups (9 modes that fit four at a time go 3 + 3 + 3, not 4 + 4 + 1: the items are dealt by count)
      const int groups = (nm + n - 1) / n;
      n = (nm + groups - 1) / groups;
      const size_t per_buf2 = sizeof(c128) * ((size_t)L1e * gf_row_pitch(n * C::NBB) + 8);
      int nbuf = (int)((limit - fixed) / per_buf2);
      if (nbuf > GF_MAX_BUF) nbuf = GF_MAX_BUF;
      *smem_out = fixed + nbuf * per_buf2;
      *nug_out = n;
      *nbuf_out = nbuf;
      return true;
    }
  }
  return false;
}

template <int NB>
static cudaError_t launch_gf(const GridFusedParams &p0, int num_sms, cudaStream_t st) {
  GridFusedParams p = p0;
  size_t smem = 0;
  const int var = p.gt != nullptr ? 2 : (p.cons_out != nullptr ? 1 : 0);
  if (!gf_plan<NB>(p.nm, p.L1, var, &p.nug, &p.nbuf, &smem)) return cudaErrorInvalidConfiguration;
  p.ngroups = (int)ceil_div(p.nm, p.nug);
  p.nquads = (p.cnt + 3) / 4;
  const int64_t total = p.slab * p.nbatch * p.ngroups * p.nquads;
  const int nw = var == 2 ? GFShape<NB, 2>::NW : GFShape<NB, 0>::NW;
  const int64_t want = ceil_div(total, nw / GFShape<NB, 0>::WPQ);
  const unsigned grid = (unsigned)(want < num_sms ? want : num_sms);
#define EPW_GF_LAUNCH(KSP_, CONS_)                                                                                    \
  do {                                                                                                                \
    cudaError_t e = cudaFuncSetAttribute(grid_fused_kernel<NB, KSP_, CONS_>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                         (int)smem);                                                                  \
    if (e != cudaSuccess) return e;                                                                                   \
    grid_fused_kernel<NB, KSP_, CONS_><<<grid, nw * 32, smem, st>>>(p);                                         \
  } while (0)
  if (p.L1 <= 8) {
    if (var == 2) EPW_GF_LAUNCH(4, 2);
    else if (var == 1) EPW_GF_LAUNCH(4, 1);
    else EPW_GF_LAUNCH(4, 0);
  } else if (p.L1 > 2 * GF_MAX_KSP) {
    EPW_GF_LAUNCH(9, 2);   // pass-only (gf_plan admits no other variant at this L1)
  } else {
    if (var == 2) EPW_GF_LAUNCH(8, 2);
    else if (var == 1) EPW_GF_LAUNCH(8, 1);
    else EPW_GF_LAUNCH(8, 0);
  }
#undef EPW_GF_LAUNCH
  return cudaGetLastError();
}

}  // namespace epw
