// grid_rotate_g2.cu -- uniform-grid path, small Nb: the LAST axis pass of S2 fused with S4b and |g|^2, so that
// g~(k,q) never goes to HBM.
//
//   g~_{m'n' nu}(k,q) = sum_{n1} e^{2 pi i (i1+s1) n1 / N1} T2[n1][(i2,i3)][nu,n',m']      (last axis of the factorised
//                                                         Re -> k sum, re_to_k_grid.cu; Eq. 10)
//   g_{mn nu}(k,q)    = sum_{m'n'} conj(U_{k+q}[m',m]) g~_{m'n' nu} U_k[n',n],   out = |g_{mn nu}|^2   (
//                                                         BASELINE.json north_star stage 4; reading G4)
// In the unfused grid path the last pass writes g~ (16 Nb^2 Nm bytes per pair) and rotate_g2.cu reads it back: that
// round trip is the largest HBM stream of the step once S2 is factorised.  Here one CTA owns one (i2,i3) cell of the
// grid (and a group of modes nu): it loads the L1 rows T2[.][cell][group] into shared memory ONCE (T2 is L2-resident:
// 16 ncols L1 N2 N3 bytes), and its warps walk along i1; for each k = (i1, cell) a warp
//   1. forms the A fragments of product 1 directly in registers: lane (g,t) needs one real component of
//      g~[nu][n' = 2ks + t/2][m' = g], a sum of L1 complex products p[n1] * T2s[n1][..] (2 DFMA each, operands by LDS.128);
//   2. runs the two small products of rotate_g2.cu on the FP64 tensor path (mma.sync.m8n8k4.f64, SASS DMMA), T through a
//      per-warp shared-memory staging buffer, U_k / conj(U_{k+q}) embedded in registers;
//   3. writes |.|^2.
// (lane (g,t) needs Re or Im of each product, i.e. c0 v.x + c1 v.y with (c0,c1) = (Re p, -Im p) or (Im p, Re p).)
// HBM traffic per pair: 32 Nb^2 (the two U) + 8 Nb^2 Nm (output) bytes instead of 16 Nb^2 Nm (g~ written) +
// 16 Nb^2 Nm (read) + the same.  FP64 work per pair: 8 L1 Nb^2 Nm (pass) + 16 Nb^3 Nm (rotation) flops.
#include "common.cuh"
#include "dmma_pipe.cuh"

namespace epw {

__host__ __device__ constexpr int grot_pitch(int nb) { return nb + ((6 - (nb & 3)) & 3); }  // = 2 (mod 4), >= nb
// Row pitch of the T2 rows (nu, n') in shared memory.  A quarter-warp of the pass reads rows n' = 2ks, 2ks+1 at
// m' = 2j, 2j+1: a pitch = 2 (mod 4) complex puts the four 16-byte words in different banks.  For Nb = 8 the same is
// achieved without padding by swapping the two halves of every odd row (m' ^ 4).
__host__ __device__ constexpr int grot_t2_pitch(int nb) { return nb == 8 ? 8 : grot_pitch(nb); }
template <int NB>
__device__ __forceinline__ int grot_t2_pos(int np_, int mp) { return NB == 8 ? (mp ^ ((np_ & 1) << 2)) : mp; }

template <int NB, int W, int MINB>
__global__ void __launch_bounds__(W * 32, MINB)
    grid_rotate_g2_kernel(const c128 *__restrict__ T2, int64_t slab, int ncols, int L1, const c128 *__restrict__ P1c,
                          int cnt, int i1_per_cta, const c128 *__restrict__ Uk, const c128 *__restrict__ Ukq,
                          const int32_t *__restrict__ kq_idx, int nm, int nug, const uint8_t *__restrict__ mask,
                          double *__restrict__ g2) {
  constexpr int KS = (2 * NB + 3) / 4;  // k-steps of 4 real
  constexpr int NT = (2 * NB + 7) / 8;  // column tiles of 8 real
  constexpr int SP = grot_pitch(NB);
  constexpr int NBB = NB * NB;
  static_assert(2 * KS <= SP, "T pitch must cover the padded K range");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = lane >> 2, t = lane & 3, comp = t & 1;
  const int64_t cell = blockIdx.x;
  const int nu0 = blockIdx.y * nug;
  const int nuc = nm - nu0 < nug ? nm - nu0 : nug;
  const int rows = nuc * NB;
  const int MT = (rows + 7) >> 3;
  const int MTmax = (nug * NB + 7) >> 3;
  constexpr int SPT = grot_t2_pitch(NB);
  const int Egmax = nug * NB * SPT;  // per-n1 stride of sT2: rows (nu, n') of SPT complex, conflict-free LDS.128
  const int64_t E = (int64_t)nm * NBB;
  c128 *sT2 = reinterpret_cast<c128 *>(smem_raw);                         // [L1][Egmax]
  c128 *sP = sT2 + (size_t)L1 * Egmax + (size_t)warp * L1;                // [W][L1], this warp's phases
  double *sT = reinterpret_cast<double *>(sT2 + (size_t)L1 * Egmax + (size_t)W * L1) +
               (size_t)warp * MTmax * 8 * SP * 2;                         // [W][MTmax*8][SP] complex

  // ---- the L1 rows of T2 this CTA needs, and zeroed staging buffers (padding must stay finite) ----
  {
    const int Eg = nuc * NBB;
    for (int idx = threadIdx.x; idx < L1 * Eg; idx += W * 32) {
      const int n1 = idx / Eg, c = idx - n1 * Eg;
      const int rw = c / NB, mp = c - rw * NB;   // rw = (nu, n')
      sT2[(size_t)n1 * Egmax + rw * SPT + grot_t2_pos<NB>(rw % NB, mp)] = T2[((int64_t)n1 * slab + cell) * ncols + (int64_t)nu0 * NBB + c];
    }
    double *z = reinterpret_cast<double *>(sT2 + (size_t)L1 * Egmax + (size_t)W * L1);
    for (int i = threadIdx.x; i < W * MTmax * 8 * SP * 2; i += W * 32) z[i] = 0.0;
  }
  __syncthreads();

  const int j_lo = blockIdx.z * i1_per_cta;
  const int j_hi = j_lo + i1_per_cta < cnt ? j_lo + i1_per_cta : cnt;
  for (int j = j_lo + warp; j < j_hi; j += W) {
    const int64_t kc = (int64_t)j * slab + cell;   // k index relative to the chunk
    if (mask != nullptr && mask[kc] == 0) {
      // energy-window pre-screening: a skipped pair reports zeros and costs no arithmetic
      double *dz = g2 + kc * E + (int64_t)nu0 * NBB;
      for (int i = lane; i < rows * NB; i += 32) dz[i] = 0.0;
      continue;
    }
    if (lane < L1) sP[lane] = P1c[(int64_t)lane * cnt + j];
    // ---- B' = embedding of Uk (product 1); fragment (ks, nt): k-row 4 ks + t, column 8 nt + g.  For Nb > 8 the
    //      embedding B'' of conj(Ukq) is built only after product 1 (its lines are prefetched into L1 here), which
    //      keeps one fragment set live at a time and lets 12 warps share the SM instead of 8. ----
    constexpr bool LATE_B2 = NB > 8;
    const c128 *uk = Uk + kc * NBB;
    const c128 *ukq = Ukq + (kq_idx ? (int64_t)kq_idx[kc] : kc) * NBB;
    double b1[KS][NT], b2[KS][NT];
    if (LATE_B2) {
      if (lane * 8 < NBB) asm volatile("prefetch.global.L1 [%0];" ::"l"(ukq + lane * 8));
    }
#pragma unroll
    for (int ks = 0; ks < KS; ks++)
#pragma unroll
      for (int nt = 0; nt < NT; nt++) {
        const int r = 2 * ks + (t >> 1), a = t & 1;   // complex row (n' or m'), real sub-row
        const int c = 4 * nt + (g >> 1), b = g & 1;   // complex column (n or m), real sub-column
        c128 x = make_double2(0.0, 0.0), y = make_double2(0.0, 0.0);
        if (r < NB && c < NB) {
          x = uk[r + NB * c];
          if (!LATE_B2) y = ukq[r + NB * c];
        }
        y.y = -y.y;  // conj(Ukq)
        b1[ks][nt] = a == 0 ? (b ? x.y : x.x) : (b ? x.x : -x.y);
        if (!LATE_B2) b2[ks][nt] = a == 0 ? (b ? y.y : y.x) : (b ? y.x : -y.y);
      }
    __syncwarp();
    // ---- last axis pass + product 1: T[(nu,m')][n] = sum_n' g~[nu][n'][m'] Uk[n'][n] ----
    for (int mt = 0; mt < MT; mt++) {
      const int row = 8 * mt + g;
      const bool rv = row < rows;
      const int nu = row / NB, mp = row - nu * NB;
      double a[KS];
#pragma unroll
      for (int ks = 0; ks < KS; ks++) a[ks] = 0.0;
      const c128 *tsrc = sT2 + (size_t)nu * NB * SPT;
      for (int n1 = 0; n1 < L1; n1++) {
        // this lane needs Re (comp = 0) or Im (comp = 1) of p * v:  c0 v.x + c1 v.y  with (c0,c1) = (pr,-pi) or (pi,pr)
        const c128 p = sP[n1];
        const double c0 = comp ? p.y : p.x, c1 = comp ? p.x : -p.y;
#pragma unroll
        for (int ks = 0; ks < KS; ks++) {
          const int np_ = 2 * ks + (t >> 1);
          if (rv && np_ < NB) {
            const c128 v = tsrc[(size_t)n1 * Egmax + np_ * SPT + grot_t2_pos<NB>(np_, mp)];
            a[ks] = fma(c0, v.x, fma(c1, v.y, a[ks]));
          }
        }
      }
      double acc[NT][2];
#pragma unroll
      for (int nt = 0; nt < NT; nt++) acc[nt][0] = acc[nt][1] = 0.0;
#pragma unroll
      for (int ks = 0; ks < KS; ks++)
#pragma unroll
        for (int nt = 0; nt < NT; nt++) dmma884(acc[nt][0], acc[nt][1], a[ks], b1[ks][nt]);
      // thread owns T_nu[m' = mp][n = 4 nt + t]  ->  sT[(nu, n)][m']
      if (rv) {
#pragma unroll
        for (int nt = 0; nt < NT; nt++) {
          const int n = 4 * nt + t;
          if (n < NB)
            *reinterpret_cast<double2 *>(sT + ((size_t)(nu * NB + n) * SP + mp) * 2) = make_double2(acc[nt][0], acc[nt][1]);
        }
      }
    }
    __syncwarp();
    if (LATE_B2) {
#pragma unroll
      for (int ks = 0; ks < KS; ks++)
#pragma unroll
        for (int nt = 0; nt < NT; nt++) {
          const int r = 2 * ks + (t >> 1), a = t & 1;
          const int c = 4 * nt + (g >> 1), b = g & 1;
          c128 y = make_double2(0.0, 0.0);
          if (r < NB && c < NB) y = ukq[r + NB * c];
          y.y = -y.y;  // conj(Ukq)
          b2[ks][nt] = a == 0 ? (b ? y.y : y.x) : (b ? y.x : -y.y);
        }
    }
    // ---- product 2: |sum_m' T[(nu,n)][m'] conj(Ukq[m'][m])|^2 ----
    double *dst = g2 + kc * E + (int64_t)nu0 * NBB;
    for (int mt = 0; mt < MT; mt++) {
      const int row = 8 * mt + g;
      const double *arow = sT + (size_t)row * SP * 2 + t;
      double acc[NT][2];
#pragma unroll
      for (int nt = 0; nt < NT; nt++) acc[nt][0] = acc[nt][1] = 0.0;
#pragma unroll
      for (int ks = 0; ks < KS; ks++) {
        const double a = arow[4 * ks];
#pragma unroll
        for (int nt = 0; nt < NT; nt++) dmma884(acc[nt][0], acc[nt][1], a, b2[ks][nt]);
      }
      if (row < rows) {
#pragma unroll
        for (int nt = 0; nt < NT; nt++) {
          const int m = 4 * nt + t;
          if (m < NB) dst[(int64_t)row * NB + m] = acc[nt][0] * acc[nt][0] + acc[nt][1] * acc[nt][1];
        }
      }
    }
    __syncwarp();
  }
}

template <int NB, int W, int MINB>
static cudaError_t launch_grot(const c128 *T2, int64_t slab, int ncols, int L1, const c128 *P1c, int cnt, const c128 *Uk,
                               const c128 *Ukq, const int32_t *kq_idx, int nm, int num_sms, const uint8_t *mask, double *g2,
                               cudaStream_t st) {
  if (L1 > 32) return cudaErrorInvalidConfiguration;
  // modes per CTA: as many as keep (T2 rows + W staging buffers + phases) within ~100 KB, i.e. two CTAs per SM
  const size_t budget = MINB == 2 ? ((size_t)110 << 10) : ((size_t)220 << 10);
  int nug = 0;
  size_t smem = 0;
  for (int n = nm; n >= 1; n--) {
    const size_t MTmax = ((size_t)n * NB + 7) / 8;
    const size_t need = sizeof(c128) * ((size_t)L1 * n * NB * grot_t2_pitch(NB) + (size_t)W * L1 + (size_t)W * MTmax * 8 * grot_pitch(NB));
    if (need <= budget) { nug = n; smem = need; break; }
  }
  if (nug == 0) return cudaErrorInvalidConfiguration;
  cudaError_t e = cudaFuncSetAttribute(grid_rotate_g2_kernel<NB, W, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  const int ngroups = (nm + nug - 1) / nug;
  // split the i1 walk so that the grid has a few waves of (2 CTAs per SM)
  const int64_t base = slab * ngroups;
  int64_t nsplit = ceil_div((int64_t)8 * num_sms, base);
  const int64_t max_split = ceil_div(cnt, W);
  if (nsplit > max_split) nsplit = max_split;
  if (nsplit < 1) nsplit = 1;
  const int i1_per_cta = (int)(ceil_div(ceil_div(cnt, nsplit), W) * W);
  nsplit = ceil_div(cnt, i1_per_cta);
  if (slab > 2147483647LL || nsplit > 65535) return cudaErrorInvalidConfiguration;
  dim3 grid((unsigned)slab, (unsigned)ngroups, (unsigned)nsplit);
  grid_rotate_g2_kernel<NB, W, MINB><<<grid, W * 32, smem, st>>>(T2, slab, ncols, L1, P1c, cnt, i1_per_cta, Uk, Ukq, kq_idx, nm,
                                                          nug, mask, g2);
  return cudaGetLastError();
}

bool grid_rotate_g2_supported(int nb, int nm, int L1) {
  if (nb < 1 || nb > 16 || L1 > 32) return false;
  const int W = nb <= 8 ? 8 : 12;
  const size_t need = sizeof(c128) * ((size_t)L1 * nb * grot_t2_pitch(nb) + (size_t)W * L1 + (size_t)W * (((size_t)nb + 7) / 8) * 8 * grot_pitch(nb));
  (void)nm;
  return need <= (nb <= 8 ? ((size_t)110 << 10) : ((size_t)220 << 10));
}

// T2 c128 [L1][slab][ncols] (the g columns are the first Nb^2 Nm of each row); P1c c128 [L1][cnt]: phases of the cnt
// i1 planes of this chunk; Uk, Ukq, kq_idx, g2 are relative to the first k of the chunk (k = j*slab + cell).
cudaError_t launch_grid_rotate_g2(const c128 *T2, int64_t slab, int ncols, int L1, const c128 *P1c, int cnt,
                                  const c128 *Uk, const c128 *Ukq, const int32_t *kq_idx, int nb, int nm, int num_sms,
                                  const uint8_t *mask, double *g2, cudaStream_t st) {
  if (slab <= 0 || cnt <= 0) return cudaSuccess;
  switch (nb) {
#define EPW_GROT_CASE(NB_, W_) \
  case NB_: return launch_grot<NB_, W_, (NB_ <= 8 ? 2 : 1)>(T2, slab, ncols, L1, P1c, cnt, Uk, Ukq, kq_idx, nm, num_sms, mask, g2, st);
    EPW_GROT_CASE(1, 8) EPW_GROT_CASE(2, 8) EPW_GROT_CASE(3, 8) EPW_GROT_CASE(4, 8) EPW_GROT_CASE(5, 8)
    EPW_GROT_CASE(6, 8) EPW_GROT_CASE(7, 8) EPW_GROT_CASE(8, 8) EPW_GROT_CASE(9, 12) EPW_GROT_CASE(10, 12)
    EPW_GROT_CASE(11, 12) EPW_GROT_CASE(12, 12) EPW_GROT_CASE(13, 12) EPW_GROT_CASE(14, 12) EPW_GROT_CASE(15, 12)
    EPW_GROT_CASE(16, 12)
#undef EPW_GROT_CASE
    default: return cudaErrorInvalidConfiguration;
  }
}

}  // namespace epw
