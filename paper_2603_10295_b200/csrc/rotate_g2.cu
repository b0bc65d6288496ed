// rotate_g2.cu -- S4b: band rotation and |g|^2 (Eq. 10: U_{mm'k+q} ... U*_{nn'k}; with paper-U = V^dagger,
// V the eigenvector columns, reading G4):
//     g_{mn nu}(k,q) = sum_{m'n'} conj(Ukq[m',m]) g~_{m'n' nu}(k,q) Uk[n',n],     out = |g_{mn nu}|^2.
// The mode rotation and the 1/sqrt(2 omega) amplitude were already applied to g(Re,q) (pack.cu), so g~ arrives in
// the mode basis.  Two successive small matrix products per mode ("successive multiplication"):
//     T[nu][n][m'] = sum_n' g~[nu][n'][m'] Uk[n'][n]          then      g[nu][n][m] = sum_m' T[nu][n][m'] conj(Ukq[m'][m]).
//
// Small-Nb kernel (Nb <= 16): both products run on the FP64 tensor path (mma.sync.m8n8k4.f64, SASS DMMA) -- the same
// FP64 pipe as plain DFMA, but one fragment register feeds 8 FMAs per lane, which removes the shared-memory operand
// traffic that bound the scalar version (short_scoreboard stalls, profiles/r01b_full_summary.md).
//   product 1:  rows (nu,m') [Nm*Nb, tiles of 8]  x  K = n' (2 Nb real)  x  columns n (2 Nb real)
//               A' fragments = re/im of g~ straight from global memory (8 consecutive m' = 128 contiguous bytes),
//               B' fragments = 2x2 real embedding of Uk, built once per pair in registers;
//   T goes through shared memory [nu][n][m'] (row pitch = 2 mod 4 complex: conflict-free STS.128 and LDS.64);
//   product 2:  rows (nu,n)  x  K = m'  x  columns m,  B'' = embedding of conj(Ukq);  epilogue re^2 + im^2 -> g2.
// WPP warps share one pair (its row tiles are dealt round-robin); a CTA of 4 warps works on 4 / WPP pairs at a time.
// Work: 16 Nb^3 Nm flops per pair; reads 16 (Nb^2 Nm + 2 Nb^2) bytes (L2 / HBM), writes 8 Nb^2 Nm bytes per pair.
#include "common.cuh"
#include "dmma_pipe.cuh"

namespace epw {

constexpr int ROT_WARPS = 4;
constexpr int ROT_THREADS = ROT_WARPS * 32;

// shared-memory row pitch of T in complex elements: >= NB and = 2 (mod 4)
__host__ __device__ constexpr int rot_pitch(int nb) { return nb + ((6 - (nb & 3)) & 3); }

template <int NB, int WPP>
__global__ void __launch_bounds__(ROT_THREADS)
    rotate_g2_dmma_kernel(const c128 *__restrict__ gt, int64_t stride_gt, const c128 *__restrict__ Uk,
                          const c128 *__restrict__ Ukq, const int32_t *__restrict__ kq_idx, int nm, int64_t nk,
                          const uint8_t *__restrict__ mask, double *__restrict__ g2) {
  constexpr int KS = (2 * NB + 3) / 4;  // k-steps of 4 real
  constexpr int NT = (2 * NB + 7) / 8;  // column tiles of 8 real
  constexpr int SP = rot_pitch(NB);
  constexpr int PPC = ROT_WARPS / WPP;  // pairs in flight per CTA
  static_assert(2 * KS <= SP, "T pitch must cover the padded K range");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = lane >> 2, t = lane & 3;
  const int slot = warp / WPP, sub = warp - slot * WPP;
  const int rows = nm * NB;               // rows of either product
  const int MT = (rows + 7) >> 3;
  double *sT = reinterpret_cast<double *>(smem_raw) + (size_t)slot * MT * 8 * SP * 2;  // [MT*8 rows][SP] complex

  // zero the staging buffers once: padded K columns and padded rows must stay finite (they meet zero B'' entries)
  for (int i = threadIdx.x; i < PPC * MT * 8 * SP * 2; i += ROT_THREADS) reinterpret_cast<double *>(smem_raw)[i] = 0.0;
  __syncthreads();

  const int64_t npass = (nk + (int64_t)gridDim.x * PPC - 1) / ((int64_t)gridDim.x * PPC);
  for (int64_t pass = 0; pass < npass; pass++) {
    const int64_t ik = (pass * gridDim.x + blockIdx.x) * PPC + slot;
    const bool have = ik < nk;
    const int64_t ikc = have ? ik : 0;
    // energy-window pre-screening: a skipped pair reports zeros and costs no arithmetic.  The decision is
    // uniform over the WPP warps of a pair; with WPP > 1 every warp still takes the two block-wide barriers below.
    const bool skip = mask != nullptr && have && mask[ikc] == 0;
    if (skip) {
      double *dz = g2 + ikc * (int64_t)rows * NB;
      for (int i = sub * 32 + lane; i < rows * NB; i += WPP * 32) dz[i] = 0.0;
    }
    if (skip && WPP == 1) continue;
    // ---- B' = embedding of Uk, B'' = embedding of conj(Ukq); fragment (ks, nt): k-row 4 ks + t, column 8 nt + g ----
    double b1[KS][NT], b2[KS][NT];
    {
      const c128 *uk = Uk + ikc * (NB * NB);
      const c128 *ukq = Ukq + (kq_idx ? (int64_t)kq_idx[ikc] : ikc) * (NB * NB);
#pragma unroll
      for (int ks = 0; ks < KS; ks++)
#pragma unroll
        for (int nt = 0; nt < NT; nt++) {
          const int r = 2 * ks + (t >> 1), a = t & 1;   // complex row (n' or m'), real sub-row
          const int c = 4 * nt + (g >> 1), b = g & 1;   // complex column (n or m), real sub-column
          c128 x = make_double2(0.0, 0.0), y = make_double2(0.0, 0.0);
          if (r < NB && c < NB) {
            x = uk[r + NB * c];
            y = ukq[r + NB * c];
          }
          y.y = -y.y;  // conj(Ukq)
          b1[ks][nt] = a == 0 ? (b ? x.y : x.x) : (b ? x.x : -x.y);
          b2[ks][nt] = a == 0 ? (b ? y.y : y.x) : (b ? y.x : -y.y);
        }
    }
    // ---- product 1: T[(nu,m')][n] ----
    const double *gsrc = reinterpret_cast<const double *>(gt + ikc * stride_gt);
    // A' fragments of tile mt: lane (g,t) holds one real component of g~[nu][n' = 2ks + t/2][m'] for row (nu,m') = 8 mt + g.
    // The fragments of the NEXT tile are requested before the DMMAs of the current one (software pipeline): with loads
    // issued only at their point of use a warp had 4 x 256 bytes in flight and the kernel ran at half the HBM rate.
    auto load_a = [&](int mt, double (&dst)[KS]) {
      const int row = 8 * mt + g;
      const bool rv = row < rows;
      const int nu = row / NB, mp = row - nu * NB;
#pragma unroll
      for (int ks = 0; ks < KS; ks++) {
        const int np_ = 2 * ks + (t >> 1);
        dst[ks] = (rv && np_ < NB) ? gsrc[(((int64_t)nu * NB + np_) * NB + mp) * 2 + (t & 1)] : 0.0;
      }
    };
    // (only when one warp owns the pair, i.e. small Nb: for Nb > 8 the extra registers cost more occupancy than the
    // pipeline gains)
    constexpr bool PIPE = WPP == 1;
    double a_next[KS];
    if (PIPE && !skip && sub < MT) load_a(sub, a_next);
    for (int mt = sub; mt < (skip ? 0 : MT); mt += WPP) {
      const int row = 8 * mt + g;
      const bool rv = row < rows;
      const int nu = row / NB, mp = row - nu * NB;
      double a[KS];
      if (PIPE) {
#pragma unroll
        for (int ks = 0; ks < KS; ks++) a[ks] = a_next[ks];
        if (mt + WPP < MT) load_a(mt + WPP, a_next);
      } else {
        load_a(mt, a);
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
    if (WPP == 1) __syncwarp();
    else __syncthreads();
    // ---- product 2: |sum_m' T[(nu,n)][m'] conj(Ukq[m'][m])|^2 ----
    double *dst = g2 + ikc * (int64_t)rows * NB;
    for (int mt = sub; mt < (skip ? 0 : MT); mt += WPP) {
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
      if (have && row < rows) {
#pragma unroll
        for (int nt = 0; nt < NT; nt++) {
          const int m = 4 * nt + t;
          if (m < NB) dst[(int64_t)row * NB + m] = acc[nt][0] * acc[nt][0] + acc[nt][1] * acc[nt][1];
        }
      }
    }
    if (WPP == 1) __syncwarp();
    else __syncthreads();
  }
}


// ---------------------------------------------------------------------------------------------------------------
// The same two products with g~ of a pair brought into shared memory by ONE 1-D bulk TMA copy (g~ of a pair is a
// contiguous run of 16 Nb^2 Nm bytes), two warps per pair, persistent CTAs of 64 threads.  The register-staged kernel
// above waits for its A' fragments at their point of use (long-scoreboard stalls: 198 us per q on configs[2] for 93 us of
// DMMA work and 63 us of HBM time); here the copy of the NEXT pair is issued as soon as product 1 has read the buffer, so it
// flies during product 2, the U loads and the epilogue, and the fragments come from shared memory.
// ---------------------------------------------------------------------------------------------------------------
constexpr int ROTT_WARPS = 2;

template <int NB>
__global__ void __launch_bounds__(ROTT_WARPS * 32)
    rotate_g2_tma_kernel(const c128 *__restrict__ gt, int64_t stride_gt, const c128 *__restrict__ Uk,
                         const c128 *__restrict__ Ukq, const int32_t *__restrict__ kq_idx, int nm, int64_t nk,
                         const uint8_t *__restrict__ mask, double *__restrict__ g2) {
  constexpr int KS = (2 * NB + 3) / 4, NT = (2 * NB + 7) / 8, SP = rot_pitch(NB);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = lane >> 2, t = lane & 3;
  const int rows = nm * NB, MT = (rows + 7) >> 3;
  const uint32_t gbytes = (uint32_t)(sizeof(c128) * rows * NB);
  constexpr uint32_t ubytes = (uint32_t)(sizeof(c128) * NB * NB);
  double *sGt = reinterpret_cast<double *>(smem_raw);                                   // g~ of the pair [nu][n'][m']
  double *sU = reinterpret_cast<double *>(smem_raw + ((gbytes + 127) & ~127u));         // U_k, U_{k+q} of the pair
  double *sT = sU + 2 * NB * NB * 2;                                                    // [MT*8 rows][SP] complex
  uint64_t *bar = reinterpret_cast<uint64_t *>(sT + (size_t)MT * 8 * SP * 2);
  const uint32_t bar_a = smem_u32(bar);
  for (int i = threadIdx.x; i < MT * 8 * SP * 2; i += ROTT_WARPS * 32) sT[i] = 0.0;   // padding must stay finite
  if (threadIdx.x == 0) {
    mbar_init(bar_a, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  // the pairs of this CTA: ik = blockIdx.x, + gridDim.x, ...; skipped pairs (energy window) are not loaded
  auto next_live = [&](int64_t ik) {
    while (ik < nk && mask != nullptr && mask[ik] == 0) {
      double *dz = g2 + ik * (int64_t)rows * NB;
      for (int i = threadIdx.x; i < rows * NB; i += ROTT_WARPS * 32) dz[i] = 0.0;   // a skipped pair reports zeros
      ik += gridDim.x;
    }
    return ik;
  };
  auto issue = [&](int64_t ik) {
    if (threadIdx.x == 0 && ik < nk) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_expect_tx(bar_a, gbytes + 2 * ubytes);
      tma_bulk_g2s(smem_u32(sGt), gt + ik * stride_gt, gbytes, bar_a);
      tma_bulk_g2s(smem_u32(sU), Uk + ik * (NB * NB), ubytes, bar_a);
      tma_bulk_g2s(smem_u32(sU + NB * NB * 2), Ukq + (kq_idx ? (int64_t)kq_idx[ik] : ik) * (NB * NB), ubytes, bar_a);
    }
  };
  int64_t ik = next_live(blockIdx.x);
  issue(ik);
  uint32_t phase = 0;
  while (ik < nk) {
    mbar_wait(bar_a, phase);
    phase ^= 1;
    // ---- B', B'' fragments of this pair, from the two U matrices that came with g~ ----
    double b1[KS][NT], b2[KS][NT];
    {
      const double *uk = sU + ((t & 1) ^ (g & 1));
      const double *ukq = sU + NB * NB * 2 + ((t & 1) ^ (g & 1));
      const bool n1 = (t & 1) == 1 && (g & 1) == 0, n2 = (t & 1) == 0 && (g & 1) == 1;   // sign of the embedding entries
#pragma unroll
      for (int ks = 0; ks < KS; ks++)
#pragma unroll
        for (int nt = 0; nt < NT; nt++) {
          const int r = 2 * ks + (t >> 1), c = 4 * nt + (g >> 1);
          const bool ok = r < NB && c < NB;
          const double x = ok ? uk[(r + NB * c) * 2] : 0.0, y = ok ? ukq[(r + NB * c) * 2] : 0.0;
          b1[ks][nt] = n1 ? -x : x;
          b2[ks][nt] = n2 ? -y : y;
        }
    }
    // ---- product 1: T[(nu,m')][n], row tiles dealt to the two warps ----
    for (int mt = warp; mt < MT; mt += ROTT_WARPS) {
      const int row = 8 * mt + g;
      const bool rv = row < rows;
      const int nu = row / NB, mp = row - nu * NB;
      double a[KS];
#pragma unroll
      for (int ks = 0; ks < KS; ks++) {
        const int np_ = 2 * ks + (t >> 1);
        a[ks] = (rv && np_ < NB) ? sGt[(((size_t)nu * NB + np_) * NB + mp) * 2 + (t & 1)] : 0.0;
      }
      double acc[NT][2];
#pragma unroll
      for (int nt = 0; nt < NT; nt++) acc[nt][0] = acc[nt][1] = 0.0;
#pragma unroll
      for (int ks = 0; ks < KS; ks++)
#pragma unroll
        for (int nt = 0; nt < NT; nt++) dmma884(acc[nt][0], acc[nt][1], a[ks], b1[ks][nt]);
      if (rv) {
#pragma unroll
        for (int nt = 0; nt < NT; nt++) {
          const int n = 4 * nt + t;
          if (n < NB)
            *reinterpret_cast<double2 *>(sT + ((size_t)(nu * NB + n) * SP + mp) * 2) = make_double2(acc[nt][0], acc[nt][1]);
        }
      }
    }
    __syncthreads();   // T complete; g~ buffer free: the copy of the next pair flies during product 2
    const int64_t ik_next = next_live(ik + gridDim.x);
    issue(ik_next);
    // ---- product 2: |sum_m' T[(nu,n)][m'] conj(Ukq[m'][m])|^2 ----
    double *dst = g2 + ik * (int64_t)rows * NB;
    for (int mt = warp; mt < MT; mt += ROTT_WARPS) {
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
    __syncthreads();   // T buffer free for the next pair
    ik = ik_next;
  }
}

template <int NB>
static cudaError_t launch_rot_tma(const c128 *gt, int64_t stride_gt, const c128 *Uk, const c128 *Ukq, const int32_t *kq_idx,
                                  int nm, int64_t nk, const uint8_t *mask, double *g2, cudaStream_t st) {
  const int rows = nm * NB, MT = (rows + 7) / 8;
  const size_t gbytes = sizeof(c128) * (size_t)rows * NB;
  const size_t smem = ((gbytes + 127) & ~(size_t)127) + 2 * sizeof(c128) * NB * NB + sizeof(c128) * (size_t)MT * 8 * rot_pitch(NB) + 16;
  cudaError_t e = cudaFuncSetAttribute(rotate_g2_tma_kernel<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int per_sm = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, rotate_g2_tma_kernel<NB>, ROTT_WARPS * 32, smem);
  if (e != cudaSuccess) return e;
  if (per_sm < 1) return cudaErrorInvalidConfiguration;
  const unsigned grid = grid_cap(nk, per_sm);
  rotate_g2_tma_kernel<NB><<<grid, ROTT_WARPS * 32, smem, st>>>(gt, stride_gt, Uk, Ukq, kq_idx, nm, nk, mask, g2);
  return cudaGetLastError();
}

template <int NB, int WPP>
static cudaError_t launch_rot(const c128 *gt, int64_t stride_gt, const c128 *Uk, const c128 *Ukq, const int32_t *kq_idx,
                              int nm, int64_t nk, const uint8_t *mask, double *g2, size_t smem_per_pair, cudaStream_t st) {
  constexpr int PPC = ROT_WARPS / WPP;
  const size_t smem = smem_per_pair * PPC;
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(rotate_g2_dmma_kernel<NB, WPP>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem);
    if (e != cudaSuccess) return e;
  }
  const int64_t want = ceil_div(nk, PPC);
  const unsigned grid = grid_cap(want, 16);
  rotate_g2_dmma_kernel<NB, WPP><<<grid, ROT_THREADS, smem, st>>>(gt, stride_gt, Uk, Ukq, kq_idx, nm, nk, mask, g2);
  return cudaGetLastError();
}

template <int NB>
static cudaError_t launch_rot_nb(const c128 *gt, int64_t stride_gt, const c128 *Uk, const c128 *Ukq,
                                 const int32_t *kq_idx, int nm, int64_t nk, const uint8_t *mask, double *g2,
                                 cudaStream_t st) {
  const int MT = (nm * NB + 7) / 8;
  const size_t per_pair = sizeof(c128) * (size_t)MT * 8 * rot_pitch(NB);
  if (per_pair > (size_t)200 * 1024) return cudaErrorInvalidConfiguration;
  // g~ of a pair through shared memory by bulk TMA when it and the T buffer leave room for at least four CTAs per SM and
  // there are pairs enough to fill the GPU; the copy needs 16-byte aligned runs (always: complex rows)
  const size_t tma_smem = sizeof(c128) * ((size_t)nm + 2) * NB * NB + per_pair + 144;
  if (tma_smem <= (size_t)56 * 1024 && nk >= 1024)
    return launch_rot_tma<NB>(gt, stride_gt, Uk, Ukq, kq_idx, nm, nk, mask, g2, st);
  // one warp per pair while four staging buffers fit comfortably; otherwise 2 or 4 warps share a pair
  if (per_pair <= (size_t)12 * 1024) return launch_rot<NB, 1>(gt, stride_gt, Uk, Ukq, kq_idx, nm, nk, mask, g2, per_pair, st);
  if (per_pair <= (size_t)24 * 1024) return launch_rot<NB, 2>(gt, stride_gt, Uk, Ukq, kq_idx, nm, nk, mask, g2, per_pair, st);
  return launch_rot<NB, 4>(gt, stride_gt, Uk, Ukq, kq_idx, nm, nk, mask, g2, per_pair, st);
}

bool rotate_g2_small_supported(int nb, int nm) {
  if (nb < 1 || nb > 16) return false;
  const int MT = (nm * nb + 7) / 8;
  return sizeof(c128) * (size_t)MT * 8 * rot_pitch(nb) <= (size_t)200 * 1024;
}

cudaError_t launch_rotate_g2(const c128 *gt, int64_t stride_gt, const c128 *Uk, const c128 *Ukq, const int32_t *kq_idx,
                             int nb, int nm, int64_t nk, const uint8_t *mask, double *g2, cudaStream_t st) {
  if (nk <= 0) return cudaSuccess;
  switch (nb) {
#define EPW_ROT_CASE(NB_) \
  case NB_: return launch_rot_nb<NB_>(gt, stride_gt, Uk, Ukq, kq_idx, nm, nk, mask, g2, st);
    EPW_ROT_CASE(1) EPW_ROT_CASE(2) EPW_ROT_CASE(3) EPW_ROT_CASE(4) EPW_ROT_CASE(5) EPW_ROT_CASE(6) EPW_ROT_CASE(7)
    EPW_ROT_CASE(8) EPW_ROT_CASE(9) EPW_ROT_CASE(10) EPW_ROT_CASE(11) EPW_ROT_CASE(12) EPW_ROT_CASE(13)
    EPW_ROT_CASE(14) EPW_ROT_CASE(15) EPW_ROT_CASE(16)
#undef EPW_ROT_CASE
    default: return cudaErrorInvalidConfiguration;  // Nb > 16: the large-Nb path (zgemm_strided.cu) does S4b
  }
}

}  // namespace epw
