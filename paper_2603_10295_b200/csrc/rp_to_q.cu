// rp_to_q.cu -- S1, Eq. 9:  g(Re,q) = sum_Rp g(Re,Rp) w_p e^{i q.Rp}.
//
// The paper runs this as one ZGEMV per q: every q re-reads all 16 Nb^2 Nm Ne Np bytes of g,
// 0.5 flop/byte, HBM-bound.  Here NQ q-points share one streaming pass over g (a skinny GEMM,
// [rows x Np] . [Np x NQ]): g is read once per batch with coalesced 16-byte loads, NQ complex accumulators
// live in registers, and the phase columns are broadcast from shared memory.  HBM roofline: 16*rows*Np bytes
// read + 16*rows*NQ bytes written per launch.
#include "common.cuh"
#include "dmma_pipe.cuh"

namespace epw {

// Where the sum of a row goes.  Normally g1[iq][row].  With a destination table (the Rp-sharded form, PAPER.md:L186-188,
// L514-522) the partial sum of this GPU's lattice vectors is ADDED to dst_tab[iq][row] instead -- dst_tab[iq] is the
// buffer of the rank that owns q-point iq and may be PEER memory (NVLink P2P mapping): the exchange step of the sharded
// path (a reduce-scatter over q of the partial g(Re,q)) then happens inside the streaming pass, row tile by row tile,
// as red.global.add.f64 at system scope, instead of as a collective after it.
__device__ __forceinline__ void emit_row(c128 *__restrict__ g1, c128 *const *__restrict__ dst_tab, int iq, int64_t rows,
                                         int64_t row, c128 v) {
  if (dst_tab == nullptr) {
    g1[(int64_t)iq * rows + row] = v;
  } else {
    double *d = reinterpret_cast<double *>(dst_tab[iq] + row);
    atomicAdd_system(d, v.x);
    atomicAdd_system(d + 1, v.y);
  }
}

template <int NQ>
__global__ void __launch_bounds__(256) rp_to_q_kernel(const c128 *__restrict__ g, int64_t rows, int np,
                                                      const c128 *__restrict__ Pq, c128 *__restrict__ g1,
                                                      c128 *const *__restrict__ dst_tab) {
  extern __shared__ double2 sP[];  // [np][NQ]
  for (int e = threadIdx.x; e < np * NQ; e += blockDim.x) {
    const int ip = e / NQ, iq = e - ip * NQ;
    sP[e] = Pq[(int64_t)iq * np + ip];
  }
  __syncthreads();
  const int64_t row = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (row >= rows) return;
  c128 acc[NQ];
#pragma unroll
  for (int iq = 0; iq < NQ; iq++) acc[iq] = cmake(0.0, 0.0);
  const c128 *col = g + row;
  // software pipeline: the U loads of the next block of Rp are issued before the NQ x U complex FMAs of the current one,
  // so that a thread always has loads in flight while it computes (with NQ = 8 the arithmetic of a block is as long as
  // the latency it has to hide)
  constexpr int U = NQ >= 5 ? 4 : 8;  // independent 16-byte loads per block
  c128 cur[U], nxt[U];
  const int nblk = np / U;
  if (nblk > 0) {
#pragma unroll
    for (int u = 0; u < U; u++) cur[u] = __ldcs(col + (int64_t)u * rows);
  }
  for (int b = 0; b < nblk; b++) {
    const int ip = b * U;
    if (b + 1 < nblk) {
#pragma unroll
      for (int u = 0; u < U; u++) nxt[u] = __ldcs(col + (int64_t)(ip + U + u) * rows);
    }
#pragma unroll
    for (int u = 0; u < U; u++) {
#pragma unroll
      for (int iq = 0; iq < NQ; iq++) cfma(acc[iq], cur[u], sP[(ip + u) * NQ + iq]);
    }
#pragma unroll
    for (int u = 0; u < U; u++) cur[u] = nxt[u];
  }
  for (int ip = nblk * U; ip < np; ip++) {
    const c128 v = __ldcs(col + (int64_t)ip * rows);
#pragma unroll
    for (int iq = 0; iq < NQ; iq++) cfma(acc[iq], v, sP[ip * NQ + iq]);
  }
#pragma unroll
  for (int iq = 0; iq < NQ; iq++) emit_row(g1, dst_tab, iq, rows, row, acc[iq]);
}

// NQ >= 5: bulk-TMA staged variant.  With 8 q per pass the arithmetic of one Rp block (32 DFMA per 16 bytes) takes as
// long as the HBM latency it has to hide, and register-staged loads cannot keep enough bytes in flight (measured: time =
// memory time + FP64 time, 3.6 TB/s).  Here one producer thread streams [RP_IPS lattice vectors] x [RB rows] tiles of g
// into a RP_STAGES-deep shared-memory ring with 1-D bulk TMA copies (cp.async.bulk + mbarrier complete_tx, SASS UBLKCP:
// each Rp column of a row tile is one contiguous run of RB x 16 bytes), ~96 KB in flight per SM, while RB consumer
// threads (one row each, NQ complex accumulators in registers) read the tiles with conflict-free LDS.128 and the phases
// by broadcast.  Persistent CTAs, one per SM; the row-tile height is chosen on the host for whole waves.
constexpr int RP_IPS = 4;       // lattice vectors per stage
constexpr int RP_STAGES = 4;
constexpr int RP_MAX_RB = 512;  // rows per tile (= consumer threads), multiple of 32
constexpr int RP_THREADS = RP_MAX_RB + 32;

template <int NQ>
__global__ void __launch_bounds__(RP_THREADS, 1)
    rp_to_q_tma_kernel(const c128 *__restrict__ g, int64_t rows, int np, const c128 *__restrict__ Pq,
                       c128 *__restrict__ g1, c128 *const *__restrict__ dst_tab, int RB, int64_t num_tiles) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  c128 *ring = reinterpret_cast<c128 *>(smem_raw);                                        // [STAGES][IPS][RB]
  uint64_t *bars = reinterpret_cast<uint64_t *>(smem_raw + sizeof(c128) * (size_t)RP_STAGES * RP_IPS * RB);
  double2 *sP = reinterpret_cast<double2 *>(bars + 2 * RP_STAGES);                       // [np][NQ]
  const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + RP_STAGES);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int cwarps = RB >> 5;
  for (int e = threadIdx.x; e < np * NQ; e += RP_THREADS) {
    const int ip = e / NQ, iq = e - ip * NQ;
    sP[e] = Pq[(int64_t)iq * np + ip];
  }
  if (threadIdx.x == 0) {
    for (int s = 0; s < RP_STAGES; s++) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, cwarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int nblk = (np + RP_IPS - 1) / RP_IPS;

  if (warp == RP_MAX_RB / 32) {
    // ================= producer: one elected lane =================
    if (lane == 0) {
      uint32_t stage = 0, phase = 0;
      for (int64_t tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
        const int64_t row0 = tile * RB;
        const int64_t nrow = rows - row0 < RB ? rows - row0 : RB;
        for (int b = 0; b < nblk; b++) {
          const int ip0 = b * RP_IPS;
          const int nip = np - ip0 < RP_IPS ? np - ip0 : RP_IPS;
          mbar_wait(empty0 + 8 * stage, phase ^ 1);
          const uint32_t bar = full0 + 8 * stage;
          mbar_expect_tx(bar, (uint32_t)(nip * nrow * sizeof(c128)));
          for (int u = 0; u < nip; u++)
            tma_bulk_g2s(smem_u32(ring + ((size_t)stage * RP_IPS + u) * RB), g + (int64_t)(ip0 + u) * rows + row0,
                         (uint32_t)(nrow * sizeof(c128)), bar);
          if (++stage == RP_STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
    return;
  }
  if (warp >= cwarps) return;

  // ================= consumers: one row per thread =================
  uint32_t stage = 0, phase = 0;
  for (int64_t tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
    const int64_t row = tile * RB + threadIdx.x;
    const bool valid = row < rows;
    c128 acc[NQ];
#pragma unroll
    for (int iq = 0; iq < NQ; iq++) acc[iq] = cmake(0.0, 0.0);
    for (int b = 0; b < nblk; b++) {
      const int ip0 = b * RP_IPS;
      const int nip = np - ip0 < RP_IPS ? np - ip0 : RP_IPS;
      mbar_wait(full0 + 8 * stage, phase);
      const c128 *src = ring + (size_t)stage * RP_IPS * RB + threadIdx.x;
      if (valid) {
        if (nip == RP_IPS) {
#pragma unroll
          for (int u = 0; u < RP_IPS; u++) {
            const c128 v = src[(size_t)u * RB];
#pragma unroll
            for (int iq = 0; iq < NQ; iq++) cfma(acc[iq], v, sP[(ip0 + u) * NQ + iq]);
          }
        } else {
          for (int u = 0; u < nip; u++) {
            const c128 v = src[(size_t)u * RB];
#pragma unroll
            for (int iq = 0; iq < NQ; iq++) cfma(acc[iq], v, sP[(ip0 + u) * NQ + iq]);
          }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(empty0 + 8 * stage);
      if (++stage == RP_STAGES) { stage = 0; phase ^= 1; }
    }
    if (valid) {
#pragma unroll
      for (int iq = 0; iq < NQ; iq++) emit_row(g1, dst_tab, iq, rows, row, acc[iq]);
    }
  }
}

template <int NQ>
static cudaError_t launch_nq(const c128 *g, int64_t rows, int np, const c128 *Pq, c128 *g1, c128 *const *dst_tab,
                             cudaStream_t st);

template <int NQ>
static cudaError_t launch_nq_tma(const c128 *g, int64_t rows, int np, const c128 *Pq, c128 *g1, c128 *const *dst_tab,
                                 cudaStream_t st) {
  const int nsm = device_sm_count();
  // row-tile height: the multiple of 32 in [256, 512] whose tile count fills whole waves best
  int RB = RP_MAX_RB;
  double best = -1.0;
  for (int rb = RP_MAX_RB; rb >= 256; rb -= 32) {
    const int64_t tiles = ceil_div(rows, rb);
    const double eff = (double)rows / ((double)ceil_div(tiles, nsm) * nsm * rb);
    if (eff > best + 1e-9) { best = eff; RB = rb; }
  }
  const size_t smem = sizeof(c128) * (size_t)RP_STAGES * RP_IPS * RB + 2 * RP_STAGES * sizeof(uint64_t) +
                      sizeof(double2) * (size_t)np * NQ;
  if (smem > (size_t)225 * 1024 || rows < 4 * (int64_t)nsm * 32) return launch_nq<NQ>(g, rows, np, Pq, g1, dst_tab, st);
  cudaError_t e = cudaFuncSetAttribute(rp_to_q_tma_kernel<NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  const int64_t tiles = ceil_div(rows, RB);
  const int grid = (int)(tiles < nsm ? tiles : nsm);
  rp_to_q_tma_kernel<NQ><<<grid, RP_THREADS, smem, st>>>(g, rows, np, Pq, g1, dst_tab, RB, tiles);
  return cudaGetLastError();
}

template <int NQ>
static cudaError_t launch_nq(const c128 *g, int64_t rows, int np, const c128 *Pq, c128 *g1, c128 *const *dst_tab,
                             cudaStream_t st) {
  const size_t smem = sizeof(double2) * (size_t)np * NQ;
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(rp_to_q_kernel<NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  rp_to_q_kernel<NQ><<<(unsigned)ceil_div(rows, 256), 256, smem, st>>>(g, rows, np, Pq, g1, dst_tab);
  return cudaGetLastError();
}

// The kernels keep the phase table [np][NQ] of a pass in shared memory (16 np NQ bytes): the largest NQ <= 8 that fits
// the 227 KB a CTA may use, 0 if not even one q-point fits (Np > ~14,000).
int rp_to_q_max_nq(int np) {
  const size_t limit = (size_t)220 * 1024;
  for (int nq = 8; nq >= 1; nq--)
    if (sizeof(double2) * (size_t)np * nq <= limit) return nq;
  return 0;
}

cudaError_t launch_rp_to_q(const c128 *g, int64_t rows, int np, const c128 *Pq, int nq, c128 *g1, cudaStream_t st) {
  return launch_rp_to_q_dst(g, rows, np, Pq, nq, g1, nullptr, st);
}

// dst_tab (device array of nq device pointers, may be NULL): see emit_row
cudaError_t launch_rp_to_q_dst(const c128 *g, int64_t rows, int np, const c128 *Pq, int nq, c128 *g1, c128 *const *dst_tab,
                               cudaStream_t st) {
  if (nq > rp_to_q_max_nq(np)) return cudaErrorInvalidConfiguration;
  switch (nq) {
    case 1: return launch_nq<1>(g, rows, np, Pq, g1, dst_tab, st);
    case 2: return launch_nq<2>(g, rows, np, Pq, g1, dst_tab, st);
    case 3: return launch_nq<3>(g, rows, np, Pq, g1, dst_tab, st);
    case 4: return launch_nq<4>(g, rows, np, Pq, g1, dst_tab, st);
    case 5: return launch_nq_tma<5>(g, rows, np, Pq, g1, dst_tab, st);
    case 6: return launch_nq_tma<6>(g, rows, np, Pq, g1, dst_tab, st);
    case 7: return launch_nq_tma<7>(g, rows, np, Pq, g1, dst_tab, st);
    case 8: return launch_nq_tma<8>(g, rows, np, Pq, g1, dst_tab, st);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace epw
