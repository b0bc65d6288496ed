// zgemm_dmma.cu -- S2, the dominant contraction (FT part of Eq. 10):
//     g~[k][col] = sum_Re  P_k[k][Re] * B_q[Re][col]        for every k of the batch at once,
// where col runs over (nu, n', m') of the mode-rotated g^(Re,q) and, for off-grid q, over the Nb^2 extra columns
// e^{2 pi i q.Re} H(Re) that yield H(k+q) from the same pass.
// The paper evaluates this as one GEMV-like sum per k on a CPU thread; batching over k
// turns it into a dense complex-FP64 GEMM, executed here on Blackwell's FP64 tensor path.
//
// sm_100a has no tcgen05 kind for FP64: the FP64 tensor instruction is the warp-level DMMA (mma.sync m8n8k4.f64,
// SASS DMMA.8x8x4; the m16n8k{4,8,16}.f64 shapes lower to the same instruction), measured at 37.0 TFLOP/s on this
// B200 = 64 FMA/clk/SM (epw_probe_peaks, printed in every bench line).  The kernel is built around that:
//   * complex product as a real GEMM with interleaved re/im (common.cuh): 4 real FMA per complex MAC, no waste;
//   * both operands are pre-packed in fragment order, so a (tile, k-block) chunk is ONE 16 KB 1-D bulk TMA copy
//     (cp.async.bulk ... mbarrier::complete_tx, SASS UBLKCP) and every fragment load is a conflict-free LDS.128;
//   * warp-specialised: 1 producer warp drives a STAGES-deep mbarrier ring, 8 consumer warps (2 x 4, warp tile
//     64 x 32 real) issue 32 independent DMMAs per k-step (6 LDS.128 per 32 DMMA);
//   * persistent CTAs (one per SM, grid = min(tiles, #SM)), tiles ordered n-fastest so that concurrently running
//     CTAs share the same A panel in L2; the epilogue of a tile overlaps the producer's prefetch of the next.
// Roofline: 8 * M * N * K flops (N, K complex) against the measured DMMA peak.
#include "common.cuh"
#include "dmma_pipe.cuh"

namespace epw {

constexpr int GEMM_STAGES = 6;
constexpr int GEMM_CONSUMER_WARPS = 8;
constexpr int GEMM_THREADS = (GEMM_CONSUMER_WARPS + 1) * 32;
constexpr uint32_t GEMM_STAGE_BYTES = 2 * GEMM_CHUNK * sizeof(double);  // A chunk + B chunk
constexpr size_t GEMM_SMEM_BYTES = (size_t)GEMM_STAGES * GEMM_STAGE_BYTES + 2 * GEMM_STAGES * sizeof(uint64_t) + 128;

__global__ void __launch_bounds__(GEMM_THREADS, 1)
    zgemm_dmma_kernel(const double *__restrict__ Apack, const double *__restrict__ Bpack, c128 *__restrict__ C,
                      int64_t M, int N, int KB, int64_t ldc, int NT, int64_t num_tiles) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double *stage_base = reinterpret_cast<double *>(smem_raw);
  uint64_t *bars = reinterpret_cast<uint64_t *>(smem_raw + (size_t)GEMM_STAGES * GEMM_STAGE_BYTES);
  const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + GEMM_STAGES);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < GEMM_STAGES; s++) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, GEMM_CONSUMER_WARPS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp == GEMM_CONSUMER_WARPS) {
    // ===================== producer warp: one elected lane feeds the ring with bulk TMA copies ============
    if (lane == 0) {
      uint32_t stage = 0, phase = 0;
      for (int64_t tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
        const int64_t mt = tile / NT;
        const int nt = (int)(tile - mt * NT);
        const double *a_src = Apack + (mt * KB) * (int64_t)GEMM_CHUNK;
        const double *b_src = Bpack + ((int64_t)nt * KB) * (int64_t)GEMM_CHUNK;
        for (int kb = 0; kb < KB; kb++) {
          mbar_wait(empty0 + 8 * stage, phase ^ 1);
          const uint32_t dst = smem_u32(stage_base + (size_t)stage * 2 * GEMM_CHUNK);
          mbar_expect_tx(full0 + 8 * stage, GEMM_STAGE_BYTES);
          tma_bulk_g2s(dst, a_src + (int64_t)kb * GEMM_CHUNK, GEMM_CHUNK * 8, full0 + 8 * stage);
          tma_bulk_g2s(dst + GEMM_CHUNK * 8, b_src + (int64_t)kb * GEMM_CHUNK, GEMM_CHUNK * 8, full0 + 8 * stage);
          if (++stage == GEMM_STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
    return;
  }

  // ========================= consumer warps: DMMA main loop + epilogue ===================================
  const int wm = warp >> 2, wn = warp & 3;
  const int g = lane >> 2, t = lane & 3;
  uint32_t stage = 0, phase = 0;
  for (int64_t tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
    const int64_t mt = tile / NT;
    const int nt = (int)(tile - mt * NT);
    double acc[8][4][2];
#pragma unroll
    for (int i = 0; i < 8; i++)
#pragma unroll
      for (int j = 0; j < 4; j++) acc[i][j][0] = acc[i][j][1] = 0.0;

    for (int kb = 0; kb < KB; kb++) {
      mbar_wait(full0 + 8 * stage, phase);
      const double2 *sA = reinterpret_cast<const double2 *>(stage_base + (size_t)stage * 2 * GEMM_CHUNK);
      const double2 *sB = sA + GEMM_CHUNK / 2;
#pragma unroll
      for (int ks = 0; ks < 4; ks++) {
        double a[8], b[4];
#pragma unroll
        for (int i2 = 0; i2 < 4; i2++) {
          const double2 v = sA[((wm * 4 + ks) * 4 + i2) * 32 + lane];
          a[2 * i2] = v.x;
          a[2 * i2 + 1] = v.y;
        }
#pragma unroll
        for (int j2 = 0; j2 < 2; j2++) {
          const double2 v = sB[((wn * 4 + ks) * 2 + j2) * 32 + lane];
          b[2 * j2] = v.x;
          b[2 * j2 + 1] = v.y;
        }
#pragma unroll
        for (int i = 0; i < 8; i++)
#pragma unroll
          for (int j = 0; j < 4; j++) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(empty0 + 8 * stage);
      if (++stage == GEMM_STAGES) { stage = 0; phase ^= 1; }
    }

    // epilogue: thread owns complex C[row][col] for row = ..+i*8+g, col = ..+j*4+t  (16-byte stores; the four
    // lanes of a group write 64 contiguous bytes)
    const int64_t row0 = mt * GEMM_BM + wm * 64 + g;
    const int col0 = nt * 64 + wn * 16 + t;
#pragma unroll
    for (int i = 0; i < 8; i++) {
      const int64_t row = row0 + i * 8;
      if (row < M) {
        c128 *crow = C + row * ldc;
#pragma unroll
        for (int j = 0; j < 4; j++) {
          const int col = col0 + j * 4;
          if (col < N) crow[col] = make_double2(acc[i][j][0], acc[i][j][1]);
        }
      }
    }
  }
}

cudaError_t launch_zgemm_dmma(const double *Apack, const double *Bpack, c128 *C, int64_t M, int N, int KB, int64_t ldc,
                              int num_sms, cudaStream_t st) {
  if (M <= 0 || N <= 0 || KB <= 0) return cudaSuccess;
  // the shared-memory opt-in is a per-device attribute: set it on every launch (cheap) instead of caching it per process
  {
    cudaError_t e = cudaFuncSetAttribute(zgemm_dmma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)GEMM_SMEM_BYTES);
    if (e != cudaSuccess) return e;
  }
  const int NT = (int)ceil_div(2 * (int64_t)N, GEMM_BN);
  const int64_t MT = ceil_div(M, GEMM_BM);
  const int64_t tiles = MT * NT;
  const int grid = (int)(tiles < num_sms ? tiles : num_sms);
  zgemm_dmma_kernel<<<grid, GEMM_THREADS, GEMM_SMEM_BYTES, st>>>(Apack, Bpack, C, M, N, KB, ldc, NT, tiles);
  return cudaGetLastError();
}

}  // namespace epw
