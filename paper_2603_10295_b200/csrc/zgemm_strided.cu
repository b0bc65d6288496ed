// zgemm_strided.cu -- the FP64 tensor-path (DMMA) contraction of the LARGE-Nb path (Nb > 16; BASELINE.json configs[4],
// the stanene-nanoribbon-like case, Table III), where every operand is too big to be re-packed:
//
//   S4a  g^(Re,q)[x][nu]      = sum_ka  g(Re,q)[x][ka] e_q[ka][nu]/sqrt(2 omega_nu)        x = (Re,n',m')   PAPER.md:L114 u_{ka,nu}(q)
//   S2   g~(k,q)[c][k]        = sum_Re  g^(Re,q)[c][Re] P_k[Re][k]                         c = (nu,n',m')   PAPER.md:L112-118 (Eq. 10, "FT w.r.t. Re")
//   S4b  T_k[(nu,m')][n]      = sum_n'  g~_k[(nu,m')][n'] U_k[n'][n]                                        PAPER.md:L114, L104 ("successive
//        |g|^2_k[(nu,n)][m]   = | sum_m' T_k[(nu,n)][m'] conj(U_{k+q}[m'][m]) |^2                            multiplication")
//
// All four are  C[row][col] = sum_r A[row][r] B[r][col]  with a huge `row` range (10^5..10^7), a small B (packed once
// in DMMA fragment order, common.cuh) and an A operand that is read IN PLACE: its rows are contiguous for fixed r,
//     A[row][r] at  A + (row / a_rb) * a_bs + (row % a_rb) + r * a_ks        (c128 elements),
// so a (128-row, 8-r) tile is 8..16 one-dimensional bulk-TMA copies (cp.async.bulk, SASS UBLKCP) into a padded
// shared-memory panel [r][132] whose DMMA fragment loads (LDS.64) are bank-conflict free.  Everything else is the
// pipeline of zgemm_dmma.cu: one producer warp feeding a 6-stage mbarrier ring, 8 consumer warps with 64 x 32 (real)
// warp tiles issuing 32 independent mma.sync.m8n8k4.f64 (SASS DMMA) per r-step, persistent CTAs, n-fastest tiles.
// The epilogue writes   C + (row / c_rb) * c_bs + (row % c_rb) * c_rs + col * c_cs   either as c128 or, for the last
// contraction of the path, as |.|^2 in FP64 -- the layout of the consumer, so no transposition pass exists either.
// `batch` independent problems (one per k of a k-chunk) share one launch; B of batch b is b_gather ? b_gather[b] : b.
// Roofline: 8 * batch * M * N * K flops against the measured DMMA peak.
#include "common.cuh"
#include "dmma_pipe.cuh"

namespace epw {

constexpr int SA_STAGES = 6;
constexpr int SA_CONSUMER_WARPS = 8;
constexpr int SA_THREADS = (SA_CONSUMER_WARPS + 1) * 32;
constexpr int SA_LD = 132;                                        // complex elements per r-line of the A panel
constexpr uint32_t SA_A_BYTES = 8 * SA_LD * sizeof(c128);          // 16,896
constexpr uint32_t SA_B_BYTES = GEMM_CHUNK * sizeof(double);       // 16,384
constexpr uint32_t SA_STAGE_BYTES = SA_A_BYTES + SA_B_BYTES;
constexpr size_t SA_SMEM_BYTES = (size_t)SA_STAGES * SA_STAGE_BYTES + 2 * SA_STAGES * sizeof(uint64_t) + 128;

struct StridedGemmParams {
  const c128 *A;
  int64_t a_rb, a_bs, a_ks, a_batch;  // row-block length, block stride, r stride, batch stride (c128 elements)
  const double *Bpack;                // [batch or gathered][NT][KB][2048]
  const int32_t *b_gather;            // NULL or [batch]
  void *C;
  int64_t c_rb, c_bs, c_rs, c_cs, c_batch;  // element strides (c128 or double elements, see abs2)
  int64_t M;
  int N, K, KB, NT;
  int64_t MT, tiles_per_batch, num_tiles;
  int abs2;
};

__global__ void __launch_bounds__(SA_THREADS, 1) zgemm_strided_kernel(const StridedGemmParams p) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t *bars = reinterpret_cast<uint64_t *>(smem_raw + (size_t)SA_STAGES * SA_STAGE_BYTES);
  const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + SA_STAGES);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  // rows >= M and r >= K of a panel are never copied: start from zeros so that they stay finite (they only ever
  // multiply zero-padded B entries or feed rows that are not stored)
  {
    double2 *z = reinterpret_cast<double2 *>(smem_raw);
    for (uint32_t i = threadIdx.x; i < SA_STAGES * SA_STAGE_BYTES / 16; i += SA_THREADS) z[i] = make_double2(0.0, 0.0);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (threadIdx.x == 0) {
    for (int s = 0; s < SA_STAGES; s++) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, SA_CONSUMER_WARPS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp == SA_CONSUMER_WARPS) {
    // ============ producer warp: lanes 0..7 each copy one r-line of the A panel, lane 0 also the B chunk ============
    if (lane < 8) {
      uint32_t stage = 0, phase = 0;
      for (int64_t tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
        const int64_t b = tile / p.tiles_per_batch;
        const int64_t rem = tile - b * p.tiles_per_batch;
        const int64_t mt = rem / p.NT;
        const int nt = (int)(rem - mt * p.NT);
        const int64_t row0 = mt * GEMM_BM;
        const int64_t rend = row0 + GEMM_BM < p.M ? row0 + GEMM_BM : p.M;
        const c128 *a_src = p.A + b * p.a_batch;
        const int64_t bb = p.b_gather ? (int64_t)p.b_gather[b] : b;
        const double *b_src = p.Bpack + ((bb * p.NT + nt) * (int64_t)p.KB) * GEMM_CHUNK;
        for (int kb = 0; kb < p.KB; kb++) {
          mbar_wait(empty0 + 8 * stage, phase ^ 1);
          const uint32_t dst = smem_u32(smem_raw + (size_t)stage * SA_STAGE_BYTES);
          const uint32_t bar = full0 + 8 * stage;
          const int kvalid = p.K - kb * 8 < 8 ? p.K - kb * 8 : 8;
          if (lane == 0) {
            mbar_expect_tx(bar, (uint32_t)(kvalid * (rend - row0) * sizeof(c128)) + SA_B_BYTES);
            tma_bulk_g2s(dst + SA_A_BYTES, b_src + (int64_t)kb * GEMM_CHUNK, SA_B_BYTES, bar);
          }
          if (lane < kvalid) {
            const int64_t r = (int64_t)kb * 8 + lane;
            int64_t row = row0;
            int64_t blk = row / p.a_rb;
            int64_t off = row - blk * p.a_rb;
            while (row < rend) {
              int64_t len = p.a_rb - off;
              if (len > rend - row) len = rend - row;
              tma_bulk_g2s(dst + (uint32_t)((lane * SA_LD + (row - row0)) * sizeof(c128)),
                           a_src + blk * p.a_bs + off + r * p.a_ks, (uint32_t)(len * sizeof(c128)), bar);
              row += len;
              blk++;
              off = 0;
            }
          }
          if (++stage == SA_STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
    return;
  }

  // ================================ consumer warps: DMMA main loop + epilogue ====================================
  const int wm = warp >> 2, wn = warp & 3;
  const int g = lane >> 2, t = lane & 3;
  uint32_t stage = 0, phase = 0;
  for (int64_t tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
    const int64_t b = tile / p.tiles_per_batch;
    const int64_t rem = tile - b * p.tiles_per_batch;
    const int64_t mt = rem / p.NT;
    const int nt = (int)(rem - mt * p.NT);
    double acc[8][4][2];
#pragma unroll
    for (int i = 0; i < 8; i++)
#pragma unroll
      for (int j = 0; j < 4; j++) acc[i][j][0] = acc[i][j][1] = 0.0;

    for (int kb = 0; kb < p.KB; kb++) {
      mbar_wait(full0 + 8 * stage, phase);
      const double *sA = reinterpret_cast<const double *>(smem_raw + (size_t)stage * SA_STAGE_BYTES);
      const double2 *sB = reinterpret_cast<const double2 *>(smem_raw + (size_t)stage * SA_STAGE_BYTES + SA_A_BYTES);
      // real k index 4 ks + t  <->  complex r = 2 ks + (t >> 1), component t & 1   (the order of the packed B', common.cuh)
      const double *aBase = sA + (((t >> 1) * SA_LD + wm * 64 + g) << 1) + (t & 1);
#pragma unroll
      for (int ks = 0; ks < 4; ks++) {
        double a[8], bf[4];
#pragma unroll
        for (int i = 0; i < 8; i++) a[i] = aBase[(2 * ks * SA_LD + 8 * i) << 1];
#pragma unroll
        for (int j2 = 0; j2 < 2; j2++) {
          const double2 v = sB[((wn * 4 + ks) * 2 + j2) * 32 + lane];
          bf[2 * j2] = v.x;
          bf[2 * j2 + 1] = v.y;
        }
#pragma unroll
        for (int i = 0; i < 8; i++)
#pragma unroll
          for (int j = 0; j < 4; j++) dmma884(acc[i][j][0], acc[i][j][1], a[i], bf[j]);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(empty0 + 8 * stage);
      if (++stage == SA_STAGES) { stage = 0; phase ^= 1; }
    }

    // epilogue: thread owns complex C[row0 + 8 i][col0 + 4 j]
    const int64_t row0 = mt * GEMM_BM + wm * 64 + g;
    const int col0 = nt * 64 + wn * 16 + t;
#pragma unroll
    for (int i = 0; i < 8; i++) {
      const int64_t row = row0 + i * 8;
      if (row < p.M) {
        const int64_t blk = row / p.c_rb;
        const int64_t base = b * p.c_batch + blk * p.c_bs + (row - blk * p.c_rb) * p.c_rs;
#pragma unroll
        for (int j = 0; j < 4; j++) {
          const int col = col0 + j * 4;
          if (col < p.N) {
            const int64_t at = base + (int64_t)col * p.c_cs;
            if (p.abs2)
              reinterpret_cast<double *>(p.C)[at] = acc[i][j][0] * acc[i][j][0] + acc[i][j][1] * acc[i][j][1];
            else
              reinterpret_cast<c128 *>(p.C)[at] = make_double2(acc[i][j][0], acc[i][j][1]);
          }
        }
      }
    }
  }
}

cudaError_t launch_zgemm_strided(const c128 *A, int64_t a_rb, int64_t a_bs, int64_t a_ks, int64_t a_batch,
                                 const double *Bpack, const int32_t *b_gather, void *C, int64_t c_rb, int64_t c_bs,
                                 int64_t c_rs, int64_t c_cs, int64_t c_batch, int abs2, int64_t M, int N, int K,
                                 int64_t batch, int num_sms, cudaStream_t st) {
  if (M <= 0 || N <= 0 || K <= 0 || batch <= 0) return cudaSuccess;
  if (a_rb <= 0 || c_rb <= 0) return cudaErrorInvalidValue;
  // the shared-memory opt-in is a per-device attribute: set it on every launch (cheap) instead of caching it per process
  {
    cudaError_t e = cudaFuncSetAttribute(zgemm_strided_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)SA_SMEM_BYTES);
    if (e != cudaSuccess) return e;
  }
  StridedGemmParams p;
  p.A = A; p.a_rb = a_rb; p.a_bs = a_bs; p.a_ks = a_ks; p.a_batch = a_batch;
  p.Bpack = Bpack; p.b_gather = b_gather;
  p.C = C; p.c_rb = c_rb; p.c_bs = c_bs; p.c_rs = c_rs; p.c_cs = c_cs; p.c_batch = c_batch;
  p.M = M; p.N = N; p.K = K;
  p.KB = (int)ceil_div(2 * (int64_t)K, GEMM_BK);
  p.NT = (int)ceil_div(2 * (int64_t)N, GEMM_BN);
  p.MT = ceil_div(M, GEMM_BM);
  p.tiles_per_batch = p.MT * p.NT;
  p.num_tiles = p.tiles_per_batch * batch;
  p.abs2 = abs2;
  const int grid = (int)(p.num_tiles < num_sms ? p.num_tiles : num_sms);
  zgemm_strided_kernel<<<grid, SA_THREADS, SA_SMEM_BYTES, st>>>(p);
  return cudaGetLastError();
}

}  // namespace epw
