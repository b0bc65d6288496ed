// interp.cu -- handle, memory plan, stage orchestration and the extern "C" boundary (include/epw_interp.h).
//
// Loop structure = the paper's nested-loop algorithm (Fig. 1b; Fig. 12): Eq. 9 once
// per q in the outer loop, Eq. 10 for every k in the inner loop -- except that here the inner loop is a batched
// tensor contraction on the device instead of one CPU thread per k, nothing returns to the host inside the loop
// (the paper copies x to and y from the device every q), and q-points are taken q_batch at a
// time through S1 so that g(Re,Rp) is streamed from HBM once per batch rather than once per q.
#include <algorithm>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "common.cuh"

using namespace epw;

namespace {

std::string g_create_error;

struct DevBuf {
  void *p = nullptr;
  size_t bytes = 0;
  cudaError_t reserve(size_t want) {
    if (want <= bytes) return cudaSuccess;
    if (p) cudaFree(p);
    p = nullptr;
    bytes = 0;
    cudaError_t e = cudaMalloc(&p, want);
    if (e == cudaSuccess) bytes = want;
    return e;
  }
  void release() {
    if (p) cudaFree(p);
    p = nullptr;
    bytes = 0;
  }
  template <class T>
  T *as() const { return reinterpret_cast<T *>(p); }
};

__global__ void gather_eps_kernel(const double *__restrict__ eps_k, const int32_t *__restrict__ kq_idx, int nb,
                                  int64_t nk, double *__restrict__ eps_kq) {
  const int64_t total = nk * nb;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t ik = i / nb;
    const int b = (int)(i - ik * nb);
    eps_kq[i] = eps_k[(int64_t)kq_idx[ik] * nb + b];
  }
}

// Number of 128-row m-tiles per k-chunk of the S2 contraction.  The chunk of C must stay within `l2_budget` bytes;
// among the admissible sizes pick the largest one whose tile count (mtiles * NT) wastes at most 3 % of its last
// wave on the `sms` persistent CTAs (wave quantisation), else the one with the best wave efficiency.
int64_t choose_mtiles_per_chunk(int NT, int sms, size_t bytes_per_mtile, int64_t MT, size_t l2_budget) {
  int64_t max_mt = std::max<int64_t>(1, (int64_t)(l2_budget / bytes_per_mtile));
  if (max_mt >= MT) return MT;
  int64_t best = 1;
  double best_eff = 0.0;
  for (int64_t mt = max_mt; mt >= 1; mt--) {
    const int64_t tiles = mt * NT;
    const double eff = (double)tiles / (double)(ceil_div(tiles, sms) * sms);
    if (eff >= 0.97) return mt;
    if (eff > best_eff) { best_eff = eff; best = mt; }
  }
  return best;
}

// out[b][c][r] = in[b][r][c] for blocks of rows (the phase table [k][Re] of a k-chunk as [Re][k])
__global__ void transpose_blocks_kernel(const c128 *__restrict__ in, int64_t rows, int cols, int64_t rows_per_block,
                                        c128 *__restrict__ out) {
  const int64_t total = rows * cols;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / cols;
    const int c = (int)(i - r * cols);
    const int64_t b = r / rows_per_block, rl = r - b * rows_per_block;
    const int64_t nr = rows - b * rows_per_block < rows_per_block ? rows - b * rows_per_block : rows_per_block;
    out[b * rows_per_block * cols + (int64_t)c * nr + rl] = in[i];
  }
}

__global__ void fill_ones_kernel(double *p, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = 1.0;
}

}  // namespace

struct epw_interp {
  epw_interp_config cfg{};
  int nb = 0, nm = 0, ne = 0, np = 0, nbb = 0, nmm = 0;
  int64_t rows = 0;  // Nb^2 Ne Nm = rows of Fig. 13's A(m,n)
  int num_sms = 0;   // set by epw_interp_create from the device
  int q_batch = 4;
  bool operators_set = false;
  std::vector<char> slab_set;
  // Rp shard (NEXT-1): this handle keeps only slabs [rp_lo, rp_lo + rp_cnt) of g(Re,Rp)
  int rp_lo = 0, rp_cnt = 0;
  bool sharded = false;
  // energy-window pre-screening (NEXT-3)
  bool window_on = false;
  double emin = 0.0, emax = 0.0;
  uint8_t *mask_out = nullptr;   // caller's device buffer [nq][nk] or NULL
  DevBuf maskbuf;
  // NEXT-4 consumer: Im Sigma_nk accumulator
  struct Consumer { bool on = false; double mu = 0, kT = 0, sigma = 0; const double *w_q = nullptr; double *out = nullptr; } cons;
  DevBuf g2_scratch;   // |g|^2 of one q when the caller passes g2 = NULL (consumer on)
  const c128 *ext_g1 = nullptr;  // g(Re,q) supplied by the caller (already summed over every rank's Rp) for this call
  // resident operators
  DevBuf g, H, D, Re, Rp, we, wp, ones;
  // per-call workspace
  DevBuf Apack, BpackH, Hk, Uk, Pq, Pqe, Dq, eq, g1, Bpack, C, Ukq, epskq_scratch, status, eig_scratch;
  // large-Nb path only
  DevBuf Pk, BpackPk, UpackK, UpackKH, BpackE, ghat, T, Hkq;
  // uniform-grid form of S2 (re_to_k_grid.cu): bounding box of the Re list, box-ordered operand and axis passes
  int box_lo[3] = {0, 0, 0}, box_L[3] = {1, 1, 1};
  int64_t box_size = 1;
  DevBuf boxidx, X, T1, T2, Ptmp, P1raw, P2raw, P3raw, P1pack, P2pack, P3pack, klist_gen;
  DevBuf workctr;  // 3 x u64: plane rotations executed by the register-resident eigensolvers for H(k), H(k+q), D(q)
  // eigensolver work counter of slot i (0 H(k), 1 H(k+q), 2 D(q)) while stage timing is on, else NULL
  unsigned long long *work_slot(int slot) const {
    return timing && workctr.p ? workctr.as<unsigned long long>() + slot : nullptr;
  }
  int last_kmode = 0;
  // k side of the large-Nb path kept between calls on the SAME uniform grid (phases, H(k), U_k, eps_k, packed operands):
  // valid for (grid sizes, shift, operators epoch); any k-list call or new operators drop it
  // `stream` / `ev`: the stream the k side was enqueued on and an event recorded behind it, so that a later call on ANOTHER
  // stream that hits the cache waits for the cached buffers to be complete (kside_wait)
  struct KSide { bool valid = false, with_conj = false; int path = 0; int32_t N[3] = {0, 0, 0}; double s[3] = {0, 0, 0}; uint64_t epoch = 0;
                 cudaStream_t stream = nullptr; cudaEvent_t ev = nullptr; } kside;
  uint64_t op_epoch = 0;
  DevBuf PkT;         // large-Nb path: phase table of every k-chunk transposed, [chunk][Re][k]
  DevBuf dst_tab;     // destination pointers of epw_interp_rp_to_q_scatter_add
  std::vector<void *> dst_host;   // the library's pageable copy of the caller's table (source of the stream-ordered upload)
  DevBuf epsk_keep;   // eps_k of the cached k side (the caller's buffer is refilled from it)
  int64_t last_eq_slot = 0;  // slot of the last q of the last call inside the e_q buffer (debug getter)
  // host-entry output drain: while a host-buffer call runs, the |g|^2 and eps_kq slices of every finished q are copied
  // to the caller's host buffers on a second stream, overlapping the device-to-host link with the next q's kernels
  struct HostSink { double *g2 = nullptr, *eps_kq = nullptr; bool active = false; } sink;
  cudaStream_t copy_stream = nullptr;
  // large-Nb path: the phonon eigensolves (a few n = 3 Nat Jacobi solves on one thread-block cluster each, latency bound)
  // run on a second stream beside the first S1 pass over g(Re,Rp) (HBM bound, all SMs)
  cudaStream_t aux_stream = nullptr;
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  std::vector<cudaEvent_t> sink_ev;
  size_t sink_ev_used = 0;
  int drain_q(int64_t q, int64_t nk, int64_t E, const double *g2_dev, const double *eps_kq_dev, cudaStream_t st) {
    if (!sink.active) return EPW_OK;
    if (sink_ev_used == sink_ev.size()) {
      cudaEvent_t ev;
      if (cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess) return EPW_ECUDA;
      sink_ev.push_back(ev);
    }
    cudaEvent_t ev = sink_ev[sink_ev_used++];
    cudaError_t e = cudaEventRecord(ev, st);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(copy_stream, ev, 0);
    if (e == cudaSuccess)
      e = cudaMemcpyAsync(sink.g2 + q * nk * E, g2_dev + q * nk * E, sizeof(double) * (size_t)(nk * E),
                          cudaMemcpyDeviceToHost, copy_stream);
    if (e == cudaSuccess && sink.eps_kq && eps_kq_dev)
      e = cudaMemcpyAsync(sink.eps_kq + q * nk * nb, eps_kq_dev + q * nk * nb, sizeof(double) * (size_t)(nk * nb),
                          cudaMemcpyDeviceToHost, copy_stream);
    if (e != cudaSuccess) return cuda_fail(e, "drain D2H");
    return EPW_OK;
  }
  // host-entry staging
  DevBuf hs_k, hs_q, hs_map, hs_epsk, hs_epskq, hs_omega, hs_g2;
  // bookkeeping of the last call
  int64_t last_nk = 0, last_c_rows = 0, last_kchunk = 0;
  int last_path = 0, last_qb = 0;
  int last_ncols = 0;
  int64_t launches = 0;
  cudaStream_t last_stream = nullptr;
  bool timing = false;
  std::vector<cudaEvent_t> ev_pool;
  struct Span { int stage; int e0, e1; int64_t launch0; int64_t nlaunch; };
  std::vector<Span> spans;
  size_t ev_used = 0;
  std::string last_error;

  int fail(int code, const std::string &msg) {
    last_error = msg;
    return code;
  }
  // q-points per pass of S1: the configured batch, clamped so that the [Np][QB] phase table fits shared memory
  int s1_batch(int64_t nq, int *qb_out) {
    const int fit = rp_to_q_max_nq(np);
    if (fit == 0)
      return fail(EPW_EUNSUPPORTED, "Np = " + std::to_string(np) + " lattice vectors: the phase table of one q-point "
                                    "exceeds the shared memory of an SM (S1 supports Np <= 14080)");
    *qb_out = (int)std::min<int64_t>(std::min(q_batch, fit), nq);
    return EPW_OK;
  }
  // The convergence flag is STICKY: every eigensolve of every enqueued call may set it, only epw_interp_sync reads and
  // clears it, so a caller that enqueues several calls before one sync still learns of a failure in any of them.
  int ensure_status(cudaStream_t st) {
    if (status.p) return EPW_OK;
    cudaError_t e = status.reserve(sizeof(int32_t));
    // cleared ON the caller's stream (a blocking cudaMemset on the legacy stream is not ordered against a
    // cudaStreamNonBlocking stream) and waited for once, here, at allocation
    if (e == cudaSuccess) e = cudaMemsetAsync(status.p, 0, sizeof(int32_t), st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    return e == cudaSuccess ? EPW_OK : cuda_fail(e, "cudaMalloc status");
  }
  int cuda_fail(cudaError_t e, const char *where) {
    last_error = std::string(where) + ": " + cudaGetErrorString(e);
    return e == cudaErrorMemoryAllocation ? EPW_ENOMEM : EPW_ECUDA;
  }
  int begin_span(int stage, cudaStream_t st) {
    if (!timing) return -1;
    if (ev_used + 2 > ev_pool.size()) {
      const size_t old = ev_pool.size();
      ev_pool.resize(old + 64);
      for (size_t i = old; i < ev_pool.size(); i++) cudaEventCreate(&ev_pool[i]);
    }
    Span s{stage, (int)ev_used, (int)ev_used + 1, launches, 0};
    ev_used += 2;
    cudaEventRecord(ev_pool[s.e0], st);
    spans.push_back(s);
    return (int)spans.size() - 1;
  }
  void end_span(int id, cudaStream_t st) {
    if (id < 0) return;
    cudaEventRecord(ev_pool[spans[id].e1], st);
    spans[id].nlaunch = launches - spans[id].launch0;
  }
};

#define CU_OR_FAIL(h, expr, where)                        \
  do {                                                    \
    cudaError_t _e = (expr);                              \
    if (_e != cudaSuccess) return (h)->cuda_fail(_e, where); \
  } while (0)
#define LAUNCH(h, expr, where) \
  do {                         \
    (h)->launches++;           \
    CU_OR_FAIL(h, expr, where); \
  } while (0)


// The small-Nb kernels (pack_b_kernel, rotate_g2_small_kernel) keep a whole (k,q) pair in shared memory; beyond that
// (or when the caller asks for it) the large-Nb path of zgemm_strided.cu runs.
static bool use_large_path(const epw_interp *h) {
  if (h->cfg.path == EPW_PATH_SMALL) return false;
  if (h->cfg.path == EPW_PATH_LARGE) return true;
  return !rotate_g2_small_supported(h->nb, h->nm);
}

// ---------------------------------------------------------------------------------------------------------
// Large-Nb path (BASELINE.json configs[4]: Nb = 192, Nm = 288, g(Re,Rp) = 49 GB; Table III).
// Same stages, same order of the nested-loop algorithm, but S4a, S2 and both halves of S4b are
// FP64 tensor-path contractions that read their big operand in place (zgemm_strided.cu):
//   S4a  g^(Re,q) = g(Re,q) . e_q/sqrt(2 omega)       [Ne Nb^2 x Nm] . [Nm x Nm]            once per q
//   S2   g~(k,q)  = g^(Re,q)^T-contracted with P_k     [Nb^2 Nm x Ne] . [Ne x k-chunk]        per k-chunk
//   S4b  T = g~ U_k ;  |g|^2 = |T conj(U_{k+q})|^2      [Nm Nb x Nb] . [Nb x Nb], batched over the k of the chunk
// ---------------------------------------------------------------------------------------------------------
struct GridSpec;
static bool kside_matches(const epw_interp *h, const GridSpec *grid, bool need_conj, int path = EPW_PATH_LARGE);
static void kside_record(epw_interp *h, const GridSpec *grid, bool with_conj, int path = EPW_PATH_LARGE);
static void kside_wait(epw_interp *h, cudaStream_t st);

static int interpolate_large(epw_interp *h, const double *k_list, const GridSpec *grid, int64_t nk, const double *q_list,
                             int64_t nq, const int32_t *kq_map, double *eps_k, double *eps_kq, double *omega_q, double *g2,
                             cudaStream_t st) {
  const int nb = h->nb, nm = h->nm, ne = h->ne, np = h->np, nbb = h->nbb, nmm = h->nmm;
  const int64_t E = (int64_t)nbb * nm;        // elements per (k,q) pair
  if (!g2) CU_OR_FAIL(h, h->g2_scratch.reserve(sizeof(double) * (size_t)nk * E), "cudaMalloc |g|^2 scratch");
  double *const g2_base = g2 ? g2 : h->g2_scratch.as<double>();
  const int64_t g2_qs = g2 ? nk * E : 0;
  auto G2 = [&](int64_t q, int64_t k0) { return g2_base + q * g2_qs + k0 * E; };
  const int64_t xrows = (int64_t)ne * nbb;    // rows of the S4a contraction
  const int64_t MR = (int64_t)nm * nb;        // rows of the two S4b contractions
  const int KBe = (int)ceil_div(2 * (int64_t)ne, GEMM_BK), KBb = (int)ceil_div(2 * (int64_t)nb, GEMM_BK);
  const int KBm = (int)ceil_div(2 * (int64_t)nm, GEMM_BK);
  const int NTb = (int)ceil_div(2 * (int64_t)nb, GEMM_BN), NTm = (int)ceil_div(2 * (int64_t)nm, GEMM_BN);
  const int NTH = (int)ceil_div(2 * (int64_t)nbb, GEMM_BN);
  const int64_t NTk = ceil_div(nk, 64);
  const int64_t MTk = ceil_div(nk, GEMM_BM);
  const int64_t upack = (int64_t)NTb * KBb * GEMM_CHUNK;  // doubles of one packed Nb x Nb operand

  // q per pass over g(Re,Rp): g(Re,q) is 16 Nb^2 Nm Ne bytes per q here (2.9 GB for configs[4]); keep the batch <= 8 GB
  int QB = 1;
  { const int rc = h->s1_batch(nq, &QB); if (rc != EPW_OK) return rc; }
  {
    const size_t per_q = sizeof(c128) * (size_t)h->rows;
    QB = (int)std::max<int64_t>(1, std::min<int64_t>(QB, (int64_t)(((size_t)8 << 30) / per_q)));
  }
  // k per chunk: g~ and T are 16 E bytes per k each; whole 64-column tiles of the S2 contraction
  const size_t cap = h->cfg.workspace_bytes ? h->cfg.workspace_bytes : ((size_t)24 << 30);
  int64_t kc = (int64_t)(cap / (2 * sizeof(c128) * (size_t)E));
  if (kc >= nk) kc = nk;
  else if (kc >= 64) kc = kc / 64 * 64;
  else return h->fail(EPW_ENOMEM, "epw_interp_interpolate: workspace_bytes too small for one 64-k chunk of g~ and T");

  // S2 as the DMMA last-axis pass when the lattice-vector list is short and the columns split into groups of 64
  const bool s2_pass = E % 64 == 0 && E / 64 <= 2147483647LL && E <= 2147483647LL && grid_pass_dmma_supported(8, ne);
  CU_OR_FAIL(h, h->Apack.reserve(sizeof(double) * (size_t)MTk * KBe * GEMM_CHUNK), "cudaMalloc Apack");
  CU_OR_FAIL(h, h->BpackH.reserve(sizeof(double) * (size_t)NTH * KBe * GEMM_CHUNK), "cudaMalloc BpackH");
  CU_OR_FAIL(h, h->Hk.reserve(sizeof(c128) * (size_t)nk * nbb), "cudaMalloc Hk");
  CU_OR_FAIL(h, h->Uk.reserve(sizeof(c128) * (size_t)nk * nbb), "cudaMalloc Uk");
  CU_OR_FAIL(h, h->Pk.reserve(sizeof(c128) * (size_t)nk * ne), "cudaMalloc Pk");
  if (s2_pass) CU_OR_FAIL(h, h->PkT.reserve(sizeof(c128) * (size_t)nk * ne), "cudaMalloc PkT");
  CU_OR_FAIL(h, h->BpackPk.reserve(sizeof(double) * (size_t)NTk * KBe * GEMM_CHUNK), "cudaMalloc BpackPk");
  CU_OR_FAIL(h, h->UpackK.reserve(sizeof(double) * (size_t)nk * upack), "cudaMalloc UpackK");
  CU_OR_FAIL(h, h->UpackKH.reserve(sizeof(double) * (size_t)nk * upack), "cudaMalloc UpackKH");
  // the q side is small next to g: phases, D(q) and its eigen-system for ALL q of the call at once (a 288 x 288 solve
  // occupies one thread-block cluster; one at a time would leave the rest of the GPU idle)
  CU_OR_FAIL(h, h->Pq.reserve(sizeof(c128) * (size_t)nq * np), "cudaMalloc Pq");
  CU_OR_FAIL(h, h->Dq.reserve(sizeof(c128) * (size_t)nq * nmm), "cudaMalloc Dq");
  CU_OR_FAIL(h, h->eq.reserve(sizeof(c128) * (size_t)nq * nmm), "cudaMalloc e_q");
  if (!h->ext_g1) CU_OR_FAIL(h, h->g1.reserve(sizeof(c128) * (size_t)QB * h->rows), "cudaMalloc g(Re,q)");
  CU_OR_FAIL(h, h->BpackE.reserve(sizeof(double) * (size_t)NTm * KBm * GEMM_CHUNK), "cudaMalloc BpackE");
  CU_OR_FAIL(h, h->ghat.reserve(sizeof(c128) * (size_t)ne * E), "cudaMalloc g^(Re,q)");
  CU_OR_FAIL(h, h->C.reserve(sizeof(c128) * (size_t)kc * E), "cudaMalloc g~");
  CU_OR_FAIL(h, h->T.reserve(sizeof(c128) * (size_t)kc * E), "cudaMalloc T");
  if (!kq_map) {
    CU_OR_FAIL(h, h->Pqe.reserve(sizeof(c128) * (size_t)nq * ne), "cudaMalloc Pqe");
    CU_OR_FAIL(h, h->Hkq.reserve(sizeof(c128) * (size_t)nk * nbb), "cudaMalloc Hkq");
    CU_OR_FAIL(h, h->Ukq.reserve(sizeof(c128) * (size_t)nk * nbb), "cudaMalloc Ukq");
    if (!eps_kq) CU_OR_FAIL(h, h->epskq_scratch.reserve(sizeof(double) * (size_t)nk * nb), "cudaMalloc eps scratch");
  }
  { const int rc = h->ensure_status(st); if (rc != EPW_OK) return rc; }
  if (h->window_on && !h->mask_out) CU_OR_FAIL(h, h->maskbuf.reserve((size_t)nk), "cudaMalloc mask");
  {
    const size_t need = std::max(eigh_large_scratch_bytes(nb, nk), eigh_large_scratch_bytes(nm, nq));
    if (need) CU_OR_FAIL(h, h->eig_scratch.reserve(need), "cudaMalloc eig scratch");
  }
  h->last_nk = nk;
  h->last_c_rows = kc;
  h->last_ncols = (int)E;
  h->last_path = EPW_PATH_LARGE;
  h->last_eq_slot = nq - 1;
  h->last_qb = QB;
  h->last_kchunk = kc;

  const int t_total = h->begin_span(7, st);

  // ---- k side: phases, H(k) (same DMMA contraction as the small path), eigensolve, packed U_k.  Once per call -- or, when
  //      the k-points are the uniform grid of the previous call and the operators have not changed, not at all: every
  //      buffer below is still valid (configs[4]: 200 cluster eigensolves of 192 x 192 = 13 % of a 2-q call) ----
  int sp;
  const bool k_cached = kside_matches(h, grid, kq_map != nullptr);
  if (k_cached) {
    kside_wait(h, st);
    CU_OR_FAIL(h, cudaMemcpyAsync(eps_k, h->epsk_keep.p, sizeof(double) * (size_t)nk * nb, cudaMemcpyDeviceToDevice, st),
               "copy cached eps_k");
  } else {
  h->kside.valid = false;
  sp = h->begin_span(0, st);
  LAUNCH(h, launch_phase_pack_a(k_list, nk, h->Re.as<int32_t>(), h->we.as<double>(), ne, h->Apack.as<double>(), st),
         "phase_pack_a");
  LAUNCH(h, launch_phase_table(k_list, nk, h->Re.as<int32_t>(), h->we.as<double>(), ne, h->Pk.as<c128>(), st),
         "phase_table(k,Re)");
  LAUNCH(h, launch_pack_b_strided(h->Pk.as<c128>(), 1, ne, 0, 1, 0, nullptr, 0.0, ne, (int)nk, h->BpackPk.as<double>(), st),
         "pack P_k");
  if (s2_pass) {
    h->launches++;
    transpose_blocks_kernel<<<grid_cap(ceil_div(nk * ne, 256), 8), 256, 0, st>>>(h->Pk.as<c128>(), nk, ne, kc, h->PkT.as<c128>());
    CU_OR_FAIL(h, cudaGetLastError(), "transpose P_k");
  }
  h->end_span(sp, st);
  sp = h->begin_span(3, st);
  LAUNCH(h,
         launch_pack_b(nullptr, nullptr, nullptr, 0.0, h->H.as<c128>(), nullptr, nbb, nm, ne, 0, nbb,
                       h->BpackH.as<double>(), st),
         "pack_b(H)");
  LAUNCH(h, launch_zgemm_dmma(h->Apack.as<double>(), h->BpackH.as<double>(), h->Hk.as<c128>(), nk, nbb, KBe, nbb,
                              h->num_sms, st),
         "zgemm H(k)");
  LAUNCH(h, launch_eigh_batched(h->Hk.as<c128>(), nbb, nb, nk, eps_k, h->Uk.as<c128>(), 0, h->status.as<int32_t>(),
                                h->eig_scratch.as<c128>(), h->work_slot(0), st),
         "eigh H(k)");
  LAUNCH(h, launch_pack_b_strided(h->Uk.as<c128>(), 1, nb, nbb, nk, 0, nullptr, 0.0, nb, nb, h->UpackK.as<double>(), st),
         "pack U_k");
  if (kq_map)
    LAUNCH(h, launch_pack_b_strided(h->Uk.as<c128>(), 1, nb, nbb, nk, 1, nullptr, 0.0, nb, nb, h->UpackKH.as<double>(), st),
           "pack conj U_k");
  h->end_span(sp, st);
  if (grid) {
    CU_OR_FAIL(h, h->epsk_keep.reserve(sizeof(double) * (size_t)nk * nb), "cudaMalloc eps_k cache");
    CU_OR_FAIL(h, cudaMemcpyAsync(h->epsk_keep.p, eps_k, sizeof(double) * (size_t)nk * nb, cudaMemcpyDeviceToDevice, st),
               "keep eps_k");
    kside_record(h, grid, kq_map != nullptr);
  }
  }

  // ---- q side, once per call ----
  sp = h->begin_span(0, st);
  LAUNCH(h, launch_phase_table(q_list, nq, h->Rp.as<int32_t>(), h->wp.as<double>(), np, h->Pq.as<c128>(), st),
         "phase_table(q,Rp)");
  if (!kq_map)
    LAUNCH(h, launch_phase_table(q_list, nq, h->Re.as<int32_t>(), h->ones.as<double>(), ne, h->Pqe.as<c128>(), st),
           "phase_table(q,Re)");
  h->end_span(sp, st);
  // D(q) and the phonon eigensolves go to the second stream; the caller's stream joins it before the first mode rotation
  if (!h->aux_stream) {
    CU_OR_FAIL(h, cudaStreamCreateWithFlags(&h->aux_stream, cudaStreamNonBlocking), "cudaStreamCreate");
    CU_OR_FAIL(h, cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming), "cudaEventCreate");
    CU_OR_FAIL(h, cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming), "cudaEventCreate");
  }
  CU_OR_FAIL(h, cudaEventRecord(h->ev_fork, st), "cudaEventRecord");
  CU_OR_FAIL(h, cudaStreamWaitEvent(h->aux_stream, h->ev_fork, 0), "cudaStreamWaitEvent");
  LAUNCH(h, launch_interp_operator(h->D.as<c128>(), nm, np, h->Pq.as<c128>(), nq, h->Dq.as<c128>(), h->aux_stream), "D(q)");
  LAUNCH(h, launch_eigh_batched(h->Dq.as<c128>(), nmm, nm, nq, omega_q, h->eq.as<c128>(), 1, h->status.as<int32_t>(),
                                h->eig_scratch.as<c128>(), h->work_slot(2), h->aux_stream),
         "eigh D(q)");
  CU_OR_FAIL(h, cudaEventRecord(h->ev_join, h->aux_stream), "cudaEventRecord");
  bool joined = false;

  for (int64_t q0 = 0; q0 < nq; q0 += QB) {
    const int qb = (int)std::min<int64_t>(QB, nq - q0);
    const c128 *Pq_b = h->Pq.as<c128>() + q0 * np, *Pqe_b = h->Pqe.as<c128>() + q0 * ne, *eq_b = h->eq.as<c128>() + q0 * nmm;
    sp = h->begin_span(1, st);
    const c128 *g1b = h->ext_g1 ? h->ext_g1 + q0 * h->rows : h->g1.as<c128>();
    if (!h->ext_g1)
      LAUNCH(h, launch_rp_to_q(h->g.as<c128>(), h->rows, np, Pq_b, qb, h->g1.as<c128>(), st), "rp_to_q");
    h->end_span(sp, st);
    if (!joined) {
      sp = h->begin_span(2, st);   // what is left of the phonon side once the first S1 pass is done
      CU_OR_FAIL(h, cudaStreamWaitEvent(st, h->ev_join, 0), "cudaStreamWaitEvent");
      h->end_span(sp, st);
      joined = true;
    }

    for (int iq = 0; iq < qb; iq++) {
      const int64_t q = q0 + iq;
      // ---- S4a (hoisted): g^(Re,q)[Re][nu][n'][m'] = sum_ka g(Re,q)[ka][Re][n'][m'] e_q[ka][nu] / sqrt(2 omega_nu) ----
      sp = h->begin_span(8, st);
      LAUNCH(h, launch_pack_b_strided(eq_b + (int64_t)iq * nmm, 1, nm, 0, 1, 0, omega_q + q * nm,
                                      h->cfg.omega_min, nm, nm, h->BpackE.as<double>(), st),
             "pack e_q");
      LAUNCH(h, launch_zgemm_strided(g1b + (int64_t)iq * h->rows, xrows, 0, xrows, 0,
                                     h->BpackE.as<double>(), nullptr, h->ghat.p, nbb, E, 1, nbb, 0, 0, xrows, nm, nm, 1,
                                     h->num_sms, st),
             "zgemm S4a");
      h->end_span(sp, st);
      const double *Bconj = h->UpackKH.as<double>();
      if (!kq_map) {
        // ---- off-grid q: H(k+q) for every k, eigensolve, packed conj(U_{k+q}) ----
        sp = h->begin_span(5, st);
        LAUNCH(h,
               launch_pack_b(nullptr, nullptr, nullptr, 0.0, h->H.as<c128>(), Pqe_b + (int64_t)iq * ne, nbb,
                             nm, ne, 0, nbb, h->BpackH.as<double>(), st),
               "pack_b(H e^{iqR})");
        LAUNCH(h, launch_zgemm_dmma(h->Apack.as<double>(), h->BpackH.as<double>(), h->Hkq.as<c128>(), nk, nbb, KBe, nbb,
                                    h->num_sms, st),
               "zgemm H(k+q)");
        double *eps_dst = eps_kq ? eps_kq + q * nk * nb : h->epskq_scratch.as<double>();
        LAUNCH(h, launch_eigh_batched(h->Hkq.as<c128>(), nbb, nb, nk, eps_dst, h->Ukq.as<c128>(), 0,
                                      h->status.as<int32_t>(), h->eig_scratch.as<c128>(), h->work_slot(1), st),
               "eigh H(k+q)");
        LAUNCH(h, launch_pack_b_strided(h->Ukq.as<c128>(), 1, nb, nbb, nk, 1, nullptr, 0.0, nb, nb,
                                        h->UpackKH.as<double>(), st),
               "pack conj U_{k+q}");
        h->kside.with_conj = false;   // the packed conj(U_k) of a kq_map call is gone
        h->end_span(sp, st);
      } else if (eps_kq) {
        sp = h->begin_span(5, st);
        h->launches++;
        gather_eps_kernel<<<grid_cap(ceil_div(nk * nb, 256), 8), 256, 0, st>>>(
            eps_k, kq_map + q * nk, nb, nk, eps_kq + q * nk * nb);
        CU_OR_FAIL(h, cudaGetLastError(), "gather_eps");
        h->end_span(sp, st);
      }
      for (int64_t k0 = 0; k0 < nk; k0 += kc) {
        const int64_t kn = std::min(kc, nk - k0);
        // ---- S2: g~[k][nu][n'][m'] = sum_Re g^[Re][nu][n'][m'] P_k[k][Re] ----
        sp = h->begin_span(4, st);
        if (s2_pass)
          // few lattice vectors (a ribbon: Ne = 17): g~ = sum_Re g^(Re) P_k as the last-axis DMMA pass of grid_fused.cuh on
          // column groups of 64 -- K = 2 Ne real exactly (the tiled contraction pads 34 to 48) and the 34 GB of g~ per q
          // stream out of 16 warps per SM: 11 instead of 22 ms per q on configs[4]
          LAUNCH(h, launch_grid_pass_dmma(h->ghat.as<c128>(), 1, (int)E, ne, h->PkT.as<c128>() + k0 * ne, (int)kn, 8,
                                          (int)(E / 64), h->num_sms, h->C.as<c128>(), E, 1, 0, 0, st),
                 "S2 (DMMA pass)");
        else
        LAUNCH(h, launch_zgemm_strided(h->ghat.as<c128>(), E, 0, E, 0,
                                       h->BpackPk.as<double>() + (k0 / 64) * (int64_t)KBe * GEMM_CHUNK, nullptr, h->C.p, E, 0,
                                       1, E, 0, 0, E, (int)kn, ne, 1, h->num_sms, st),
               "zgemm S2");
        h->end_span(sp, st);
        // ---- S4b: T[k][nu][m'][n] = sum_n' g~[k][nu][n'][m'] U_k[n'][n];  |g|^2[k][nu][n][m] = |sum_m' T conj(U_{k+q}[m'][m])|^2 ----
        sp = h->begin_span(6, st);
        LAUNCH(h, launch_zgemm_strided(h->C.as<c128>(), nb, nbb, nb, E, h->UpackK.as<double>() + k0 * upack, nullptr,
                                       h->T.p, MR, 0, nb, 1, E, 0, MR, nb, nb, kn, h->num_sms, st),
               "zgemm S4b (U_k)");
        LAUNCH(h, launch_zgemm_strided(h->T.as<c128>(), nb, nbb, nb, E, kq_map ? Bconj : Bconj + k0 * upack,
                                       kq_map ? kq_map + q * nk + k0 : nullptr, G2(q, k0), MR, 0, nb, 1, E,
                                       1, MR, nb, nb, kn, h->num_sms, st),
               "zgemm S4b (U_{k+q}) + |g|^2");
        if (h->window_on) {
          // the in-place contractions of this kernel family cannot skip pairs: screened pairs are zeroed afterwards
          uint8_t *m = (h->mask_out ? h->mask_out + q * nk : h->maskbuf.as<uint8_t>()) + k0;
          const double *ekq = kq_map ? nullptr : (eps_kq ? eps_kq + (q * nk + k0) * nb : h->epskq_scratch.as<double>() + k0 * nb);
          LAUNCH(h, launch_window_mask(eps_k + k0 * nb, ekq, eps_k, kq_map ? kq_map + q * nk + k0 : nullptr, nb, kn, h->emin,
                                       h->emax, m, st), "window mask");
          LAUNCH(h, launch_zero_masked(m, kn, E, G2(q, k0), st), "zero screened pairs");
        }
        if (h->cons.on) {
          const double *ekq = kq_map ? nullptr : (eps_kq ? eps_kq + (q * nk + k0) * nb : h->epskq_scratch.as<double>() + k0 * nb);
          LAUNCH(h, launch_selfenergy_accumulate(G2(q, k0), eps_k + k0 * nb, ekq, eps_k, kq_map ? kq_map + q * nk + k0 : nullptr,
                                                 omega_q + q * nm, h->cons.w_q, q, h->cons.mu, h->cons.kT, h->cons.sigma, nb,
                                                 nm, kn, h->cons.out + k0 * nb, st),
                 "Im Sigma accumulate");
        }
        h->end_span(sp, st);
      }
      if (g2) { const int rc = h->drain_q(q, nk, E, g2, eps_kq, st); if (rc != EPW_OK) return rc; }
    }
  }
  h->end_span(t_total, st);
  return EPW_OK;
}

// Uniform k-grid handed to the small-Nb path instead of a k-list (epw_interp_interpolate_grid).
struct GridSpec {
  int32_t N[3];
  double s[3];
};

static int interpolate_small(epw_interp *h, const double *k_list, const GridSpec *grid, int64_t nk, const double *q_list,
                             int64_t nq, const int32_t *kq_map, double *eps_k, double *eps_kq, double *omega_q,
                             double *g2, cudaStream_t st);

static bool kside_matches(const epw_interp *h, const GridSpec *grid, bool need_conj, int path) {
  if (!grid || !h->kside.valid || h->kside.epoch != h->op_epoch || h->kside.path != path) return false;
  for (int d = 0; d < 3; d++)
    if (h->kside.N[d] != grid->N[d] || h->kside.s[d] != grid->s[d]) return false;
  return h->kside.with_conj || !need_conj;
}
// A cache hit on a stream other than the one the k side was computed on: make that stream wait for the cached buffers.
static void kside_wait(epw_interp *h, cudaStream_t st) {
  if (h->kside.ev && h->kside.stream != st) cudaStreamWaitEvent(st, h->kside.ev, 0);
}
static void kside_record(epw_interp *h, const GridSpec *grid, bool with_conj, int path) {
  if (!h->kside.ev && cudaEventCreateWithFlags(&h->kside.ev, cudaEventDisableTiming) != cudaSuccess) {
    h->kside.ev = nullptr;
    cudaGetLastError();
    h->kside.valid = false;   // no event, no cache: every call recomputes the k side
    return;
  }
  h->kside.stream = h->last_stream;
  cudaEventRecord(h->kside.ev, h->last_stream);   // behind the last kernel / copy of the k side
  h->kside.valid = true;
  h->kside.path = path;
  h->kside.with_conj = with_conj;
  h->kside.epoch = h->op_epoch;
  for (int d = 0; d < 3; d++) {
    h->kside.N[d] = grid->N[d];
    h->kside.s[d] = grid->s[d];
  }
}

extern "C" {

const char *epw_version(void) { return "epw-interp-b200 0.1 (sm_100a, FP64 DMMA)"; }

const char *epw_interp_last_error(epw_interp_t h) { return h ? h->last_error.c_str() : g_create_error.c_str(); }

int epw_interp_create(epw_interp_t *out, const epw_interp_config *cfg) {
  if (!out) return EPW_EINVAL;
  *out = nullptr;
  if (!cfg || cfg->nbnd <= 0 || cfg->nmodes <= 0 || cfg->ne <= 0 || cfg->np <= 0) {
    g_create_error = "epw_interp_create: nbnd, nmodes, ne, np must be positive";
    return EPW_EINVAL;
  }
  if (cfg->path < EPW_PATH_AUTO || cfg->path > EPW_PATH_LARGE) {
    g_create_error = "epw_interp_create: path must be EPW_PATH_AUTO, EPW_PATH_SMALL or EPW_PATH_LARGE";
    return EPW_EINVAL;
  }
  if ((cfg->flags & ~(EPW_FLAG_GRID_UNFUSED | EPW_FLAG_GRID_FUSED)) ||
      cfg->flags == (EPW_FLAG_GRID_UNFUSED | EPW_FLAG_GRID_FUSED)) {
    g_create_error = "epw_interp_create: unknown bit in flags";
    return EPW_EINVAL;
  }
  if (!(cfg->omega_min >= 0.0)) {   // also rejects NaN
    g_create_error = "epw_interp_create: omega_min must be >= 0 (a negative cut-off would let soft modes into 1/sqrt(2 omega))";
    return EPW_EINVAL;
  }
  if (cfg->q_batch < 0 || cfg->q_batch > 8) {
    g_create_error = "epw_interp_create: q_batch must be in 0..8";
    return EPW_EINVAL;
  }
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || cfg->device < 0 || cfg->device >= ndev) {
    g_create_error = std::string("epw_interp_create: no usable CUDA device (") +
                     (e != cudaSuccess ? cudaGetErrorString(e) : "bad ordinal") + "); there is no CPU fallback";
    return EPW_ECUDA;
  }
  cudaDeviceProp prop;
  if (cudaSetDevice(cfg->device) != cudaSuccess || cudaGetDeviceProperties(&prop, cfg->device) != cudaSuccess) {
    g_create_error = "epw_interp_create: cudaSetDevice failed";
    return EPW_ECUDA;
  }
  if (prop.major != 10) {
    g_create_error = "epw_interp_create: this library is built for sm_100a (Blackwell B200) only";
    return EPW_ECUDA;
  }
  epw_interp *h = new (std::nothrow) epw_interp();
  if (!h) return EPW_ENOMEM;
  h->cfg = *cfg;
  h->nb = cfg->nbnd;
  h->nm = cfg->nmodes;
  h->ne = cfg->ne;
  h->np = cfg->np;
  h->nbb = h->nb * h->nb;
  h->nmm = h->nm * h->nm;
  h->rows = (int64_t)h->nbb * h->ne * h->nm;
  h->num_sms = prop.multiProcessorCount;
  h->q_batch = cfg->q_batch > 0 ? cfg->q_batch : 8;
  h->slab_set.assign(h->np, 0);
  h->rp_cnt = h->np;
  *out = h;
  return EPW_OK;
}

void epw_interp_destroy(epw_interp_t h) {
  if (!h) return;
  cudaSetDevice(h->cfg.device);
  cudaDeviceSynchronize();   // kernels of this handle may still be reading its buffers
  DevBuf *all[] = {&h->g, &h->H, &h->D, &h->Re, &h->Rp, &h->we, &h->wp, &h->ones, &h->Apack, &h->BpackH, &h->Hk,
                   &h->Uk, &h->Pq, &h->Pqe, &h->Dq, &h->eq, &h->g1, &h->Bpack, &h->C, &h->Ukq, &h->epskq_scratch,
                   &h->status, &h->eig_scratch, &h->hs_k, &h->hs_q, &h->hs_map, &h->hs_epsk, &h->hs_epskq,
                   &h->hs_omega, &h->hs_g2, &h->epsk_keep, &h->dst_tab, &h->PkT, &h->Pk, &h->BpackPk, &h->UpackK, &h->UpackKH, &h->BpackE,
                   &h->ghat, &h->T, &h->Hkq, &h->boxidx, &h->X, &h->T1, &h->T2, &h->Ptmp, &h->P1raw, &h->P2raw, &h->P3raw, &h->P1pack, &h->P2pack,
                   &h->P3pack, &h->klist_gen, &h->workctr, &h->maskbuf, &h->g2_scratch};
  for (DevBuf *b : all) b->release();
  for (cudaEvent_t ev : h->ev_pool) cudaEventDestroy(ev);
  for (cudaEvent_t ev : h->sink_ev) cudaEventDestroy(ev);
  if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
  if (h->aux_stream) cudaStreamDestroy(h->aux_stream);
  if (h->ev_fork) cudaEventDestroy(h->ev_fork);
  if (h->ev_join) cudaEventDestroy(h->ev_join);
  if (h->kside.ev) cudaEventDestroy(h->kside.ev);
  delete h;
}

int epw_interp_set_g_slabs(epw_interp_t h, int32_t ip_start, int32_t ip_count, const void *g_slabs, int on_device) {
  if (!h) return EPW_EINVAL;
  if (!g_slabs || ip_start < h->rp_lo || ip_count <= 0 || ip_start + ip_count > h->rp_lo + h->rp_cnt)
    return h->fail(EPW_EINVAL, "epw_interp_set_g_slabs: bad slab range (outside this handle's Rp shard) or null pointer");
  CU_OR_FAIL(h, cudaSetDevice(h->cfg.device), "cudaSetDevice");
  const size_t total = (size_t)h->rows * h->rp_cnt * sizeof(c128);
  CU_OR_FAIL(h, h->g.reserve(total), "cudaMalloc g(Re,Rp)");
  const size_t slab = (size_t)h->rows * sizeof(c128);
  CU_OR_FAIL(h,
             cudaMemcpy(h->g.as<char>() + slab * (ip_start - h->rp_lo), g_slabs, slab * ip_count,
                        on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice),
             "cudaMemcpy g slabs");
  for (int i = 0; i < ip_count; i++) h->slab_set[ip_start + i] = 1;
  return EPW_OK;
}

int epw_interp_set_wannier_operators(epw_interp_t h, const void *H_R, const void *D_R, const void *g_RR,
                                     const int32_t *Re, const double *w_e, const int32_t *Rp, const double *w_p,
                                     int on_device) {
  if (!h) return EPW_EINVAL;
  if (!H_R || !D_R || !Re || !w_e || !Rp || !w_p)
    return h->fail(EPW_EINVAL, "epw_interp_set_wannier_operators: null operator pointer");
  CU_OR_FAIL(h, cudaSetDevice(h->cfg.device), "cudaSetDevice");
  const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  struct Item { DevBuf *buf; const void *src; size_t bytes; };
  const Item items[] = {{&h->H, H_R, sizeof(c128) * (size_t)h->nbb * h->ne},
                        {&h->D, D_R, sizeof(c128) * (size_t)h->nmm * h->np},
                        {&h->Re, Re, sizeof(int32_t) * 3 * (size_t)h->ne},
                        {&h->we, w_e, sizeof(double) * (size_t)h->ne},
                        {&h->Rp, Rp, sizeof(int32_t) * 3 * (size_t)h->np},
                        {&h->wp, w_p, sizeof(double) * (size_t)h->np}};
  for (const Item &it : items) {
    CU_OR_FAIL(h, it.buf->reserve(it.bytes), "cudaMalloc operators");
    CU_OR_FAIL(h, cudaMemcpy(it.buf->p, it.src, it.bytes, kind), "cudaMemcpy operators");
  }
  {
    // bounding box of the Re list and the position of every vector inside it (uniform-grid form of S2)
    std::vector<int32_t> re(3 * (size_t)h->ne), idx(h->ne);
    CU_OR_FAIL(h, cudaMemcpy(re.data(), h->Re.p, sizeof(int32_t) * re.size(), cudaMemcpyDeviceToHost), "cudaMemcpy Re");
    int hi[3];
    for (int d = 0; d < 3; d++) h->box_lo[d] = hi[d] = re[d];
    for (int i = 0; i < h->ne; i++)
      for (int d = 0; d < 3; d++) {
        h->box_lo[d] = std::min(h->box_lo[d], (int)re[3 * i + d]);
        hi[d] = std::max(hi[d], (int)re[3 * i + d]);
      }
    h->box_size = 1;
    for (int d = 0; d < 3; d++) {
      h->box_L[d] = hi[d] - h->box_lo[d] + 1;
      h->box_size *= h->box_L[d];
    }
    for (int i = 0; i < h->ne; i++)
      idx[i] = ((re[3 * i] - h->box_lo[0]) * h->box_L[1] + (re[3 * i + 1] - h->box_lo[1])) * h->box_L[2] +
               (re[3 * i + 2] - h->box_lo[2]);
    CU_OR_FAIL(h, h->boxidx.reserve(sizeof(int32_t) * (size_t)h->ne), "cudaMalloc box index");
    CU_OR_FAIL(h, cudaMemcpy(h->boxidx.p, idx.data(), sizeof(int32_t) * (size_t)h->ne, cudaMemcpyHostToDevice),
               "cudaMemcpy box index");
  }
  const int nmax = std::max(h->ne, h->np);
  CU_OR_FAIL(h, h->ones.reserve(sizeof(double) * nmax), "cudaMalloc ones");
  fill_ones_kernel<<<(nmax + 255) / 256, 256>>>(h->ones.as<double>(), nmax);
  CU_OR_FAIL(h, cudaDeviceSynchronize(), "fill_ones");
  h->operators_set = true;
  h->op_epoch++;
  h->kside.valid = false;
  if (g_RR) {
    // g_RR holds every slab; a sharded handle keeps its own range only
    const char *src = reinterpret_cast<const char *>(g_RR) + (size_t)h->rows * sizeof(c128) * h->rp_lo;
    return epw_interp_set_g_slabs(h, h->rp_lo, h->rp_cnt, src, on_device);
  }
  return EPW_OK;
}

int epw_interp_enable_stage_timing(epw_interp_t h, int on) {
  if (!h) return EPW_EINVAL;
  h->timing = on != 0;
  h->spans.clear();  // (re)enabling starts a fresh accumulation
  h->ev_used = 0;
  if (h->timing) {
    CU_OR_FAIL(h, cudaSetDevice(h->cfg.device), "cudaSetDevice");
    CU_OR_FAIL(h, h->workctr.reserve(3 * sizeof(unsigned long long)), "cudaMalloc work counters");
    CU_OR_FAIL(h, cudaMemset(h->workctr.p, 0, 3 * sizeof(unsigned long long)), "memset work counters");
  }
  return EPW_OK;
}

static int check_interpolate_args(epw_interp *h, const void *k_src, int64_t nk, const double *q_list, int64_t nq,
                                  const double *eps_k, const double *omega_q, const double *g2, const char *who) {
  if (!k_src || !q_list || !eps_k || !omega_q || (!g2 && !h->cons.on) || nk <= 0 || nq <= 0)
    return h->fail(EPW_EINVAL, std::string(who) + ": null pointer or non-positive nk/nq");
  if (!h->operators_set) return h->fail(EPW_EINVAL, std::string(who) + ": operators not set");
  if (!h->ext_g1) {
    if (h->sharded)
      return h->fail(EPW_EINVAL, std::string(who) + ": this handle holds an Rp shard of g(Re,Rp); use "
                                                   "epw_interp_rp_to_q_partial + an all-reduce + epw_interp_set_gq");
    for (int ip = 0; ip < h->np; ip++)
      if (!h->slab_set[ip]) return h->fail(EPW_EINVAL, std::string(who) + ": g(Re,Rp) slab missing");
  }
  return EPW_OK;
}

int epw_interp_interpolate(epw_interp_t h, const double *k_list, int64_t nk, const double *q_list, int64_t nq,
                           const int32_t *kq_map, double *eps_k, double *eps_kq, double *omega_q, double *g2,
                           void *cuda_stream) {
  if (!h) return EPW_EINVAL;
  const int rc = check_interpolate_args(h, k_list, nk, q_list, nq, eps_k, omega_q, g2, "epw_interp_interpolate");
  if (rc != EPW_OK) return rc;
  CU_OR_FAIL(h, cudaSetDevice(h->cfg.device), "cudaSetDevice");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  h->last_stream = st;
  h->launches = 0;
  h->last_kmode = 0;
  const int rc2 = use_large_path(h)
                      ? interpolate_large(h, k_list, nullptr, nk, q_list, nq, kq_map, eps_k, eps_kq, omega_q, g2, st)
                      : interpolate_small(h, k_list, nullptr, nk, q_list, nq, kq_map, eps_k, eps_kq, omega_q, g2, st);
  if (rc2 != EPW_OK) h->kside.valid = false;   // a call that failed half-way leaves no cached k side behind
  return rc2;
}

int epw_interp_interpolate_grid(epw_interp_t h, const int32_t *k_grid, const double *k_shift, const double *q_list,
                                int64_t nq, const int32_t *kq_map, double *eps_k, double *eps_kq, double *omega_q,
                                double *g2, void *cuda_stream) {
  if (!h) return EPW_EINVAL;
  if (!k_grid || k_grid[0] <= 0 || k_grid[1] <= 0 || k_grid[2] <= 0)
    return h->fail(EPW_EINVAL, "epw_interp_interpolate_grid: k_grid must hold three positive sizes");
  GridSpec g;
  for (int d = 0; d < 3; d++) {
    g.N[d] = k_grid[d];
    g.s[d] = k_shift ? k_shift[d] : 0.0;
  }
  const int64_t nk = (int64_t)g.N[0] * g.N[1] * g.N[2];
  const int rc = check_interpolate_args(h, k_grid, nk, q_list, nq, eps_k, omega_q, g2, "epw_interp_interpolate_grid");
  if (rc != EPW_OK) return rc;
  CU_OR_FAIL(h, cudaSetDevice(h->cfg.device), "cudaSetDevice");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  h->last_stream = st;
  h->launches = 0;
  if (use_large_path(h)) {
    // the large-Nb kernels take a k-list (their grids are one-dimensional: nothing to factorise)
    h->last_kmode = 0;
    CU_OR_FAIL(h, h->klist_gen.reserve(sizeof(double) * 3 * (size_t)nk), "cudaMalloc k-list");
    if (!kside_matches(h, &g, kq_map != nullptr))
      LAUNCH(h, launch_grid_klist(g.N, g.s, h->klist_gen.as<double>(), st), "grid k-list");
    const int rl = interpolate_large(h, h->klist_gen.as<double>(), &g, nk, q_list, nq, kq_map, eps_k, eps_kq, omega_q, g2, st);
    if (rl != EPW_OK) h->kside.valid = false;
    return rl;
  }
  h->last_kmode = 1;
  const int rs = interpolate_small(h, nullptr, &g, nk, q_list, nq, kq_map, eps_k, eps_kq, omega_q, g2, st);
  if (rs != EPW_OK) h->kside.valid = false;   // a call that failed half-way leaves no cached k side behind
  return rs;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------
// Small-Nb path (Nb <= 16; BASELINE.json configs[0..3]).  k-points come either as a list (dense S2: one FP64
// tensor-path contraction over all Re, zgemm_dmma.cu) or as a uniform grid (factorised S2: one contraction per
// crystal axis, re_to_k_grid.cu); everything after S2 is shared.
// ---------------------------------------------------------------------------------------------------------
static int interpolate_small(epw_interp *h, const double *k_list, const GridSpec *grid, int64_t nk, const double *q_list,
                             int64_t nq, const int32_t *kq_map, double *eps_k, double *eps_kq, double *omega_q,
                             double *g2, cudaStream_t st) {
  const int nb = h->nb, nm = h->nm, ne = h->ne, np = h->np, nbb = h->nbb, nmm = h->nmm;
  // (the two kernel families share the H(k), U_k buffers: a cached k side is valid for the family that made it; on a
  //  uniform grid the small-Nb family keeps U_k and eps_k between calls too -- 10^6 solves per call on configs[3])
  const bool k_cached = kside_matches(h, grid, false, EPW_PATH_SMALL);
  if (k_cached) kside_wait(h, st);
  else h->kside.valid = false;
  const int ncols_g = nbb * nm;
  const int ncols_h = kq_map ? 0 : nbb;
  const int ncols = ncols_g + ncols_h;
  const int KB = (int)ceil_div(2 * (int64_t)ne, GEMM_BK);
  const int NT = (int)ceil_div(2 * (int64_t)ncols, GEMM_BN);
  const int NTH = (int)ceil_div(2 * (int64_t)nbb, GEMM_BN);
  const int64_t MT = ceil_div(nk, GEMM_BM);
  int QB = 1;
  { const int rc = h->s1_batch(nq, &QB); if (rc != EPW_OK) return rc; }
  const int64_t E = (int64_t)ncols_g;
  const size_t cap = h->cfg.workspace_bytes ? h->cfg.workspace_bytes : ((size_t)6 << 30);
  // |g|^2 of pair (q, k0..): the caller's buffer, or (consumer on, g2 = NULL) the library's one-q scratch -- or nothing at
  // all when the consumer is folded into the one-kernel grid form (see below)
  double *g2_base = g2;
  const int64_t g2_qs = g2 ? nk * E : 0;
  auto G2 = [&](int64_t q, int64_t k0) { return g2_base ? g2_base + q * g2_qs + k0 * E : nullptr; };

  int64_t kchunk, c_rows;
  int hbatch = 0;            // grid mode, one-kernel form: q-points whose H(k+q) side is taken in one go (0 = per q)
  // grid mode: extents of the three axis passes (re_to_k_grid.cu)
  const int *L = h->box_L;
  int64_t slab = 0;          // k-points per i1 plane
  int cs = 0, nchunks = 1;   // i1 planes per k-chunk
  int KB1 = 0, NTc = 0;
  // grid mode: the last axis pass, S4b and |g|^2 run as ONE all-DMMA kernel (grid_fused.cu; g~ never reaches HBM) for
  // Nb <= 8, where the U fragments of four pairs stay in registers: measured (bench.py --grid-fused / --grid-unfused)
  // 16.7 vs 18.8 ms per 32-q step on configs[1] and 91 vs 110 ms per 13-q step on configs[3].  For 9 <= Nb <= 16 the fused
  // kernel reloads its U fragments per mode and is no faster than the two-kernel form (21.0 vs 20.7 ms on configs[2]),
  // which stays the default there.  EPW_FLAG_GRID_FUSED / EPW_FLAG_GRID_UNFUSED force either form.
  const bool can_fuse = grid && grid_fused_supported(nb, nm, h->box_L[0]);
  const bool fused = can_fuse && ((h->cfg.flags & EPW_FLAG_GRID_FUSED) != 0 ||
                                  (nb <= 8 && (h->cfg.flags & EPW_FLAG_GRID_UNFUSED) == 0));
  if (!g2 && !fused) {
    CU_OR_FAIL(h, h->g2_scratch.reserve(sizeof(double) * (size_t)nk * E), "cudaMalloc |g|^2 scratch");
    g2_base = h->g2_scratch.as<double>();
  }
  int ncolsC = fused ? ncols_h : ncols;   // columns of the [g~ | H(k+q)] buffer that reach HBM (hbatch: g~ only, see below)
  if (!grid) {
    // k-chunk: one chunk of [g~ | H(k+q)] (16*ncols bytes per k) must stay L2-resident for the eigensolve and the
    // rotation that follow it, and its tile count should fill whole waves of the persistent contraction kernel
    // (the thread-per-matrix eigensolver of the per-pair H(k+q) solves needs tens of thousands of matrices per launch
    // to fill the GPU; it is worth more than L2 residency of the chunk: 16*ncols bytes per k written and read once
    // more from HBM is a few per cent of the S2 time)
    const size_t chunk_budget =
        (!kq_map && (eigh_thread_supported(nb) || eigh_cols_supported(nb))) ? ((size_t)512 << 20) : ((size_t)64 << 20);
    kchunk = choose_mtiles_per_chunk(NT, h->num_sms, (size_t)GEMM_BM * ncols * 16, MT, chunk_budget) * GEMM_BM;
    // rows of the g~ buffer kept (all of nk when it fits the cap; else a multiple of kchunk that is reused)
    c_rows = MT * GEMM_BM;
    if ((size_t)c_rows * ncols * 16 > cap)
      c_rows = std::max<int64_t>(kchunk, (int64_t)(cap / ((size_t)ncols * 16)) / kchunk * kchunk);
  } else {
    // k-chunk = whole i1 planes.  The last axis pass writes 64 complex columns (i1 values) per tile: prefer chunks of
    // a multiple of 64 planes (or all of them); 512 MB of [g~ | H(k+q)] per chunk unless that gives fewer than 16 planes.
    slab = (int64_t)grid->N[1] * grid->N[2];
    // per-k workspace of a chunk: [g~ | H(k+q)] (unfused) or only the H(k+q) block (fused), plus U_{k+q} and eps
    const size_t plane_bytes = (size_t)slab * ((fused ? ncols_h : ncols) + (kq_map ? 0 : nbb + nb)) * 16 + 16;
    const size_t soft = fused ? ((size_t)2 << 30) : ((size_t)512 << 20);
    int64_t fit = (int64_t)(std::min(cap, soft) / plane_bytes);
    if (fit < 16 && cap > soft) fit = std::min<int64_t>(64, (int64_t)(cap / plane_bytes));
    if (fit < 1) return h->fail(EPW_ENOMEM, "epw_interp_interpolate_grid: workspace_bytes too small for one i1 plane of g~");
    if (fit >= grid->N[0]) fit = grid->N[0];
    else if (fit > 64) fit = fit / 64 * 64;
    cs = (int)fit;
    // Per-pair H(k+q) on a grid: H(k+q) depends on q and H(Re) only, so its three axis passes and its
    // eigensolves are taken for QBH q-points of the S1 batch AT ONCE, before the g passes of those q (one eigensolver
    // launch of QBH*nk matrices instead of QBH launches of nk: 64,000 solves are 3.4 batches per persistent group of the
    // thread-per-matrix kernel -- a quarter of the GPU idles through the last round of every launch).  Needs the
    // H(k+q), U_{k+q} (and eps) of QBH q within the workspace cap; otherwise the per-q, chunked form below runs.
    if (!kq_map) {
      // (the two-kernel form also keeps g~ of one q, all k, in the same workspace)
      const size_t per_q = (size_t)nk * (2 * (size_t)nbb * 16 + (size_t)nb * 8 + (fused ? 0 : (size_t)ncols_g * 16));
      const size_t room = std::min(cap, (size_t)4 << 30);
      if (per_q <= room && axis_pass_supported(L[0]) && axis_pass_supported(L[1]) && axis_pass_supported(L[2])) {
        hbatch = (int)std::min<size_t>(room / per_q, (size_t)QB);
        cs = grid->N[0];
        ncolsC = fused ? 0 : ncols_g;
      }
    }
    nchunks = (int)ceil_div(grid->N[0], cs);
    kchunk = cs * slab;
    c_rows = nchunks == 1 ? nk : kchunk;
    KB1 = (int)ceil_div(2 * (int64_t)L[0], GEMM_BK);
    NTc = (int)ceil_div(2 * (int64_t)cs, GEMM_BN);
  }

  // ---- workspace ----
  if (!grid) {
    CU_OR_FAIL(h, h->Apack.reserve(sizeof(double) * (size_t)MT * KB * GEMM_CHUNK), "cudaMalloc Apack");
    CU_OR_FAIL(h, h->BpackH.reserve(sizeof(double) * (size_t)NTH * KB * GEMM_CHUNK), "cudaMalloc BpackH");
    CU_OR_FAIL(h, h->Bpack.reserve(sizeof(double) * (size_t)QB * NT * KB * GEMM_CHUNK), "cudaMalloc Bpack");
  } else {
    // columns of the axis-pass buffers: [g~ | H(k+q)] of one q, or (hbatch) g~ of one q and the H(k+q) of hbatch q in turn
    const int nc = hbatch ? std::max(ncols_g, hbatch * nbb) : std::max(ncols, nbb);
    const int maxN = std::max(std::max(grid->N[0], grid->N[1]), grid->N[2]);
    const int maxL = std::max(std::max(L[0], L[1]), L[2]);
    CU_OR_FAIL(h, h->X.reserve(sizeof(c128) * (size_t)h->box_size * nc), "cudaMalloc X");
    CU_OR_FAIL(h, h->T1.reserve(sizeof(c128) * (size_t)L[0] * L[1] * grid->N[2] * nc), "cudaMalloc T1");
    CU_OR_FAIL(h, h->T2.reserve(sizeof(c128) * (size_t)L[0] * slab * nc), "cudaMalloc T2");
    CU_OR_FAIL(h, h->Ptmp.reserve(sizeof(c128) * (size_t)maxL * maxN), "cudaMalloc axis phases");
    CU_OR_FAIL(h, h->P3pack.reserve(sizeof(double) * (size_t)ceil_div(2 * (int64_t)grid->N[2], GEMM_BN) *
                                    ceil_div(2 * (int64_t)L[2], GEMM_BK) * GEMM_CHUNK), "cudaMalloc P3pack");
    CU_OR_FAIL(h, h->P2pack.reserve(sizeof(double) * (size_t)ceil_div(2 * (int64_t)grid->N[1], GEMM_BN) *
                                    ceil_div(2 * (int64_t)L[1], GEMM_BK) * GEMM_CHUNK), "cudaMalloc P2pack");
    CU_OR_FAIL(h, h->P1pack.reserve(sizeof(double) * (size_t)nchunks * NTc * KB1 * GEMM_CHUNK), "cudaMalloc P1pack");
    CU_OR_FAIL(h, h->P1raw.reserve(sizeof(c128) * (size_t)nchunks * L[0] * cs), "cudaMalloc P1raw");
    CU_OR_FAIL(h, h->P2raw.reserve(sizeof(c128) * (size_t)L[1] * grid->N[1]), "cudaMalloc P2raw");
    CU_OR_FAIL(h, h->P3raw.reserve(sizeof(c128) * (size_t)L[2] * grid->N[2]), "cudaMalloc P3raw");
  }
  CU_OR_FAIL(h, h->Hk.reserve(sizeof(c128) * (size_t)nk * nbb), "cudaMalloc Hk");
  CU_OR_FAIL(h, h->Uk.reserve(sizeof(c128) * (size_t)nk * nbb), "cudaMalloc Uk");
  // the q side is small (16 (Np + Ne + 2 Nm^2) bytes per q): phases, D(q) and its eigen-system for ALL q of the call at once
  CU_OR_FAIL(h, h->Pq.reserve(sizeof(c128) * (size_t)nq * np), "cudaMalloc Pq");
  CU_OR_FAIL(h, h->Pqe.reserve(sizeof(c128) * (size_t)nq * ne), "cudaMalloc Pqe");
  CU_OR_FAIL(h, h->Dq.reserve(sizeof(c128) * (size_t)nq * nmm), "cudaMalloc Dq");
  CU_OR_FAIL(h, h->eq.reserve(sizeof(c128) * (size_t)nq * nmm), "cudaMalloc e_q");
  if (!h->ext_g1) CU_OR_FAIL(h, h->g1.reserve(sizeof(c128) * (size_t)QB * h->rows), "cudaMalloc g(Re,q)");
  const size_t hb = hbatch ? hbatch : 1;
  if (ncolsC) CU_OR_FAIL(h, h->C.reserve(sizeof(c128) * (size_t)c_rows * ncolsC), "cudaMalloc g~");
  if (hbatch) CU_OR_FAIL(h, h->Hkq.reserve(sizeof(c128) * hb * (size_t)nk * nbb), "cudaMalloc H(k+q)");
  if (!kq_map) CU_OR_FAIL(h, h->Ukq.reserve(sizeof(c128) * hb * (size_t)c_rows * nbb), "cudaMalloc Ukq");
  if (!kq_map && !eps_kq) CU_OR_FAIL(h, h->epskq_scratch.reserve(sizeof(double) * hb * (size_t)c_rows * nb), "cudaMalloc eps scratch");
  { const int rc = h->ensure_status(st); if (rc != EPW_OK) return rc; }
  if (h->window_on && !h->mask_out) CU_OR_FAIL(h, h->maskbuf.reserve((size_t)nk), "cudaMalloc mask");
  {
    const size_t need = std::max(eigh_large_scratch_bytes(nb, nk), eigh_large_scratch_bytes(nm, nq));
    if (need) CU_OR_FAIL(h, h->eig_scratch.reserve(need), "cudaMalloc eig scratch");
  }
  h->last_nk = nk;
  h->last_c_rows = c_rows;
  h->last_ncols = ncolsC;
  h->last_kmode = grid ? (fused ? 2 : 1) : 0;
  h->last_eq_slot = nq - 1;
  h->last_path = EPW_PATH_SMALL;
  h->last_qb = QB;
  h->last_kchunk = kchunk;

  // the two leading axis passes of the factorised S2: X [L1][L2][L3][nc] -> T1 [L1][L2][N3][nc] -> T2 [L1][N2][N3][nc]
  // Axis passes: a streaming kernel when the box extent is small (always, for Wigner-Seitz lists), else the in-place
  // tensor-path contraction with the packed phase table.
  // (nbat > 1: the same passes for nbat operands stored one after the other -- the outermost box index simply runs on)
  const bool dmma_axis2 = grid && grid_pass_dmma_supported(nb, L[1]);   // the pass-only variant runs it
  auto grid_pass_ab = [&](int nc, int nbat) -> cudaError_t {
    const int64_t N2 = grid->N[1], N3 = grid->N[2];
    const int64_t B = (int64_t)nbat * L[0];   // outermost extent of X, T1, T2
    cudaError_t e;
    if (axis_pass_supported(L[2]))
      e = launch_axis_pass(h->X.as<c128>(), nc, (int64_t)L[2] * nc, nc, B * L[1] * nc, h->P3raw.as<c128>(), L[2],
                           (int)N3, h->T1.as<c128>(), nc, N3 * nc, nc, h->num_sms, st);
    else
      e = launch_zgemm_strided(h->X.as<c128>(), nc, (int64_t)L[2] * nc, nc, 0, h->P3pack.as<double>(), nullptr, h->T1.p, nc,
                               N3 * nc, 1, nc, 0, 0, B * L[1] * nc, (int)N3, L[2], 1, h->num_sms, st);
    if (e != cudaSuccess) return e;
    h->launches++;
    // axis 2 as the DMMA product of grid_fused.cuh (pass-only form): B independent problems [L2][N3][nc] -> [N2][N3][nc].  The
    // columns are Nb^2 wide "modes" to that kernel: nc / Nb^2 of them.
    // (worth it for large passes only: 7.1 vs 8.3 ms of S2 per 13 q on configs[3], 3.5e7 outputs per pass; on configs[1], [2]
    //  -- 4.3e6 and 1.7e6 outputs -- the persistent kernel's start-up costs more than the streaming pass it replaces)
    if (dmma_axis2 && nc % nbb == 0 && L[1] >= 3 && N2 >= 4 && B * N2 * N3 * nc >= ((int64_t)1 << 24))
      return launch_grid_pass_dmma(h->T1.as<c128>(), N3, nc, L[1], h->P2raw.as<c128>(), (int)N2, nb, nc / nbb, h->num_sms,
                                   h->T2.as<c128>(), nc, (int)B, (int64_t)L[1] * N3 * nc, N2 * N3 * nc, st);
    if (axis_pass_supported(L[1]))
      return launch_axis_pass(h->T1.as<c128>(), N3 * nc, (int64_t)L[1] * N3 * nc, N3 * nc, B * N3 * nc,
                              h->P2raw.as<c128>(), L[1], (int)N2, h->T2.as<c128>(), N3 * nc, N2 * N3 * nc, N3 * nc,
                              h->num_sms, st);
    return launch_zgemm_strided(h->T1.as<c128>(), N3 * nc, (int64_t)L[1] * N3 * nc, N3 * nc, 0, h->P2pack.as<double>(),
                                nullptr, h->T2.p, N3 * nc, N2 * N3 * nc, 1, N3 * nc, 0, 0, B * N3 * nc,
                                (int)N2, L[1], 1, h->num_sms, st);
  };
  // the last axis pass for the i1 planes of chunk ci: T2 -> out [i1][i2][i3][nc]
  auto grid_pass_c = [&](int nc, int ci, c128 *out) -> cudaError_t {
    const int cnt = std::min(cs, grid->N[0] - ci * cs);
    const int64_t Mrows = slab * nc;
    if (axis_pass_supported(L[0]))
      return launch_axis_pass(h->T2.as<c128>(), Mrows, 0, Mrows, Mrows, h->P1raw.as<c128>() + (int64_t)ci * L[0] * cs, L[0],
                              cnt, out, Mrows, 0, Mrows, h->num_sms, st);
    return launch_zgemm_strided(h->T2.as<c128>(), Mrows, 0, Mrows, 0,
                                h->P1pack.as<double>() + (int64_t)ci * NTc * KB1 * GEMM_CHUNK, nullptr, out, Mrows, 0, 1,
                                Mrows, 0, 0, Mrows, cnt, L[0], 1, h->num_sms, st);
  };

  const int t_total = h->begin_span(7, st);

  // ---- k side (once per call): S0 phases, H(k) by the same contraction as S2, eigensolve ----
  int sp = h->begin_span(0, st);
  if (!grid) {
    LAUNCH(h, launch_phase_pack_a(k_list, nk, h->Re.as<int32_t>(), h->we.as<double>(), ne, h->Apack.as<double>(), st),
           "phase_pack_a");
  } else {
    // one small phase table per crystal axis, packed as the B operand of its pass
    struct Axis { int d; DevBuf *pack; };
    const Axis ax[2] = {{2, &h->P3pack}, {1, &h->P2pack}};
    for (const Axis &a : ax) {
      c128 *raw = (a.d == 2 ? h->P3raw : h->P2raw).as<c128>();   // [L_d][N_d], kept for the streaming axis pass
      LAUNCH(h, launch_grid_axis_phase(grid->N[a.d], 0, grid->N[a.d], grid->s[a.d], h->box_lo[a.d], L[a.d], raw, st),
             "axis phases");
      LAUNCH(h, launch_pack_b_strided(raw, grid->N[a.d], 1, 0, 1, 0, nullptr, 0.0, L[a.d], grid->N[a.d],
                                      a.pack->as<double>(), st), "pack axis phases");
    }
    for (int ci = 0; ci < nchunks; ci++) {
      const int cnt = std::min(cs, grid->N[0] - ci * cs);
      c128 *raw = h->P1raw.as<c128>() + (int64_t)ci * L[0] * cs;   // [L1][cnt], kept for the fused kernel
      LAUNCH(h, launch_grid_axis_phase(grid->N[0], ci * cs, cnt, grid->s[0], h->box_lo[0], L[0], raw, st), "axis phases");
      LAUNCH(h, launch_pack_b_strided(raw, cnt, 1, 0, 1, 0, nullptr, 0.0, L[0], cnt,
                                      h->P1pack.as<double>() + (int64_t)ci * NTc * KB1 * GEMM_CHUNK, st),
             "pack axis phases");
    }
  }
  h->end_span(sp, st);
  sp = h->begin_span(3, st);
  if (k_cached) {
    CU_OR_FAIL(h, cudaMemcpyAsync(eps_k, h->epsk_keep.p, sizeof(double) * (size_t)nk * nb, cudaMemcpyDeviceToDevice, st),
               "copy cached eps_k");
  } else {
  if (!grid) {
    LAUNCH(h,
           launch_pack_b(nullptr, nullptr, nullptr, 0.0, h->H.as<c128>(), nullptr, nbb, nm, ne, 0, nbb,
                         h->BpackH.as<double>(), st),
           "pack_b(H)");
    LAUNCH(h, launch_zgemm_dmma(h->Apack.as<double>(), h->BpackH.as<double>(), h->Hk.as<c128>(), nk, nbb, KB, nbb,
                                h->num_sms, st),
           "zgemm H(k)");
  } else {
    LAUNCH(h, launch_box_scatter(nullptr, nullptr, nullptr, 0.0, h->H.as<c128>(), nullptr, h->we.as<double>(),
                                 h->boxidx.as<int32_t>(), h->box_size, nbb, nm, ne, 0, nbb, h->X.as<c128>(), st),
           "box_scatter(H)");
    LAUNCH(h, grid_pass_ab(nbb, 1), "grid passes H(k)");
    for (int ci = 0; ci < nchunks; ci++)
      LAUNCH(h, grid_pass_c(nbb, ci, h->Hk.as<c128>() + (int64_t)ci * kchunk * nbb), "grid pass H(k)");
  }
  LAUNCH(h, launch_eigh_batched(h->Hk.as<c128>(), nbb, nb, nk, eps_k, h->Uk.as<c128>(), 0, h->status.as<int32_t>(),
                                h->eig_scratch.as<c128>(), h->work_slot(0), st),
         "eigh H(k)");
  if (grid) {
    CU_OR_FAIL(h, h->epsk_keep.reserve(sizeof(double) * (size_t)nk * nb), "cudaMalloc eps_k cache");
    CU_OR_FAIL(h, cudaMemcpyAsync(h->epsk_keep.p, eps_k, sizeof(double) * (size_t)nk * nb, cudaMemcpyDeviceToDevice, st),
               "keep eps_k");
    kside_record(h, grid, false, EPW_PATH_SMALL);
  }
  }
  h->end_span(sp, st);

  // ---- q side (once per call): S0 phases of every q, D(q), phonon eigen-systems ----
  sp = h->begin_span(0, st);
  LAUNCH(h, launch_phase_table(q_list, nq, h->Rp.as<int32_t>(), h->wp.as<double>(), np, h->Pq.as<c128>(), st),
         "phase_table(q,Rp)");
  if (ncols_h)
    LAUNCH(h, launch_phase_table(q_list, nq, h->Re.as<int32_t>(), h->ones.as<double>(), ne, h->Pqe.as<c128>(), st),
           "phase_table(q,Re)");
  h->end_span(sp, st);
  sp = h->begin_span(2, st);
  LAUNCH(h, launch_interp_operator(h->D.as<c128>(), nm, np, h->Pq.as<c128>(), nq, h->Dq.as<c128>(), st), "D(q)");
  LAUNCH(h, launch_eigh_batched(h->Dq.as<c128>(), nmm, nm, nq, omega_q, h->eq.as<c128>(), 1, h->status.as<int32_t>(),
                                h->eig_scratch.as<c128>(), h->work_slot(2), st),
         "eigh D(q)");
  h->end_span(sp, st);

  for (int64_t q0 = 0; q0 < nq; q0 += QB) {
    const int qb = (int)std::min<int64_t>(QB, nq - q0);
    const c128 *Pq_b = h->Pq.as<c128>() + q0 * np, *Pqe_b = h->Pqe.as<c128>() + q0 * ne, *eq_b = h->eq.as<c128>() + q0 * nmm;
    // ---- S1: Eq. 9 for the batch ----
    sp = h->begin_span(1, st);
    const c128 *g1b = h->ext_g1 ? h->ext_g1 + q0 * h->rows : h->g1.as<c128>();
    if (!h->ext_g1)
      LAUNCH(h, launch_rp_to_q(h->g.as<c128>(), h->rows, np, Pq_b, qb, h->g1.as<c128>(), st), "rp_to_q");
    h->end_span(sp, st);
    if (!grid) {
      sp = h->begin_span(8, st);
      for (int iq = 0; iq < qb; iq++)
        LAUNCH(h,
               launch_pack_b(g1b + (int64_t)iq * h->rows, eq_b + (int64_t)iq * nmm,
                             omega_q + (q0 + iq) * nm, h->cfg.omega_min, h->H.as<c128>(),
                             ncols_h ? Pqe_b + (int64_t)iq * ne : nullptr, nbb, nm, ne, ncols_g, ncols_h,
                             h->Bpack.as<double>() + (int64_t)iq * NT * KB * GEMM_CHUNK, st),
               "pack_b");
      h->end_span(sp, st);
    }

    for (int iq = 0; iq < qb; iq++) {
      const int64_t q = q0 + iq;
      const double *Bq = grid ? nullptr : h->Bpack.as<double>() + (int64_t)iq * NT * KB * GEMM_CHUNK;
      if (hbatch && iq % hbatch == 0) {
        // ---- S3a + S3b for the next hbatch q-points at once: H(k+q) = sum_Re e^{2 pi i (k+q).Re} H(Re) by the three axis
        //      passes on Nb^2 columns (operands of the hn q-points one after the other), then ONE eigensolver launch ----
        const int hn = std::min(hbatch, qb - iq);
        const int64_t Mh = slab * nbb;
        sp = h->begin_span(4, st);
        for (int j = 0; j < hn; j++)
          LAUNCH(h, launch_box_scatter(nullptr, nullptr, nullptr, 0.0, h->H.as<c128>(), Pqe_b + (int64_t)(iq + j) * ne,
                                       h->we.as<double>(), h->boxidx.as<int32_t>(), h->box_size, nbb, nm, ne, 0, nbb,
                                       h->X.as<c128>() + (int64_t)j * h->box_size * nbb, st),
                 "box_scatter(H e^{iqR})");
        LAUNCH(h, grid_pass_ab(nbb, hn), "grid passes H(k+q)");
        LAUNCH(h, launch_axis_pass(h->T2.as<c128>(), Mh, (int64_t)L[0] * Mh, Mh, (int64_t)hn * Mh, h->P1raw.as<c128>(), L[0],
                                   grid->N[0], h->Hkq.as<c128>(), Mh, (int64_t)grid->N[0] * Mh, Mh, h->num_sms, st),
               "grid pass H(k+q)");
        h->end_span(sp, st);
        sp = h->begin_span(5, st);
        double *eps_dst = eps_kq ? eps_kq + q * nk * nb : h->epskq_scratch.as<double>();
        LAUNCH(h, launch_eigh_batched(h->Hkq.as<c128>(), nbb, nb, (int64_t)hn * nk, eps_dst, h->Ukq.as<c128>(), 0,
                                      h->status.as<int32_t>(), h->eig_scratch.as<c128>(), h->work_slot(1), st),
               "eigh H(k+q)");
        h->end_span(sp, st);
      }
      const int hslot = hbatch ? iq % hbatch : 0;            // slot of this q in the U_{k+q} / eps scratch of its H batch
      const int nc_g = hbatch ? ncols_g : ncols;             // columns of the axis-pass buffers of this q
      if (grid) {
        sp = h->begin_span(8, st);
        LAUNCH(h, launch_box_scatter(g1b + (int64_t)iq * h->rows, eq_b + (int64_t)iq * nmm,
                                     omega_q + q * nm, h->cfg.omega_min, h->H.as<c128>(),
                                     (ncols_h && !hbatch) ? Pqe_b + (int64_t)iq * ne : nullptr, h->we.as<double>(),
                                     h->boxidx.as<int32_t>(), h->box_size, nbb, nm, ne, ncols_g, hbatch ? 0 : ncols_h,
                                     h->X.as<c128>(), st),
               "box_scatter");
        h->end_span(sp, st);
        sp = h->begin_span(4, st);
        LAUNCH(h, grid_pass_ab(nc_g, 1), "grid passes S2");
        h->end_span(sp, st);
      }
      for (int64_t k0 = 0; k0 < nk; k0 += kchunk) {
        const int64_t kn = std::min(kchunk, nk - k0);
        const int64_t crow = k0 % c_rows;
        c128 *Cc = h->C.as<c128>() + crow * ncolsC;
        // ---- S2: Re -> k contraction (+ H(k+q) columns) ----
        sp = h->begin_span(4, st);
        if (!grid) {
          LAUNCH(h, launch_zgemm_dmma(h->Apack.as<double>() + (k0 / GEMM_BM) * (int64_t)KB * GEMM_CHUNK, Bq, Cc, kn, ncols,
                                      KB, ncols, h->num_sms, st),
                 "zgemm S2");
        } else if (!fused) {
          if (hbatch && can_fuse)   // g columns only, all i1 planes: the pass as a DMMA product (grid_fused.cuh, pass-only form)
            LAUNCH(h, launch_grid_pass_dmma(h->T2.as<c128>(), slab, nc_g, L[0], h->P1raw.as<c128>(), grid->N[0], nb, nm,
                                            h->num_sms, Cc, nc_g, 1, 0, 0, st),
                   "grid pass S2 (DMMA)");
          else
            LAUNCH(h, grid_pass_c(nc_g, (int)(k0 / kchunk), Cc), "grid pass S2");
        } else if (ncols_h && !hbatch) {
          // fused form: only the H(k+q) columns of the last axis pass go to HBM (the eigensolver's input)
          const int ci = (int)(k0 / kchunk);
          const int cnt = std::min(cs, grid->N[0] - ci * cs);
          const int64_t Mh = slab * nbb;
          if (axis_pass_supported(L[0]))
            LAUNCH(h, launch_axis_pass(h->T2.as<c128>() + ncols_g, nbb, ncols, slab * ncols, Mh,
                                       h->P1raw.as<c128>() + (int64_t)ci * L[0] * cs, L[0], cnt, Cc, Mh, 0, Mh, h->num_sms, st),
                   "grid pass H(k+q)");
          else
            LAUNCH(h, launch_zgemm_strided(h->T2.as<c128>() + ncols_g, nbb, ncols, slab * ncols, 0,
                                           h->P1pack.as<double>() + (int64_t)ci * NTc * KB1 * GEMM_CHUNK, nullptr, Cc, Mh, 0,
                                           1, Mh, 0, 0, Mh, cnt, L[0], 1, h->num_sms, st),
                   "grid pass H(k+q)");
        }
        h->end_span(sp, st);
        const c128 *Ukq_ptr;
        const int32_t *kq_idx = nullptr;
        if (kq_map) {
          Ukq_ptr = h->Uk.as<c128>();
          kq_idx = kq_map + q * nk + k0;
          if (eps_kq) {
            sp = h->begin_span(5, st);
            h->launches++;
            gather_eps_kernel<<<grid_cap(ceil_div(kn * nb, 256), 8), 256, 0, st>>>(
                eps_k, kq_idx, nb, kn, eps_kq + (q * nk + k0) * nb);
            CU_OR_FAIL(h, cudaGetLastError(), "gather_eps");
            h->end_span(sp, st);
          }
        } else if (hbatch) {
          Ukq_ptr = h->Ukq.as<c128>() + (int64_t)hslot * nk * nbb;   // solved with its H batch above
        } else {
          // ---- S3b per pair: eigensolve the H(k+q) block of the contraction output ----
          sp = h->begin_span(5, st);
          c128 *Ukq_c = h->Ukq.as<c128>() + crow * nbb;
          double *eps_dst = eps_kq ? eps_kq + (q * nk + k0) * nb : h->epskq_scratch.as<double>() + crow * nb;
          LAUNCH(h, launch_eigh_batched(Cc + (ncolsC - ncols_h), ncolsC, nb, kn, eps_dst, Ukq_c, 0, h->status.as<int32_t>(),
                                        h->eig_scratch.as<c128>(), h->work_slot(1), st),
                 "eigh H(k+q)");
          h->end_span(sp, st);
          Ukq_ptr = Ukq_c;
        }
        // ---- energy-window pre-screening of the pairs of this chunk ----
        const uint8_t *mask = nullptr;
        if (h->window_on) {
          uint8_t *m = h->mask_out ? h->mask_out + q * nk + k0 : h->maskbuf.as<uint8_t>();
          const double *ekq = kq_map ? nullptr
                                     : (eps_kq ? eps_kq + (q * nk + k0) * nb
                                               : h->epskq_scratch.as<double>() + ((int64_t)hslot * nk + crow) * nb);
          sp = h->begin_span(5, st);
          LAUNCH(h, launch_window_mask(eps_k + k0 * nb, ekq, eps_k, kq_idx, nb, kn, h->emin, h->emax, m, st), "window mask");
          h->end_span(sp, st);
          mask = m;
        }
        // ---- S4b: band rotation + |g|^2 ----
        sp = h->begin_span(6, st);
        if (!fused) {
          LAUNCH(h, launch_rotate_g2(Cc, grid ? nc_g : ncols, h->Uk.as<c128>() + k0 * nbb, Ukq_ptr, kq_idx, nb, nm, kn, mask,
                                     G2(q, k0), st),
                 "rotate_g2");
        } else {
          const int ci = (int)(k0 / kchunk);
          const int cnt = std::min(cs, grid->N[0] - ci * cs);
          // the consumer, if on, is taken in the epilogue of the same kernel: |g|^2 goes from the accumulator registers into
          // Im Sigma_nk, and with g2 = NULL nothing else leaves the SM
          SelfEnergyFold fold;
          if (h->cons.on) {
            fold.out = h->cons.out + k0 * nb;
            fold.eps_k = eps_k + k0 * nb;
            fold.eps_kq = kq_map ? eps_k
                                 : (eps_kq ? eps_kq + (q * nk + k0) * nb
                                           : h->epskq_scratch.as<double>() + ((int64_t)hslot * nk + crow) * nb);
            fold.omega_q = omega_q + q * nm;
            fold.w_q = h->cons.w_q;
            fold.iq = q;
            fold.mu = h->cons.mu; fold.kT = h->cons.kT; fold.sigma = h->cons.sigma;
          }
          LAUNCH(h, launch_grid_fused(h->T2.as<c128>(), slab, nc_g, L[0], h->P1raw.as<c128>() + (int64_t)ci * L[0] * cs,
                                          cnt, h->Uk.as<c128>() + k0 * nbb, Ukq_ptr, kq_idx, nb, nm, h->num_sms, mask,
                                          G2(q, k0), h->cons.on ? &fold : nullptr, st),
                 "grid_fused");
        }
        if (h->cons.on && !fused) {
          const double *ekq = kq_map ? nullptr
                                     : (eps_kq ? eps_kq + (q * nk + k0) * nb
                                               : h->epskq_scratch.as<double>() + ((int64_t)hslot * nk + crow) * nb);
          LAUNCH(h, launch_selfenergy_accumulate(G2(q, k0), eps_k + k0 * nb, ekq, eps_k, kq_idx, omega_q + q * nm,
                                                 h->cons.w_q, q, h->cons.mu, h->cons.kT, h->cons.sigma, nb, nm, kn,
                                                 h->cons.out + k0 * nb, st),
                 "Im Sigma accumulate");
        }
        h->end_span(sp, st);
      }
      if (g2) { const int rc = h->drain_q(q, nk, E, g2, eps_kq, st); if (rc != EPW_OK) return rc; }
    }
  }
  h->end_span(t_total, st);
  return EPW_OK;
}

extern "C" {

int epw_interp_set_selfenergy_consumer(epw_interp_t h, int enabled, double mu, double kT, double sigma, const double *w_q,
                                       double *im_sigma) {
  if (!h) return EPW_EINVAL;
  if (enabled && (!(kT > 0.0) || !(sigma > 0.0) || !im_sigma))
    return h->fail(EPW_EINVAL, "epw_interp_set_selfenergy_consumer: need kT > 0, sigma > 0 and an output buffer");
  h->cons.on = enabled != 0;
  h->cons.mu = mu;
  h->cons.kT = kT;
  h->cons.sigma = sigma;
  h->cons.w_q = enabled ? w_q : nullptr;
  h->cons.out = enabled ? im_sigma : nullptr;
  return EPW_OK;
}

int epw_interp_set_energy_window(epw_interp_t h, int enabled, double emin, double emax, uint8_t *mask_out) {
  if (!h) return EPW_EINVAL;
  if (enabled && !(emin <= emax)) return h->fail(EPW_EINVAL, "epw_interp_set_energy_window: need emin <= emax");
  h->window_on = enabled != 0;
  h->emin = emin;
  h->emax = emax;
  h->mask_out = enabled ? mask_out : nullptr;
  return EPW_OK;
}

int epw_interp_set_rp_shard(epw_interp_t h, int32_t ip_start, int32_t ip_count) {
  if (!h) return EPW_EINVAL;
  if (ip_start < 0 || ip_count <= 0 || ip_start + ip_count > h->np)
    return h->fail(EPW_EINVAL, "epw_interp_set_rp_shard: range outside [0, Np)");
  if (h->g.p) return h->fail(EPW_EINVAL, "epw_interp_set_rp_shard: call before any g(Re,Rp) slab is uploaded");
  h->rp_lo = ip_start;
  h->rp_cnt = ip_count;
  h->sharded = !(ip_start == 0 && ip_count == h->np);
  return EPW_OK;
}

static int rp_to_q_partial_impl(epw_interp_t h, const double *q_list, int64_t nq, void *g1_partial, void *const *dst,
                               void *cuda_stream);

int epw_interp_rp_to_q_partial(epw_interp_t h, const double *q_list, int64_t nq, void *g1_partial, void *cuda_stream) {
  if (!h) return EPW_EINVAL;
  if (!g1_partial) return h->fail(EPW_EINVAL, "epw_interp_rp_to_q_partial: null output pointer");
  return rp_to_q_partial_impl(h, q_list, nq, g1_partial, nullptr, cuda_stream);
}

int epw_interp_rp_to_q_scatter_add(epw_interp_t h, const double *q_list, int64_t nq, void *const *dst, void *cuda_stream) {
  if (!h) return EPW_EINVAL;
  if (!dst) return h->fail(EPW_EINVAL, "epw_interp_rp_to_q_scatter_add: null destination table");
  for (int64_t i = 0; i < nq; i++)
    if (!dst[i]) return h->fail(EPW_EINVAL, "epw_interp_rp_to_q_scatter_add: null destination pointer");
  // The kernel adds with red.global.add.f64 at system scope.  Into another GPU's memory that needs native atomics over the
  // link (NVLink has them, PCIe peer access does not): ask once per peer device and refuse instead of adding wrongly.
  CU_OR_FAIL(h, cudaSetDevice(h->cfg.device), "cudaSetDevice");
  int peer_ok[64];
  for (int &v : peer_ok) v = -1;
  for (int64_t i = 0; i < nq; i++) {
    cudaPointerAttributes pa;
    if (cudaPointerGetAttributes(&pa, dst[i]) != cudaSuccess) { cudaGetLastError(); continue; }   // unknown to this process
    if (pa.type != cudaMemoryTypeDevice || pa.device == h->cfg.device || pa.device < 0 || pa.device >= 64) continue;
    if (peer_ok[pa.device] < 0) {
      int v = 0;
      if (cudaDeviceGetP2PAttribute(&v, cudaDevP2PAttrNativeAtomicSupported, h->cfg.device, pa.device) != cudaSuccess) {
        cudaGetLastError();
        v = 0;
      }
      peer_ok[pa.device] = v;
    }
    if (!peer_ok[pa.device])
      return h->fail(EPW_EUNSUPPORTED, "epw_interp_rp_to_q_scatter_add: destination " + std::to_string(i) + " lives on device " +
                                       std::to_string(pa.device) + ", to which device " + std::to_string(h->cfg.device) +
                                       " has no native peer atomics (cudaDevP2PAttrNativeAtomicSupported = 0): use "
                                       "epw_interp_rp_to_q_partial + a reduce-scatter instead");
  }
  return rp_to_q_partial_impl(h, q_list, nq, nullptr, dst, cuda_stream);
}

static int rp_to_q_partial_impl(epw_interp_t h, const double *q_list, int64_t nq, void *g1_partial, void *const *dst,
                               void *cuda_stream) {
  if (!q_list || nq <= 0) return h->fail(EPW_EINVAL, "epw_interp_rp_to_q_partial: null pointer or nq <= 0");
  if (!h->operators_set) return h->fail(EPW_EINVAL, "epw_interp_rp_to_q_partial: operators not set");
  for (int ip = h->rp_lo; ip < h->rp_lo + h->rp_cnt; ip++)
    if (!h->slab_set[ip]) return h->fail(EPW_EINVAL, "epw_interp_rp_to_q_partial: g(Re,Rp) slab of this shard missing");
  CU_OR_FAIL(h, cudaSetDevice(h->cfg.device), "cudaSetDevice");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  h->last_stream = st;
  h->launches = 0;
  int QB = 1;
  { const int rc = h->s1_batch(nq, &QB); if (rc != EPW_OK) return rc; }
  CU_OR_FAIL(h, h->Pq.reserve(sizeof(c128) * (size_t)QB * h->np), "cudaMalloc Pq");
  c128 *out = reinterpret_cast<c128 *>(g1_partial);
  c128 *const *dst_dev = nullptr;
  if (dst) {
    // The destination table on the device, copied ON the stream (so it cannot overtake the previous call's kernels, which
    // still read the old table) and without waiting for the stream.  The source is the library's own PAGEABLE copy of the
    // caller's array: a copy from pageable memory is staged by the runtime before cudaMemcpyAsync returns, so both this
    // copy and the caller's array (pinned or not) are free again on return.
    CU_OR_FAIL(h, h->dst_tab.reserve(sizeof(void *) * (size_t)nq), "cudaMalloc destination table");
    h->dst_host.assign(dst, dst + nq);
    CU_OR_FAIL(h, cudaMemcpyAsync(h->dst_tab.p, h->dst_host.data(), sizeof(void *) * (size_t)nq, cudaMemcpyHostToDevice, st),
               "cudaMemcpy destination table");
    dst_dev = h->dst_tab.as<c128 *>();
  }
  for (int64_t q0 = 0; q0 < nq; q0 += QB) {
    const int qb = (int)std::min<int64_t>(QB, nq - q0);
    int sp = h->begin_span(0, st);
    // phases of this shard's lattice vectors only: P[iq][ip - rp_lo]
    LAUNCH(h, launch_phase_table(q_list + 3 * q0, qb, h->Rp.as<int32_t>() + 3 * h->rp_lo, h->wp.as<double>() + h->rp_lo,
                                 h->rp_cnt, h->Pq.as<c128>(), st),
           "phase_table(q,Rp shard)");
    h->end_span(sp, st);
    sp = h->begin_span(1, st);
    LAUNCH(h, launch_rp_to_q_dst(h->g.as<c128>(), h->rows, h->rp_cnt, h->Pq.as<c128>(), qb, out ? out + q0 * h->rows : nullptr,
                                 dst_dev ? dst_dev + q0 : nullptr, st),
           "rp_to_q (partial)");
    h->end_span(sp, st);
  }
  return EPW_OK;
}

int epw_interp_set_gq(epw_interp_t h, const void *g1_reduced) {
  if (!h) return EPW_EINVAL;
  h->ext_g1 = reinterpret_cast<const c128 *>(g1_reduced);
  return EPW_OK;
}

int epw_interp_sync(epw_interp_t h) {
  if (!h) return EPW_EINVAL;
  CU_OR_FAIL(h, cudaSetDevice(h->cfg.device), "cudaSetDevice");
  CU_OR_FAIL(h, cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize");
  if (h->status.p) {
    int32_t s = 0;
    CU_OR_FAIL(h, cudaMemcpy(&s, h->status.p, sizeof(s), cudaMemcpyDeviceToHost), "cudaMemcpy status");
    if (s) {
      CU_OR_FAIL(h, cudaMemset(h->status.p, 0, sizeof(int32_t)), "memset status");   // read once, then cleared
      h->kside.valid = false;   // the solve that failed may have been one of H(k): the next grid call solves them again
      return h->fail(EPW_ENOTCONVERGED, "a Jacobi eigensolve did not converge within the sweep limit (in this or an "
                                        "earlier call since the last epw_interp_sync)");
    }
  }
  return EPW_OK;
}

static int interpolate_host_impl(epw_interp_t h, const double *k_list, const int32_t *k_grid, const double *k_shift,
                                 int64_t nk, const double *q_list, int64_t nq, const int32_t *kq_map, double *eps_k,
                                 double *eps_kq, double *omega_q, double *g2, void *cuda_stream) {
  if (!h) return EPW_EINVAL;
  if ((!k_list && !k_grid) || !q_list || !eps_k || !omega_q || (!g2 && !h->cons.on) || nk <= 0 || nq <= 0)
    return h->fail(EPW_EINVAL, "epw_interp_interpolate_host: null pointer or non-positive nk/nq");
  CU_OR_FAIL(h, cudaSetDevice(h->cfg.device), "cudaSetDevice");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const size_t E = (size_t)h->nbb * h->nm;
  if (k_list) CU_OR_FAIL(h, h->hs_k.reserve(sizeof(double) * 3 * nk), "cudaMalloc k staging");
  CU_OR_FAIL(h, h->hs_q.reserve(sizeof(double) * 3 * nq), "cudaMalloc q staging");
  if (kq_map) CU_OR_FAIL(h, h->hs_map.reserve(sizeof(int32_t) * nk * nq), "cudaMalloc kq_map staging");
  CU_OR_FAIL(h, h->hs_epsk.reserve(sizeof(double) * nk * h->nb), "cudaMalloc eps_k staging");
  if (eps_kq) CU_OR_FAIL(h, h->hs_epskq.reserve(sizeof(double) * nk * nq * h->nb), "cudaMalloc eps_kq staging");
  CU_OR_FAIL(h, h->hs_omega.reserve(sizeof(double) * nq * h->nm), "cudaMalloc omega staging");
  if (g2) CU_OR_FAIL(h, h->hs_g2.reserve(sizeof(double) * E * nk * nq), "cudaMalloc g2 staging");
  if (k_list)
    CU_OR_FAIL(h, cudaMemcpyAsync(h->hs_k.p, k_list, sizeof(double) * 3 * nk, cudaMemcpyHostToDevice, st), "H2D k");
  CU_OR_FAIL(h, cudaMemcpyAsync(h->hs_q.p, q_list, sizeof(double) * 3 * nq, cudaMemcpyHostToDevice, st), "H2D q");
  if (kq_map)
    CU_OR_FAIL(h, cudaMemcpyAsync(h->hs_map.p, kq_map, sizeof(int32_t) * nk * nq, cudaMemcpyHostToDevice, st), "H2D map");
  const int32_t *map_d = kq_map ? h->hs_map.as<int32_t>() : nullptr;
  double *epskq_d = eps_kq ? h->hs_epskq.as<double>() : nullptr;
  // |g|^2 (and eps_kq) leave the device q by q on a second stream while the next q is being computed
  if (!h->copy_stream) CU_OR_FAIL(h, cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking), "cudaStreamCreate");
  h->sink.g2 = g2;
  h->sink.eps_kq = eps_kq;
  h->sink.active = true;
  h->sink_ev_used = 0;
  const int rc = k_list ? epw_interp_interpolate(h, h->hs_k.as<double>(), nk, h->hs_q.as<double>(), nq, map_d,
                                                 h->hs_epsk.as<double>(), epskq_d, h->hs_omega.as<double>(),
                                                 g2 ? h->hs_g2.as<double>() : nullptr, cuda_stream)
                        : epw_interp_interpolate_grid(h, k_grid, k_shift, h->hs_q.as<double>(), nq, map_d,
                                                      h->hs_epsk.as<double>(), epskq_d, h->hs_omega.as<double>(),
                                                      g2 ? h->hs_g2.as<double>() : nullptr, cuda_stream);
  h->sink.active = false;
  if (rc != EPW_OK) {
    cudaStreamSynchronize(h->copy_stream);
    return rc;
  }
  CU_OR_FAIL(h, cudaMemcpyAsync(eps_k, h->hs_epsk.p, sizeof(double) * nk * h->nb, cudaMemcpyDeviceToHost, st), "D2H eps_k");
  CU_OR_FAIL(h, cudaMemcpyAsync(omega_q, h->hs_omega.p, sizeof(double) * nq * h->nm, cudaMemcpyDeviceToHost, st), "D2H omega");
  if (!g2 && eps_kq)   // (with g2 the eps_kq slices left with the |g|^2 of their q)
    CU_OR_FAIL(h, cudaMemcpyAsync(eps_kq, h->hs_epskq.p, sizeof(double) * nk * nq * h->nb, cudaMemcpyDeviceToHost, st),
               "D2H eps_kq");
  CU_OR_FAIL(h, cudaStreamSynchronize(h->copy_stream), "cudaStreamSynchronize(copy)");
  return epw_interp_sync(h);
}

int epw_interp_interpolate_host(epw_interp_t h, const double *k_list, int64_t nk, const double *q_list, int64_t nq,
                                const int32_t *kq_map, double *eps_k, double *eps_kq, double *omega_q, double *g2,
                                void *cuda_stream) {
  if (h && !k_list) return h->fail(EPW_EINVAL, "epw_interp_interpolate_host: null k_list");
  return interpolate_host_impl(h, k_list, nullptr, nullptr, nk, q_list, nq, kq_map, eps_k, eps_kq, omega_q, g2,
                               cuda_stream);
}

int epw_interp_interpolate_grid_host(epw_interp_t h, const int32_t *k_grid, const double *k_shift, const double *q_list,
                                     int64_t nq, const int32_t *kq_map, double *eps_k, double *eps_kq, double *omega_q,
                                     double *g2, void *cuda_stream) {
  if (!h) return EPW_EINVAL;
  if (!k_grid || k_grid[0] <= 0 || k_grid[1] <= 0 || k_grid[2] <= 0)
    return h->fail(EPW_EINVAL, "epw_interp_interpolate_grid_host: k_grid must hold three positive sizes");
  return interpolate_host_impl(h, nullptr, k_grid, k_shift, (int64_t)k_grid[0] * k_grid[1] * k_grid[2], q_list, nq, kq_map,
                               eps_k, eps_kq, omega_q, g2, cuda_stream);
}

int epw_interp_get_stage_times(epw_interp_t h, double *ms, int n) {
  if (!h || !ms || n <= 0) return EPW_EINVAL;
  CU_OR_FAIL(h, cudaSetDevice(h->cfg.device), "cudaSetDevice");
  CU_OR_FAIL(h, cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize");
  const int m = std::min(n, (int)EPW_NUM_STAGES);
  for (int i = 0; i < m; i++) ms[i] = 0.0;
  for (const auto &s : h->spans) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, h->ev_pool[s.e0], h->ev_pool[s.e1]) == cudaSuccess && s.stage < m) ms[s.stage] += t;
  }
  return m;
}

int epw_interp_get_stage_launches(epw_interp_t h, int64_t *counts, int n) {
  if (!h || !counts || n <= 0) return EPW_EINVAL;
  const int m = std::min(n, (int)EPW_NUM_STAGES);
  for (int i = 0; i < m; i++) counts[i] = 0;
  for (const auto &s : h->spans)
    if (s.stage < m) counts[s.stage] += s.nlaunch;
  return m;
}

int64_t epw_interp_last_launch_count(epw_interp_t h) { return h ? h->launches : 0; }

int epw_interp_get_eigh_rotations(epw_interp_t h, uint64_t *counts, int n) {
  if (!h || !counts || n <= 0) return EPW_EINVAL;
  const int m = std::min(n, 3);
  for (int i = 0; i < m; i++) counts[i] = 0;
  if (!h->workctr.p) return m;
  CU_OR_FAIL(h, cudaSetDevice(h->cfg.device), "cudaSetDevice");
  CU_OR_FAIL(h, cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize");
  unsigned long long v[3];
  CU_OR_FAIL(h, cudaMemcpy(v, h->workctr.p, sizeof(v), cudaMemcpyDeviceToHost), "cudaMemcpy work counters");
  for (int i = 0; i < m; i++) counts[i] = v[i];
  return m;
}

int epw_interp_last_plan(epw_interp_t h, int64_t *plan, int n) {
  if (!h || !plan || n <= 0) return EPW_EINVAL;
  const int64_t v[4] = {h->last_path, h->last_qb, h->last_kchunk, h->last_kmode};
  const int m = std::min(n, 4);
  for (int i = 0; i < m; i++) plan[i] = v[i];
  return m;
}

int64_t epw_interp_debug_get(epw_interp_t h, int what, void *dst, size_t bytes) {
  if (!h || !dst) return EPW_EINVAL;
  CU_OR_FAIL(h, cudaSetDevice(h->cfg.device), "cudaSetDevice");
  CU_OR_FAIL(h, cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize");
  const size_t nbb = h->nbb;
  const void *src = nullptr;
  size_t need = 0;
  switch (what) {
    case EPW_DBG_G_REQ: {  // g(Re,q) of the last q of the last batch: stored [ka][ie][n'][m'] = Fortran (m',n',ie,ka)
      need = sizeof(c128) * (size_t)h->rows;
      src = h->g1.p;  // caller should use nq such that the last batch has one q, or read slot 0 of the last batch
      break;
    }
    case EPW_DBG_H_K: need = sizeof(c128) * nbb * h->last_nk; src = h->Hk.p; break;
    case EPW_DBG_U_K: need = sizeof(c128) * nbb * h->last_nk; src = h->Uk.p; break;
    case EPW_DBG_U_KQ: need = sizeof(c128) * nbb * std::min(h->last_nk, h->last_c_rows); src = h->Ukq.p; break;
    case EPW_DBG_E_Q:
      need = sizeof(c128) * (size_t)h->nmm;
      src = h->eq.p ? h->eq.as<c128>() + h->last_eq_slot * h->nmm : nullptr;
      break;
    case EPW_DBG_G_TILDE: {
      // strided copy: rows of the g~ buffer are ncols wide, the first Nb^2 Nm entries are g~
      const int64_t rowsC = std::min(h->last_nk, h->last_c_rows);
      need = sizeof(c128) * nbb * h->nm * rowsC;
      if (bytes < need || !h->C.p) return h->fail(EPW_EINVAL, "epw_interp_debug_get: buffer too small or nothing computed");
      CU_OR_FAIL(h,
                 cudaMemcpy2D(dst, sizeof(c128) * nbb * h->nm, h->C.p, sizeof(c128) * (size_t)h->last_ncols,
                              sizeof(c128) * nbb * h->nm, rowsC, cudaMemcpyDeviceToHost),
                 "cudaMemcpy2D g~");
      return (int64_t)need;
    }
    default: return h->fail(EPW_EINVAL, "epw_interp_debug_get: unknown selector");
  }
  if (!src || bytes < need) return h->fail(EPW_EINVAL, "epw_interp_debug_get: buffer too small or nothing computed");
  CU_OR_FAIL(h, cudaMemcpy(dst, src, need, cudaMemcpyDeviceToHost), "cudaMemcpy debug");
  return (int64_t)need;
}

// ---------------------------------------------------------------------------------------------------------
// stage-level entry points
// ---------------------------------------------------------------------------------------------------------
static int rc_of(cudaError_t e) {
  if (e == cudaSuccess) return EPW_OK;
  if (e == cudaErrorInvalidValue) return EPW_EINVAL;
  return e == cudaErrorInvalidConfiguration ? EPW_EUNSUPPORTED : EPW_ECUDA;   // a launcher refused the shape
}

int epw_phase_table(const double *x_list, int64_t nx, const int32_t *R, const double *w, int32_t nr, void *P_out,
                    void *cuda_stream) {
  if (!x_list || !R || !w || !P_out || nx < 0 || nr <= 0) return EPW_EINVAL;
  return rc_of(launch_phase_table(x_list, nx, R, w, nr, reinterpret_cast<c128 *>(P_out),
                                  reinterpret_cast<cudaStream_t>(cuda_stream)));
}

int epw_rp_to_q(const void *g_RR, int64_t rows, int32_t np, const void *Pq, int32_t nq, void *g1_out,
                void *cuda_stream) {
  if (!g_RR || !Pq || !g1_out || rows <= 0 || np <= 0 || nq <= 0 || nq > 8) return EPW_EINVAL;
  return rc_of(launch_rp_to_q(reinterpret_cast<const c128 *>(g_RR), rows, np, reinterpret_cast<const c128 *>(Pq), nq,
                              reinterpret_cast<c128 *>(g1_out), reinterpret_cast<cudaStream_t>(cuda_stream)));
}

int epw_interp_operator(const void *Op_R, int32_t n, int32_t nr, const void *P, int64_t nx, void *out,
                        void *cuda_stream) {
  if (!Op_R || !P || !out || n <= 0 || nr <= 0 || nx < 0) return EPW_EINVAL;
  return rc_of(launch_interp_operator(reinterpret_cast<const c128 *>(Op_R), n, nr, reinterpret_cast<const c128 *>(P),
                                      nx, reinterpret_cast<c128 *>(out), reinterpret_cast<cudaStream_t>(cuda_stream)));
}

int epw_eigh_batched(const void *A, int64_t stride_a, int32_t n, int64_t batch, double *evals, void *V, int sqrt_mode,
                     int32_t *status, void *cuda_stream) {
  return epw_eigh_batched_algo(A, stride_a, n, batch, evals, V, sqrt_mode, status, EPW_EIGH_AUTO, cuda_stream);
}

int epw_eigh_batched_algo(const void *A, int64_t stride_a, int32_t n, int64_t batch, double *evals, void *V,
                          int sqrt_mode, int32_t *status, int algo, void *cuda_stream) {
  if (!A || !evals || !V || n <= 0 || batch < 0 || stride_a < (int64_t)n * n) return EPW_EINVAL;
  if (algo < EPW_EIGH_AUTO || algo > EPW_EIGH_COLS) return EPW_EINVAL;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  c128 *scratch = nullptr;
  const size_t need = eigh_large_scratch_bytes(n, batch);
  if (need && cudaMalloc(&scratch, need) != cudaSuccess) return EPW_ENOMEM;
  const cudaError_t e = launch_eigh_batched_algo(reinterpret_cast<const c128 *>(A), stride_a, n, batch, evals,
                                                 reinterpret_cast<c128 *>(V), sqrt_mode, status, scratch, algo, nullptr, st);
  if (scratch) {  // stage-level convenience path: wait so the scratch can be released
    cudaStreamSynchronize(st);
    cudaFree(scratch);
  }
  return rc_of(e);
}

int epw_zgemm(const void *A, const void *B, void *C, int64_t M, int32_t N, int32_t K, int64_t ldc, void *cuda_stream) {
  if (!A || !B || !C || M <= 0 || N <= 0 || K <= 0 || ldc < N) return EPW_EINVAL;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const int nsm = device_sm_count();
  const int KB = (int)ceil_div(2 * (int64_t)K, GEMM_BK);
  const int NT = (int)ceil_div(2 * (int64_t)N, GEMM_BN);
  const int64_t MT = ceil_div(M, GEMM_BM);
  double *Ap = nullptr, *Bp = nullptr;
  if (cudaMalloc(&Ap, sizeof(double) * (size_t)MT * KB * GEMM_CHUNK) != cudaSuccess) return EPW_ENOMEM;
  if (cudaMalloc(&Bp, sizeof(double) * (size_t)NT * KB * GEMM_CHUNK) != cudaSuccess) {
    cudaFree(Ap);
    return EPW_ENOMEM;
  }
  cudaError_t e = launch_pack_a_generic(reinterpret_cast<const c128 *>(A), M, K, Ap, st);
  if (e == cudaSuccess) e = launch_pack_b_generic(reinterpret_cast<const c128 *>(B), K, N, Bp, st);
  if (e == cudaSuccess) e = launch_zgemm_dmma(Ap, Bp, reinterpret_cast<c128 *>(C), M, N, KB, ldc, nsm, st);
  cudaStreamSynchronize(st);
  cudaFree(Ap);
  cudaFree(Bp);
  return rc_of(e);
}

int epw_zgemm_strided(const void *A, int64_t a_rb, int64_t a_bs, int64_t a_ks, int64_t a_batch, const void *B,
                      int64_t b_sr, int64_t b_sn, int64_t b_batch, int b_conj, const int32_t *b_gather, int64_t nb_mats,
                      void *C, int64_t c_rb, int64_t c_bs, int64_t c_rs, int64_t c_cs, int64_t c_batch, int abs2,
                      int64_t M, int32_t N, int32_t K, int64_t batch, void *cuda_stream) {
  if (!A || !B || !C || M <= 0 || N <= 0 || K <= 0 || batch <= 0 || a_rb <= 0 || c_rb <= 0 || nb_mats <= 0)
    return EPW_EINVAL;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const int nsm = device_sm_count();
  const int KB = (int)ceil_div(2 * (int64_t)K, GEMM_BK);
  const int NT = (int)ceil_div(2 * (int64_t)N, GEMM_BN);
  double *Bp = nullptr;
  if (cudaMalloc(&Bp, sizeof(double) * (size_t)nb_mats * NT * KB * GEMM_CHUNK) != cudaSuccess) return EPW_ENOMEM;
  cudaError_t e = launch_pack_b_strided(reinterpret_cast<const c128 *>(B), b_sr, b_sn, b_batch, nb_mats, b_conj, nullptr,
                                        0.0, K, N, Bp, st);
  if (e == cudaSuccess)
    e = launch_zgemm_strided(reinterpret_cast<const c128 *>(A), a_rb, a_bs, a_ks, a_batch, Bp, b_gather, C, c_rb, c_bs,
                             c_rs, c_cs, c_batch, abs2, M, N, K, batch, nsm, st);
  cudaStreamSynchronize(st);
  cudaFree(Bp);
  return rc_of(e);
}

int epw_axis_pass_dmma(const void *T, int64_t slab, int32_t ncols, int32_t L, const void *P, int32_t cnt, int32_t nb,
                       void *out, int64_t out_stride, int32_t nbatch, int64_t in_bstride, int64_t out_bstride,
                       void *cuda_stream) {
  if (!T || !P || !out || slab <= 0 || ncols <= 0 || L <= 0 || cnt <= 0 || nb <= 0 || nbatch <= 0 || out_stride < ncols)
    return EPW_EINVAL;
  if (nb > 16 || ncols % (nb * nb) != 0 || !grid_pass_dmma_supported(nb, L)) return EPW_EUNSUPPORTED;
  return rc_of(launch_grid_pass_dmma(reinterpret_cast<const c128 *>(T), slab, ncols, L, reinterpret_cast<const c128 *>(P), cnt,
                                     nb, ncols / (nb * nb), device_sm_count(), reinterpret_cast<c128 *>(out), out_stride,
                                     nbatch, in_bstride, out_bstride, reinterpret_cast<cudaStream_t>(cuda_stream)));
}

int epw_rotate_g2(const void *gt, int64_t stride_gt, const void *Uk, const void *Ukq, const int32_t *kq_idx, int32_t nb,
                  int32_t nm, int64_t nk, double *g2, void *cuda_stream) {
  if (!gt || !Uk || !Ukq || !g2 || nb <= 0 || nm <= 0 || nk < 0) return EPW_EINVAL;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const cudaError_t e = launch_rotate_g2(reinterpret_cast<const c128 *>(gt), stride_gt, reinterpret_cast<const c128 *>(Uk),
                                         reinterpret_cast<const c128 *>(Ukq), kq_idx, nb, nm, nk, nullptr, g2, st);
  if (e != cudaErrorInvalidConfiguration) return rc_of(e);
  // large (Nb, Nm): T[(nu,m')][n] = sum_n' g~[(nu,m')][n'] U_k[n'][n];  |g|^2[(nu,n)][m] = |sum_m' T[(nu,n)][m'] conj(Ukq[m'][m])|^2
  cudaGetLastError();
  const int64_t E = (int64_t)nb * nb * nm, MR = (int64_t)nm * nb, nbb = (int64_t)nb * nb;
  if (stride_gt != E) return EPW_EUNSUPPORTED;
  if (nk == 0) return EPW_OK;
  // Ukq may be indexed through kq_idx by values up to the size of the caller's U table: the caller guarantees nk entries
  c128 *T = nullptr;
  if (cudaMalloc(&T, sizeof(c128) * (size_t)nk * E) != cudaSuccess) return EPW_ENOMEM;
  int rc = epw_zgemm_strided(gt, nb, nbb, nb, E, Uk, 1, nb, nbb, 0, nullptr, nk, T, MR, 0, nb, 1, E, 0, MR, nb, nb, nk,
                             cuda_stream);
  if (rc == EPW_OK)
    rc = epw_zgemm_strided(T, nb, nbb, nb, E, Ukq, 1, nb, nbb, 1, kq_idx, nk, g2, MR, 0, nb, 1, E, 1, MR, nb, nb, nk,
                           cuda_stream);
  cudaFree(T);
  return rc;
}

int epw_eq6_unrotate(const void *g_bloch, const void *Uk, const void *Ukq, const void *e_q, const double *omega_q,
                     int32_t nb, int32_t nm, int64_t nkc, int64_t nqc, void *gt_out, void *cuda_stream) {
  if (!g_bloch || !Uk || !Ukq || !e_q || !omega_q || !gt_out || nb <= 0 || nm <= 0 || nkc <= 0 || nqc <= 0)
    return EPW_EINVAL;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  c128 *tmp = nullptr;
  if (cudaMalloc(&tmp, sizeof(c128) * (size_t)nkc * nqc * nb * nb * nm) != cudaSuccess) return EPW_ENOMEM;
  const cudaError_t e = launch_eq6_unrotate(reinterpret_cast<const c128 *>(g_bloch), reinterpret_cast<const c128 *>(Uk),
                                            reinterpret_cast<const c128 *>(Ukq), reinterpret_cast<const c128 *>(e_q),
                                            omega_q, nb, nm, nkc, nqc, tmp, reinterpret_cast<c128 *>(gt_out), st);
  cudaStreamSynchronize(st);
  cudaFree(tmp);
  return rc_of(e);
}

int epw_wannier_from_bloch(const void *gt, const double *kc, int64_t nkc, const double *qc, int64_t nqc, const int32_t *Re,
                           int32_t ne, const int32_t *Rp, int32_t np, int32_t nb, int32_t nm, void *g_RR_out,
                           void *cuda_stream) {
  if (!gt || !kc || !qc || !Re || !Rp || !g_RR_out || nkc <= 0 || nqc <= 0 || ne <= 0 || np <= 0 || nb <= 0 || nm <= 0)
    return EPW_EINVAL;
  if (nkc > 2147483647LL / 2 || nqc > 2147483647LL / 2) return EPW_EINVAL;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const int nsm = device_sm_count();
  const size_t rows = (size_t)nb * nb * nm * ne;
  const size_t packK = (size_t)ceil_div(2 * (int64_t)ne, GEMM_BN) * ceil_div(2 * nkc, GEMM_BK) * GEMM_CHUNK;
  const size_t packQ = (size_t)ceil_div(2 * (int64_t)np, GEMM_BN) * ceil_div(2 * nqc, GEMM_BK) * GEMM_CHUNK;
  // one allocation, carved up (all pieces 16-byte aligned)
  auto al = [](size_t b) { return (b + 255) & ~(size_t)255; };
  const size_t sz[] = {al(sizeof(double) * ne), al(sizeof(double) * np), al(sizeof(c128) * nkc * ne),
                       al(sizeof(c128) * nqc * np), al(sizeof(double) * packK), al(sizeof(double) * packQ),
                       al(sizeof(int32_t) * nqc), al(sizeof(c128) * nqc * rows)};
  size_t total = 0;
  for (size_t b : sz) total += b;
  // grow-only workspace kept between calls, one per device (cudaMalloc + cudaFree of ~1 GB cost more than the two
  // contractions); concurrent callers are serialised by the lock, which is held until the stream has drained
  static std::mutex cache_mu;
  static DevBuf cache_of[64];
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return EPW_ECUDA;
  std::lock_guard<std::mutex> lock(cache_mu);
  DevBuf &cache = cache_of[dev];
  if (cache.reserve(total) != cudaSuccess) return EPW_ENOMEM;
  char *ws = cache.as<char>();
  char *p[8];
  size_t off = 0;
  for (int i = 0; i < 8; i++) { p[i] = ws + off; off += sz[i]; }
  const cudaError_t e = launch_wannier_from_bloch(
      reinterpret_cast<const c128 *>(gt), kc, nkc, qc, nqc, Re, ne, Rp, np, nb, nm, reinterpret_cast<double *>(p[0]),
      reinterpret_cast<double *>(p[1]), reinterpret_cast<c128 *>(p[2]), reinterpret_cast<c128 *>(p[3]),
      reinterpret_cast<double *>(p[4]), reinterpret_cast<double *>(p[5]), reinterpret_cast<int32_t *>(p[6]),
      reinterpret_cast<c128 *>(p[7]), reinterpret_cast<c128 *>(g_RR_out), nsm, st);
  cudaStreamSynchronize(st);
  return rc_of(e);
}

int epw_probe_peaks(int32_t device, double *out4) {
  if (!out4) return EPW_EINVAL;
  return probe_peaks(device, out4);
}

}  // extern "C"
