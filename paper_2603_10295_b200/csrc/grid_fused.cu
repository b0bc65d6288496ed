// grid_fused.cu -- dispatch of the one-kernel last axis pass + S4b (grid_fused.cuh) over Nb.  The kernel templates are
// instantiated in four translation units (grid_fused_nb*.cu, four values of Nb each) so that they compile in parallel.
#include "grid_fused.cuh"

namespace epw {

cudaError_t launch_gf_nb1(int nb, const GridFusedParams &p, int num_sms, cudaStream_t st);
cudaError_t launch_gf_nb5(int nb, const GridFusedParams &p, int num_sms, cudaStream_t st);
cudaError_t launch_gf_nb9(int nb, const GridFusedParams &p, int num_sms, cudaStream_t st);
cudaError_t launch_gf_nb13(int nb, const GridFusedParams &p, int num_sms, cudaStream_t st);

static cudaError_t gf_dispatch(int nb, const GridFusedParams &p, int num_sms, cudaStream_t st) {
  if (nb < 1 || nb > 16) return cudaErrorInvalidConfiguration;
  if (nb <= 4) return launch_gf_nb1(nb, p, num_sms, st);
  if (nb <= 8) return launch_gf_nb5(nb, p, num_sms, st);
  if (nb <= 12) return launch_gf_nb9(nb, p, num_sms, st);
  return launch_gf_nb13(nb, p, num_sms, st);
}

bool grid_fused_supported(int nb, int nm, int L1) {
  if (nb < 1 || nb > 16 || nm < 1) return false;
  int nug = 0, nbuf = 0;
  size_t smem = 0;
  switch (nb) {
#define EPW_GF_CASE(NB_) \
  case NB_: return gf_plan<NB_>(nm, L1, 1, &nug, &nbuf, &smem);
    EPW_GF_CASE(1) EPW_GF_CASE(2) EPW_GF_CASE(3) EPW_GF_CASE(4) EPW_GF_CASE(5) EPW_GF_CASE(6) EPW_GF_CASE(7) EPW_GF_CASE(8)
    EPW_GF_CASE(9) EPW_GF_CASE(10) EPW_GF_CASE(11) EPW_GF_CASE(12) EPW_GF_CASE(13) EPW_GF_CASE(14) EPW_GF_CASE(15)
    EPW_GF_CASE(16)
#undef EPW_GF_CASE
    default: return false;
  }
}

// T2 c128 [L1][slab][ncols] (the g columns are the first Nb^2 Nm of each row); P1c c128 [L1][cnt]: phases of the cnt
// i1 planes of this chunk; Uk, Ukq, kq_idx, mask, g2 are relative to the first k of the chunk (k = j*slab + cell).
cudaError_t launch_grid_fused(const c128 *T2, int64_t slab, int ncols, int L1, const c128 *P1c, int cnt, const c128 *Uk,
                              const c128 *Ukq, const int32_t *kq_idx, int nb, int nm, int num_sms, const uint8_t *mask,
                              double *g2, const SelfEnergyFold *fold, cudaStream_t st) {
  if (slab <= 0 || cnt <= 0) return cudaSuccess;
  if (g2 == nullptr && fold == nullptr) return cudaErrorInvalidValue;
  GridFusedParams p = {};
  p.T2 = T2; p.slab = slab; p.ncols = ncols; p.L1 = L1; p.cnt = cnt; p.P1c = P1c;
  p.Uk = Uk; p.Ukq = Ukq; p.kq_idx = kq_idx; p.nm = nm; p.mask = mask; p.g2 = g2; p.nbatch = 1;
  if (fold) {
    p.cons_out = fold->out; p.eps_k = fold->eps_k; p.eps_kq = fold->eps_kq; p.omega_q = fold->omega_q; p.w_q = fold->w_q;
    p.iq = fold->iq; p.mu = fold->mu; p.kT = fold->kT; p.sigma = fold->sigma;
  }
  return gf_dispatch(nb, p, num_sms, st);
}

// The last axis pass ALONE as the same DMMA product: gt c128 [cnt*slab][gt_stride] <- g~ (first Nb^2 Nm columns of each row).
// nbatch problems of that shape: input b at T2 + b * in_bstride, output b at gt + b * out_bstride (any axis of the factorised
// transform is such a batch: the contracted index outermost within a block, the blocks one after the other).
cudaError_t launch_grid_pass_dmma(const c128 *T2, int64_t slab, int ncols, int L1, const c128 *P1c, int cnt, int nb, int nm,
                                  int num_sms, c128 *gt, int64_t gt_stride, int nbatch, int64_t in_bstride,
                                  int64_t out_bstride, cudaStream_t st) {
  if (slab <= 0 || cnt <= 0 || nbatch <= 0) return cudaSuccess;
  if (gt == nullptr) return cudaErrorInvalidValue;
  GridFusedParams p = {};
  p.T2 = T2; p.slab = slab; p.ncols = ncols; p.L1 = L1; p.cnt = cnt; p.P1c = P1c; p.nm = nm; p.gt = gt; p.gt_stride = gt_stride;
  p.nbatch = nbatch; p.in_bstride = in_bstride; p.out_bstride = out_bstride;
  return gf_dispatch(nb, p, num_sms, st);
}

// whether that kernel takes a pass with K = L lattice vectors on column groups of nb^2
bool grid_pass_dmma_supported(int nb, int L) {
  if (nb < 1 || nb > 16) return false;
  int nug = 0, nbuf = 0;
  size_t smem = 0;
  switch (nb) {
#define EPW_GF_CASE(NB_) \
  case NB_: return gf_plan<NB_>(1, L, 2, &nug, &nbuf, &smem);
    EPW_GF_CASE(1) EPW_GF_CASE(2) EPW_GF_CASE(3) EPW_GF_CASE(4) EPW_GF_CASE(5) EPW_GF_CASE(6) EPW_GF_CASE(7) EPW_GF_CASE(8)
    EPW_GF_CASE(9) EPW_GF_CASE(10) EPW_GF_CASE(11) EPW_GF_CASE(12) EPW_GF_CASE(13) EPW_GF_CASE(14) EPW_GF_CASE(15)
    EPW_GF_CASE(16)
#undef EPW_GF_CASE
    default: return false;
  }
}

}  // namespace epw
