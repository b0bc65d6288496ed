// bloch_to_wannier.cu -- Eq. 6, the step BEFORE the hot path: coarse-grid Bloch-representation
// matrix elements g_{mn nu}(k',q') -> the Wannier-representation operator g_{m'n' ka}(Re,Rp) that
// epw_interp_set_wannier_operators takes (the paper names its GPU port as ongoing work, L289).
//
//   g(Re,Rp) = 1/(Ne Np) sum_{k'q'} [ sum_{mn nu} g_{mn nu}(k',q') U*_{mm'k'+q'} U_{nn'k'} u^-1_{nu,ka}(q') ] e^{-i(q'.Rp + k'.Re)}
//
// Two entry points, the inverse of the interpolation path stage by stage:
//   epw_eq6_unrotate        the bracket (gauge part): with paper-U = V^dagger (reading G4) and
//                           u = e/sqrt(2 omega) (reading G3)
//                             g~_{m'n' ka} = sum_{mn nu} Ukq[m',m] g_{mn nu} conj(Uk[n',n]) sqrt(2 omega_nu) conj(e[ka,nu])
//                           -- three small products per (k',q') block, one thread per output element (coarse grids are
//                           10^2..10^3 points: this is preprocessing, not a throughput kernel);
//   epw_wannier_from_bloch  the two inverse Fourier sums, as two launches of the in-place FP64 tensor-path contraction of
//                           the large-Nb path (zgemm_strided.cu) with conjugated phase tables as the packed B operand:
//                             g(Re,q')[ka][Re][el] = 1/Ne sum_k' g~(k',q')[ka][el] e^{-2 pi i k'.Re}     (batched over q')
//                             g(Re,Rp)[Rp][row]    = 1/Np sum_q' g(Re,q')[row]     e^{-2 pi i q'.Rp}     row = (ka,Re,el)
//                           and the result is already in the layout of g_RR (Fig. 13's A(m,n), Rp the column).
#include "common.cuh"

namespace epw {

// out[b][x][y] (c128) for one of the three products; `which` selects the contraction, b = (iq, ik) block.
//   0: T[nu][n][m']   = sum_m  Ukq[m' + nb m]       g[nu][n][m]
//   1: W[nu][n'][m']  = sum_n  T[nu][n][m']         conj(Uk[n' + nb n])
//   2: gt[ka][n'][m'] = sum_nu W[nu][n'][m']        sqrt(2 omega_nu) conj(e[ka + nm nu])
__global__ void __launch_bounds__(256)
    eq6_unrotate_kernel(int which, const c128 *__restrict__ in, const c128 *__restrict__ Uk, const c128 *__restrict__ Ukq,
                        const c128 *__restrict__ e, const double *__restrict__ omega, int nb, int nm, int64_t nkc,
                        int64_t nblocks, c128 *__restrict__ out) {
  const int nbb = nb * nb;
  const int64_t E = (int64_t)nbb * nm;
  const int64_t total = nblocks * E;
  for (int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; idx < total;
       idx += (int64_t)gridDim.x * blockDim.x) {
    const int64_t b = idx / E;
    const int r = (int)(idx - b * E);
    const int v = r / nbb, y = (r - v * nbb) / nb, x = r - v * nbb - y * nb;   // element [v][y][x], x fastest
    const c128 *src = in + b * E;
    c128 acc = cmake(0.0, 0.0);
    if (which == 0) {
      const c128 *u = Ukq + b * nbb;
      for (int m = 0; m < nb; m++) cfma(acc, u[x + nb * m], src[(int64_t)v * nbb + y * nb + m]);
    } else if (which == 1) {
      const c128 *u = Uk + (b % nkc) * nbb;
      for (int n = 0; n < nb; n++) cfma_conj(acc, u[y + nb * n], src[(int64_t)v * nbb + n * nb + x]);
    } else {
      const int64_t iq = b / nkc;
      const c128 *eq = e + iq * nm * nm;
      const double *om = omega + iq * nm;
      for (int nu = 0; nu < nm; nu++) {
        const double amp = sqrt(2.0 * om[nu]);
        const c128 w = src[(int64_t)nu * nbb + y * nb + x];
        cfma_conj(acc, eq[v + nm * nu], cmake(amp * w.x, amp * w.y));
      }
    }
    out[idx] = acc;
  }
}

cudaError_t launch_eq6_unrotate(const c128 *g, const c128 *Uk, const c128 *Ukq, const c128 *e, const double *omega, int nb,
                                int nm, int64_t nkc, int64_t nqc, c128 *tmp, c128 *gt, cudaStream_t st) {
  const int64_t nblocks = nkc * nqc;
  const int64_t total = nblocks * nb * nb * nm;
  if (total <= 0) return cudaSuccess;
  const int64_t want = ceil_div(total, 256);
  const unsigned grid = grid_cap(want, 32);
  eq6_unrotate_kernel<<<grid, 256, 0, st>>>(0, g, Uk, Ukq, e, omega, nb, nm, nkc, nblocks, gt);
  eq6_unrotate_kernel<<<grid, 256, 0, st>>>(1, gt, Uk, Ukq, e, omega, nb, nm, nkc, nblocks, tmp);
  eq6_unrotate_kernel<<<grid, 256, 0, st>>>(2, tmp, Uk, Ukq, e, omega, nb, nm, nkc, nblocks, gt);
  return cudaGetLastError();
}

__global__ void fill_value_kernel(double *p, int n, double v) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = v;
}

// Workspace (doubles unless stated): wk[ne], wq[np], Pk c128 [nkc][ne], Pq c128 [nqc][np], packed tables, zero gather
// [nqc] int32, g1 c128 [nqc][rows].  All sized and owned by the caller (interp.cu).
cudaError_t launch_wannier_from_bloch(const c128 *gt, const double *kc, int64_t nkc, const double *qc, int64_t nqc,
                                      const int32_t *Re, int ne, const int32_t *Rp, int np, int nb, int nm, double *wk,
                                      double *wq, c128 *Pk, c128 *Pq, double *BpackK, double *BpackQ, int32_t *zero_gather,
                                      c128 *g1, c128 *g_RR, int num_sms, cudaStream_t st) {
  const int nbb = nb * nb;
  const int64_t E = (int64_t)nbb * nm, rows = E * ne;
  fill_value_kernel<<<(ne + 255) / 256, 256, 0, st>>>(wk, ne, 1.0 / (double)ne);
  fill_value_kernel<<<(np + 255) / 256, 256, 0, st>>>(wq, np, 1.0 / (double)np);
  cudaError_t e = cudaMemsetAsync(zero_gather, 0, sizeof(int32_t) * (size_t)nqc, st);
  if (e != cudaSuccess) return e;
  // conjugated, normalised phase tables as packed B operands: B[r = k'][col = Re] = e^{-2 pi i k'.Re}/Ne
  e = launch_phase_table(kc, nkc, Re, wk, ne, Pk, st);
  if (e != cudaSuccess) return e;
  e = launch_pack_b_strided(Pk, ne, 1, 0, 1, 1, nullptr, 0.0, (int)nkc, ne, BpackK, st);
  if (e != cudaSuccess) return e;
  e = launch_phase_table(qc, nqc, Rp, wq, np, Pq, st);
  if (e != cudaSuccess) return e;
  e = launch_pack_b_strided(Pq, np, 1, 0, 1, 1, nullptr, 0.0, (int)nqc, np, BpackQ, st);
  if (e != cudaSuccess) return e;
  // k' -> Re for every q':  rows (ka,el) of g~(k',q') are contiguous for fixed k'; C = g(Re,q')[ka][Re][el]
  e = launch_zgemm_strided(gt, E, 0, E, nkc * E, BpackK, zero_gather, g1, nbb, (int64_t)ne * nbb, 1, nbb, rows, 0, E, ne,
                           (int)nkc, nqc, num_sms, st);
  if (e != cudaSuccess) return e;
  // q' -> Rp:  rows (ka,Re,el) contiguous for fixed q'; C = g_RR[Rp][row]
  return launch_zgemm_strided(g1, rows, 0, rows, 0, BpackQ, nullptr, g_RR, rows, 0, 1, rows, 0, 0, rows, np, (int)nqc, 1,
                              num_sms, st);
}

}  // namespace epw
