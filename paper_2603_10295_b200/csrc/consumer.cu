// consumer.cu -- a consumer of |g|^2 on the device: instead of shipping 8 Nb^2 Nm bytes per pair
// to the caller, the |g|^2 block of every pair is reduced, right after the rotation kernel wrote it, into the per-state
// accumulator a downstream module wants.  The paper names the consumers ("ab initio Boltzmann transport", "electron
// self-energy") but prints no formula; the one built here is [DESIGN.md reading G18] the imaginary
// part of the Fan-Migdal self-energy with Gaussian-broadened energy conservation,
//   Im Sigma_nk += pi w_q sum_{m,nu} |g_{mn nu}(k,q)|^2 [ (n_qnu + f_mk+q)     delta_s(e_nk - e_mk+q + w_qnu)
//                                                      + (n_qnu + 1 - f_mk+q) delta_s(e_nk - e_mk+q - w_qnu) ],
//   delta_s(x) = exp(-(x/s)^2)/(s sqrt(pi)),  n = 1/expm1(w/kT),  f = 1/(exp((e - mu)/kT) + 1),  modes with w <= 0 skipped.
// One thread per (k, n); the sum over (nu, m) runs in a fixed order and q-points are accumulated in call order on one
// stream, so the result is deterministic.  With the consumer on, the caller may pass g2 = NULL: the library then keeps
// |g|^2 of one q at a time in its own scratch and nothing of size Nk Nq ever exists.
#include "common.cuh"

namespace epw {

__global__ void __launch_bounds__(256)
    selfenergy_accumulate_kernel(const double *__restrict__ g2q, const double *__restrict__ eps_k,
                                 const double *__restrict__ eps_kq, const double *__restrict__ eps_k_all,
                                 const int32_t *__restrict__ kq_idx, const double *__restrict__ omega_q,
                                 const double *__restrict__ w_q, int64_t iq, double mu, double kT, double sigma, int nb,
                                 int nm, int64_t nk, double *__restrict__ out) {
  const double inv_s = 1.0 / sigma, norm = inv_s * 0.56418958354775628695;  // 1/(s sqrt(pi))
  const double wq = w_q ? w_q[iq] : 1.0;
  const int64_t total = nk * nb;
  for (int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
    const int64_t ik = idx / nb;
    const int n = (int)(idx - ik * nb);
    const double e1 = eps_k[ik * nb + n];
    const double *e2 = kq_idx ? eps_k_all + (int64_t)kq_idx[ik] * nb : eps_kq + ik * nb;
    const double *blk = g2q + ik * (int64_t)nb * nb * nm;
    double s = 0.0;
    for (int nu = 0; nu < nm; nu++) {
      const double w = omega_q[nu];
      if (!(w > 0.0)) continue;
      const double *row = blk + ((int64_t)nu * nb + n) * nb;
      double bose = -1.0;  // evaluated on first use
      for (int m = 0; m < nb; m++) {
        const double em = e2[m];
        const double xa = (e1 - em + w) * inv_s, xe = (e1 - em - w) * inv_s;
        // a Gaussian below e^-50 = 2e-22 of its peak cannot reach the last bit of the sum: most (m, nu) terms of a
        // realistic broadening are skipped without evaluating any exponential
        const bool ka = xa * xa < 50.0, ke = xe * xe < 50.0;
        if (!ka && !ke) continue;
        if (bose < 0.0) bose = 1.0 / expm1(w / kT);   // expm1: no cancellation when w << kT
        const double f = 1.0 / (exp((em - mu) / kT) + 1.0);
        const double da = ka ? exp(-xa * xa) : 0.0, de = ke ? exp(-xe * xe) : 0.0;
        s += row[m] * ((bose + f) * da + (bose + 1.0 - f) * de);
      }
    }
    out[idx] += 3.14159265358979323846 * wq * norm * s;
  }
}

cudaError_t launch_selfenergy_accumulate(const double *g2q, const double *eps_k, const double *eps_kq,
                                         const double *eps_k_all, const int32_t *kq_idx, const double *omega_q,
                                         const double *w_q, int64_t iq, double mu, double kT, double sigma, int nb, int nm,
                                         int64_t nk, double *out, cudaStream_t st) {
  if (nk <= 0) return cudaSuccess;
  const int64_t blocks = ceil_div(nk * nb, 256);
  selfenergy_accumulate_kernel<<<grid_cap(blocks, 16), 256, 0, st>>>(
      g2q, eps_k, eps_kq, eps_k_all, kq_idx, omega_q, w_q, iq, mu, kT, sigma, nb, nm, nk, out);
  return cudaGetLastError();
}

}  // namespace epw
