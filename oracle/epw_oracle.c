/*
 * epw_oracle.c -- CPU ORACLE for the Wannier-to-Bloch interpolation of
 * electron-phonon matrix elements (arxiv/paper_2603_10295, EPW 6.1).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, the smoke check
 * in __graft_entry__.py and bench.py's cpu_baseline / --impl reference legs may
 * call it.  It shares no code with the CUDA library in paper_2603_10295_b200/;
 * the two meet only in the seeded inputs produced by synth/.
 *
 * It is deliberately plain and slow: the paper's definitions written out as
 * explicit loops in complex FP64 ("double-precision arithmetic
 * throughout"), in the paper's order and notation, with its own cyclic Jacobi
 * eigensolver.  No blocking, fusion or reordering beyond what the equations
 * state.  Citations are PAPER.md:L<line> (+ equation); "[north_star]" marks
 * the parts the paper leaves implicit and BASELINE.json fixes; "[reading Gn]"
 * refers to the numbered readings in DESIGN.md / SURVEY.md section 8(c).
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`):
 *   Eq. 9 + FT part of Eq. 10 ..... coarse-grid round trip against numpy.fft, single R=0 term,
 *                                   periodicity, brute-force Eq. 7 path, 1-D chain closed form
 *   operator interpolation ........ closed form eps(k) = e0 + 2t cos(2 pi k), Hermiticity
 *   Jacobi eigensolver ............ residuals, unitarity, 2x2 closed form, numpy.linalg.eigh
 *   rotations and 1/sqrt(2 omega) . unitarity sum rules, diagonal case, gauge invariance, linearity
 *   The paper prints no numerical value of g, eps or omega, so element values are pinned
 *   only by those invariants; size and multiply-count helpers are pinned by Table III / Eq. 12.
 *
 * Index conventions ("Fortran": first index fastest), all complex128:
 *   g_RR [m' + Nb*(n' + Nb*(ie + Ne*(ka + Nm*ip)))]   PAPER.md:L60 (Eq. 3), L501-511 (Fig. 13: A(m,n), n = Rp)
 *   g1   [m' + Nb*(n' + Nb*(ie + Ne*ka))]             g(Re,q),  PAPER.md:L110 (Eq. 9)
 *   gt   [m' + Nb*(n' + Nb*ka)]                       Wannier-gauge g~(k,q) after the Re sum
 *   H_R  [i + Nb*(j + Nb*ie)],  D_R [a + Nm*(b + Nm*ip)]
 *   matrices A[i + n*j] (column-major), eigenvectors are the COLUMNS of V
 *   g2   [m + Nb*(n + Nb*nu)]  = |g_{mn nu}(k,q)|^2
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex zc;

#define TWO_PI 6.283185307179586476925286766559

/* ---------------------------------------------------------------------------------------------
 * Phase  phi = 2 pi frac(x . R),  x in crystal coordinates, R an integer lattice vector.
 * PAPER.md:L84 (Eq. 7), L110 (Eq. 9), L114 (Eq. 10): the factor is exp(+i(q.Rp + k.Re)).
 * [reading G8] crystal coordinates, integer R, factor 2 pi.
 * ------------------------------------------------------------------------------------------- */
double oracle_phase(const double x[3], const int32_t R[3]) {
  double t = x[0] * (double)R[0] + x[1] * (double)R[1] + x[2] * (double)R[2];
  t -= floor(t); /* frac: exp(2 pi i t) has period 1 in t */
  return TWO_PI * t;
}

static zc expi(double phi) { return cos(phi) + I * sin(phi); }

/* ---------------------------------------------------------------------------------------------
 * Eq. 9:  g(Re,q) = sum_Rp g(Re,Rp) exp(i q.Rp), with the Wigner-Seitz weight
 * w_p(Rp) multiplying each term ([reading G7]; all configs use w = 1).
 * ------------------------------------------------------------------------------------------- */
void oracle_rp_to_q(int nb, int nm, int ne, int np, const zc *g_RR, const int32_t *Rp, const double *w_p,
                    const double q[3], zc *g1) {
  const int64_t rows = (int64_t)nb * nb * ne * nm;
  for (int64_t r = 0; r < rows; r++) g1[r] = 0.0;
  for (int ip = 0; ip < np; ip++) {
    const zc f = w_p[ip] * expi(oracle_phase(q, Rp + 3 * ip));
    const zc *col = g_RR + (int64_t)ip * rows;
    for (int64_t r = 0; r < rows; r++) g1[r] += col[r] * f;
  }
}

/* ---------------------------------------------------------------------------------------------
 * Fourier-transform part of Eq. 10, PAPER.md:L112-114:
 *   g~_{m'n' ka}(k,q) = sum_Re g_{m'n' ka}(Re,q) exp(i k.Re)   (weight w_e(Re), [reading G7]).
 * ------------------------------------------------------------------------------------------- */
void oracle_re_to_k(int nb, int nm, int ne, const zc *g1, const int32_t *Re, const double *w_e,
                    const double k[3], zc *gt) {
  const int nbb = nb * nb;
  for (int ka = 0; ka < nm; ka++)
    for (int e = 0; e < nbb; e++) {
      zc s = 0.0;
      for (int ie = 0; ie < ne; ie++) {
        const zc f = w_e[ie] * expi(oracle_phase(k, Re + 3 * ie));
        s += g1[e + (int64_t)nbb * (ie + (int64_t)ne * ka)] * f;
      }
      gt[e + nbb * ka] = s;
    }
}

/* ---------------------------------------------------------------------------------------------
 * Operator interpolation [north_star stage 3; reading G6]:
 *   Op(x) = sum_R w(R) exp(2 pi i x.R) Op(R)      (H(R) -> H(k), D(Rp) -> D(q)),
 * followed by the numerical symmetrisation (A + A^dagger)/2.
 * out[i + n*j].
 * ------------------------------------------------------------------------------------------- */
void oracle_interp_operator(int n, int nr, const zc *Op_R, const int32_t *R, const double *w, const double x[3],
                            zc *out) {
  const int nn = n * n;
  for (int e = 0; e < nn; e++) out[e] = 0.0;
  for (int ir = 0; ir < nr; ir++) {
    const zc f = w[ir] * expi(oracle_phase(x, R + 3 * ir));
    for (int e = 0; e < nn; e++) out[e] += f * Op_R[e + (int64_t)nn * ir];
  }
  for (int i = 0; i < n; i++)
    for (int j = i; j < n; j++) {
      const zc a = 0.5 * (out[i + n * j] + conj(out[j + n * i]));
      out[i + n * j] = a;
      out[j + n * i] = conj(a);
    }
}

/* ---------------------------------------------------------------------------------------------
 * Cyclic complex-Hermitian Jacobi eigensolver [north_star: "its own Jacobi eigensolver"].
 * A = V diag(lambda) V^dagger, lambda ascending, eigenvectors = columns of V.
 * For each (p,q), p<q, with a_pq = r e^{i phi}:
 *   tau = (a_qq - a_pp)/(2r),  t = sgn(tau)/(|tau| + sqrt(1+tau^2)),  c = 1/sqrt(1+t^2),  s = t c
 *   J_pp = c, J_pq = s, J_qp = -s e^{-i phi}, J_qq = c e^{-i phi};   A <- J^dagger A J,  V <- V J
 * (the phase e^{-i phi} turns the 2x2 block real symmetric, then the textbook real rotation
 * annihilates it).  Both sides of the similarity are applied in full -- no symmetry shortcuts.
 * Stop when the off-diagonal Frobenius norm <= 1e-15 * ||A||_F, at most 60 sweeps.
 * Returns the number of sweeps used, or -1 if not converged.
 * ------------------------------------------------------------------------------------------- */
int oracle_eigh_jacobi(int n, const zc *A_in, double *evals, zc *V) {
  zc *A = (zc *)malloc(sizeof(zc) * n * n);
  memcpy(A, A_in, sizeof(zc) * n * n);
  for (int j = 0; j < n; j++)
    for (int i = 0; i < n; i++) V[i + n * j] = (i == j) ? 1.0 : 0.0;
  double fro2 = 0.0;
  for (int e = 0; e < n * n; e++) fro2 += creal(A[e]) * creal(A[e]) + cimag(A[e]) * cimag(A[e]);
  const double thresh2 = 1e-30 * fro2;
  int sweeps = -1;
  for (int sweep = 0; sweep <= 60; sweep++) {
    double off2 = 0.0;
    for (int j = 0; j < n; j++)
      for (int i = 0; i < n; i++)
        if (i != j) off2 += creal(A[i + n * j]) * creal(A[i + n * j]) + cimag(A[i + n * j]) * cimag(A[i + n * j]);
    if (off2 <= thresh2) { sweeps = sweep; break; }
    if (sweep == 60) break;
    for (int p = 0; p < n - 1; p++)
      for (int q = p + 1; q < n; q++) {
        const zc apq = A[p + n * q];
        const double r = cabs(apq);
        if (r == 0.0) continue;
        const zc eiphi = apq / r;          /* e^{ i phi} */
        const zc emiphi = conj(eiphi);     /* e^{-i phi} */
        const double tau = (creal(A[q + n * q]) - creal(A[p + n * p])) / (2.0 * r);
        const double t = (tau >= 0.0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
        const double c = 1.0 / sqrt(1.0 + t * t);
        const double s = t * c;
        /* columns: A <- A J */
        for (int i = 0; i < n; i++) {
          const zc aip = A[i + n * p], aiq = A[i + n * q];
          A[i + n * p] = c * aip - s * emiphi * aiq;
          A[i + n * q] = s * aip + c * emiphi * aiq;
        }
        /* rows: A <- J^dagger A */
        for (int j = 0; j < n; j++) {
          const zc apj = A[p + n * j], aqj = A[q + n * j];
          A[p + n * j] = c * apj - s * eiphi * aqj;
          A[q + n * j] = s * apj + c * eiphi * aqj;
        }
        A[p + n * q] = 0.0;
        A[q + n * p] = 0.0;
        A[p + n * p] = creal(A[p + n * p]);
        A[q + n * q] = creal(A[q + n * q]);
        /* eigenvectors: V <- V J */
        for (int i = 0; i < n; i++) {
          const zc vip = V[i + n * p], viq = V[i + n * q];
          V[i + n * p] = c * vip - s * emiphi * viq;
          V[i + n * q] = s * vip + c * emiphi * viq;
        }
      }
  }
  /* ascending order (selection sort; permute the columns of V along) */
  for (int i = 0; i < n; i++) evals[i] = creal(A[i + n * i]);
  for (int i = 0; i < n - 1; i++) {
    int m = i;
    for (int j = i + 1; j < n; j++)
      if (evals[j] < evals[m]) m = j;
    if (m != i) {
      const double tmp = evals[i]; evals[i] = evals[m]; evals[m] = tmp;
      for (int r = 0; r < n; r++) { const zc v = V[r + n * i]; V[r + n * i] = V[r + n * m]; V[r + n * m] = v; }
    }
  }
  free(A);
  return sweeps;
}

/* omega_nu = sqrt(lambda_nu) for lambda_nu > 0, else -sqrt(-lambda_nu) (imaginary frequency reported
 * as negative) [north_star stage 3; reading G12]. */
void oracle_omega_from_lambda(int nm, const double *lambda, double *omega) {
  for (int nu = 0; nu < nm; nu++) omega[nu] = lambda[nu] > 0.0 ? sqrt(lambda[nu]) : -sqrt(-lambda[nu]);
}

/* ---------------------------------------------------------------------------------------------
 * Mode rotation and zero-point amplitude, PAPER.md:L114 (Eq. 10, factor u_{ka,nu}(q)) with
 * [north_star; reading G3]: u = e_{q,ka,nu}/sqrt(2 omega_{q nu}), e = orthonormal eigenvectors of D(q):
 *   g^_{m'n' nu} = sum_ka g~_{m'n' ka} e[ka,nu] / sqrt(2 omega_nu)
 * Modes with omega_nu <= omega_min are set to zero [reading G12].
 * ------------------------------------------------------------------------------------------- */
void oracle_mode_rotate(int nb, int nm, const zc *gt, const zc *e, const double *omega, double omega_min, zc *gh) {
  const int nbb = nb * nb;
  for (int nu = 0; nu < nm; nu++)
    for (int el = 0; el < nbb; el++) {
      zc s = 0.0;
      for (int ka = 0; ka < nm; ka++) s += gt[el + nbb * ka] * e[ka + nm * nu];
      gh[el + nbb * nu] = (omega[nu] > omega_min) ? s / sqrt(2.0 * omega[nu]) : 0.0;
    }
}

/* ---------------------------------------------------------------------------------------------
 * Band rotation, PAPER.md:L114 (Eq. 10: U_{mm' k+q} ... U*_{nn' k}) with [reading G4]
 * paper-U = V^dagger (V = eigenvector columns of H^W):
 *   g_{mn nu} = sum_{m'n'} conj(Ukq[m',m]) g^_{m'n' nu} Uk[n',n]
 * ------------------------------------------------------------------------------------------- */
void oracle_band_rotate(int nb, int nm, const zc *gh, const zc *Ukq, const zc *Uk, zc *g) {
  /* "a successive multiplication of ... U_{mm'k+q}, U*_{nn'k}": two plain matrix
   * products per mode, T = U_{k+q}^dagger g^, then g = T U_k. */
  zc *T = (zc *)malloc(sizeof(zc) * nb * nb);
  for (int nu = 0; nu < nm; nu++) {
    const zc *ghn = gh + (int64_t)nb * nb * nu;
    for (int np_ = 0; np_ < nb; np_++)
      for (int m = 0; m < nb; m++) {
        zc s = 0.0;
        for (int mp = 0; mp < nb; mp++) s += conj(Ukq[mp + nb * m]) * ghn[mp + nb * np_];
        T[m + nb * np_] = s;
      }
    for (int n = 0; n < nb; n++)
      for (int m = 0; m < nb; m++) {
        zc s = 0.0;
        for (int np_ = 0; np_ < nb; np_++) s += T[m + nb * np_] * Uk[np_ + nb * n];
        g[m + nb * (n + nb * nu)] = s;
      }
  }
  free(T);
}

/* ---------------------------------------------------------------------------------------------
 * One (k,q) pair given g(Re,q) and the phonon eigen-system of this q (nested-loop algorithm,
 * PAPER.md:L106-116, Fig. 1b: Eq. 9 once per q, Eq. 10 per k).
 * Outputs: g2[m + Nb*(n + Nb*nu)] = |g_{mn nu}|^2, eps_k[Nb], eps_kq[Nb]; optionally the complex g.
 * k+q is used un-folded (phases are 1-periodic because R is integer, [reading G9]).
 * Returns 0, or -1 if an eigensolve did not converge.
 * ------------------------------------------------------------------------------------------- */
int oracle_pair(int nb, int nm, int ne, const zc *g1, const zc *H_R, const int32_t *Re, const double *w_e,
                const zc *e_q, const double *omega_q, double omega_min, const double k[3], const double q[3],
                double *g2, double *eps_k, double *eps_kq, zc *g_out) {
  const int nbb = nb * nb;
  zc *gt = (zc *)malloc(sizeof(zc) * nbb * nm);
  zc *gh = (zc *)malloc(sizeof(zc) * nbb * nm);
  zc *g = (zc *)malloc(sizeof(zc) * nbb * nm);
  zc *Hk = (zc *)malloc(sizeof(zc) * nbb), *Hkq = (zc *)malloc(sizeof(zc) * nbb);
  zc *Uk = (zc *)malloc(sizeof(zc) * nbb), *Ukq = (zc *)malloc(sizeof(zc) * nbb);
  const double kq[3] = {k[0] + q[0], k[1] + q[1], k[2] + q[2]};
  int rc = 0;
  oracle_re_to_k(nb, nm, ne, g1, Re, w_e, k, gt);
  oracle_interp_operator(nb, ne, H_R, Re, w_e, k, Hk);
  oracle_interp_operator(nb, ne, H_R, Re, w_e, kq, Hkq);
  if (oracle_eigh_jacobi(nb, Hk, eps_k, Uk) < 0) rc = -1;
  if (oracle_eigh_jacobi(nb, Hkq, eps_kq, Ukq) < 0) rc = -1;
  oracle_mode_rotate(nb, nm, gt, e_q, omega_q, omega_min, gh);
  oracle_band_rotate(nb, nm, gh, Ukq, Uk, g);
  for (int e = 0; e < nbb * nm; e++) g2[e] = creal(g[e]) * creal(g[e]) + cimag(g[e]) * cimag(g[e]);
  if (g_out) memcpy(g_out, g, sizeof(zc) * nbb * nm);
  free(gt); free(gh); free(g); free(Hk); free(Hkq); free(Uk); free(Ukq);
  return rc;
}

/* Phonon side of one q: D(q) -> e_q (columns), omega_q.  Returns 0 or -1. */
int oracle_phonon(int nm, int np, const zc *D_R, const int32_t *Rp, const double *w_p, const double q[3], zc *e_q,
                  double *omega_q) {
  zc *Dq = (zc *)malloc(sizeof(zc) * nm * nm);
  double *lam = (double *)malloc(sizeof(double) * nm);
  oracle_interp_operator(nm, np, D_R, Rp, w_p, q, Dq);
  const int rc = oracle_eigh_jacobi(nm, Dq, lam, e_q) < 0 ? -1 : 0;
  oracle_omega_from_lambda(nm, lam, omega_q);
  free(Dq); free(lam);
  return rc;
}

/* ---------------------------------------------------------------------------------------------
 * The whole path over lists, mirroring the C ABI of the CUDA library on HOST pointers
 * (nested-loop algorithm, Fig. 12: outer q loop, inner k loop).
 *   eps_k [nk][Nb], eps_kq [nq][nk][Nb] (may be NULL), omega_q [nq][Nm], g2 [nq][nk][Nm][Nb][Nb].
 * OpenMP only across the independent k of one q.
 * ------------------------------------------------------------------------------------------- */
int oracle_interpolate(int nb, int nm, int ne, int np, const zc *H_R, const zc *D_R, const zc *g_RR,
                       const int32_t *Re, const double *w_e, const int32_t *Rp, const double *w_p, double omega_min,
                       const double *k_list, int64_t nk, const double *q_list, int64_t nq, double *eps_k,
                       double *eps_kq, double *omega_q, double *g2) {
  const int64_t E = (int64_t)nb * nb * nm;
  zc *g1 = (zc *)malloc(sizeof(zc) * E * ne);
  zc *e_q = (zc *)malloc(sizeof(zc) * nm * nm);
  int rc = 0;
  for (int64_t iq = 0; iq < nq; iq++) {
    const double *q = q_list + 3 * iq;
    oracle_rp_to_q(nb, nm, ne, np, g_RR, Rp, w_p, q, g1);
    if (oracle_phonon(nm, np, D_R, Rp, w_p, q, e_q, omega_q + iq * nm)) rc = -1;
#pragma omp parallel for schedule(dynamic, 4) reduction(min : rc)
    for (int64_t ik = 0; ik < nk; ik++) {
      double ek[512], ekq[512];
      double *ek_p = nb <= 512 ? ek : (double *)malloc(sizeof(double) * nb);
      double *ekq_p = nb <= 512 ? ekq : (double *)malloc(sizeof(double) * nb);
      const int r = oracle_pair(nb, nm, ne, g1, H_R, Re, w_e, e_q, omega_q + iq * nm, omega_min, k_list + 3 * ik, q,
                                g2 + (iq * nk + ik) * E, ek_p, ekq_p, NULL);
      if (r < rc) rc = r;
      if (iq == 0) memcpy(eps_k + ik * nb, ek_p, sizeof(double) * nb);
      if (eps_kq) memcpy(eps_kq + (iq * nk + ik) * nb, ekq_p, sizeof(double) * nb);
      if (nb > 512) { free(ek_p); free(ekq_p); }
    }
  }
  free(g1); free(e_q);
  return rc;
}

/* ---------------------------------------------------------------------------------------------
 * Second, independent code path: the single-loop algorithm, Eq. 7 evaluated directly for one
 * pair (Fig. 1a): six nested sums, no intermediate g(Re,q) buffer.
 *   g_{mn nu} = sum_{m'n' ka Re Rp} g(Re,Rp) conj(Ukq[m',m]) Uk[n',n] u[ka,nu] e^{i(q.Rp + k.Re)}
 * with u[ka,nu] = e[ka,nu]/sqrt(2 omega_nu).  Used only for the brute-force pin on tiny inputs.
 * ------------------------------------------------------------------------------------------- */
void oracle_eq7_direct(int nb, int nm, int ne, int np, const zc *g_RR, const int32_t *Re, const double *w_e,
                       const int32_t *Rp, const double *w_p, const zc *Ukq, const zc *Uk, const zc *e_q,
                       const double *omega_q, const double k[3], const double q[3], zc *g) {
  for (int nu = 0; nu < nm; nu++)
    for (int n = 0; n < nb; n++)
      for (int m = 0; m < nb; m++) {
        zc s = 0.0;
        for (int mp = 0; mp < nb; mp++)
          for (int np_ = 0; np_ < nb; np_++)
            for (int ka = 0; ka < nm; ka++)
              for (int ie = 0; ie < ne; ie++)
                for (int ip = 0; ip < np; ip++) {
                  const zc ph = expi(oracle_phase(q, Rp + 3 * ip) + oracle_phase(k, Re + 3 * ie));
                  const zc gw = g_RR[mp + nb * (np_ + nb * (ie + (int64_t)ne * (ka + (int64_t)nm * ip)))];
                  s += w_e[ie] * w_p[ip] * gw * conj(Ukq[mp + nb * m]) * Uk[np_ + nb * n] *
                       (e_q[ka + nm * nu] / sqrt(2.0 * omega_q[nu])) * ph;
                }
        g[m + nb * (n + nb * nu)] = s;
      }
}

/* ---------------------------------------------------------------------------------------------
 * Eq. 6, PAPER.md:L78-80 (Bloch -> Wannier), TEST-ONLY, in the Wannier gauge (U = u = 1):
 *   g(Re,Rp) = 1/(Ne Np) sum_{k'q'} G(k',q') exp(-i(q'.Rp + k'.Re))
 * G[m' + Nb*(n' + Nb*(ka + Nm*(ik + nkc*iq)))].  Builds the input of the round-trip pin.
 * ------------------------------------------------------------------------------------------- */
void oracle_eq6_wannier_from_bloch(int nb, int nm, int ne, int np, const zc *G, const double *kc, int nkc,
                                   const double *qc, int nqc, const int32_t *Re, const int32_t *Rp, zc *g_RR) {
  const int nbb = nb * nb;
  for (int ip = 0; ip < np; ip++)
    for (int ka = 0; ka < nm; ka++)
      for (int ie = 0; ie < ne; ie++)
        for (int el = 0; el < nbb; el++) {
          zc s = 0.0;
          for (int iq = 0; iq < nqc; iq++)
            for (int ik = 0; ik < nkc; ik++) {
              const double phi = oracle_phase(qc + 3 * iq, Rp + 3 * ip) + oracle_phase(kc + 3 * ik, Re + 3 * ie);
              s += G[el + nbb * (ka + nm * (ik + (int64_t)nkc * iq))] * expi(-phi);
            }
          g_RR[el + (int64_t)nbb * (ie + (int64_t)ne * (ka + (int64_t)nm * ip))] = s / ((double)ne * (double)np);
        }
}

/* ---------------------------------------------------------------------------------------------
 * Gauge part of Eq. 6: the factors U*_{mm'k'+q'} U_{nn'k'} u^-1_{nu,ka}(q') that take one
 * coarse-grid Bloch-representation block back to the Wannier gauge before the two inverse Fourier sums.
 * With [reading G4] paper-U = V^dagger (V = eigenvector columns) U*_{mm'} = V[m',m], U_{nn'} = conj(V[n',n]), and with
 * [reading G3] u = e/sqrt(2 omega) (e unitary) u^-1_{nu,ka} = sqrt(2 omega_nu) conj(e[ka,nu]):
 *   g~_{m'n' ka} = sum_{m n nu} Ukq[m',m] g_{mn nu} conj(Uk[n',n]) sqrt(2 omega_nu) conj(e[ka,nu])
 * g [m + Nb*(n + Nb*nu)] -> gt [m' + Nb*(n' + Nb*ka)].  The exact inverse of oracle_mode_rotate followed by
 * oracle_band_rotate (for omega > 0).
 * ------------------------------------------------------------------------------------------- */
void oracle_eq6_unrotate(int nb, int nm, const zc *g, const zc *Ukq, const zc *Uk, const zc *e, const double *omega,
                         zc *gt) {
  const int nbb = nb * nb;
  zc *T = (zc *)malloc(sizeof(zc) * nbb);
  zc *gw = (zc *)malloc(sizeof(zc) * nbb * nm);   /* Wannier band gauge, still mode basis */
  for (int nu = 0; nu < nm; nu++) {
    const zc *gn = g + (int64_t)nbb * nu;
    for (int n = 0; n < nb; n++)
      for (int mp = 0; mp < nb; mp++) {
        zc s = 0.0;
        for (int m = 0; m < nb; m++) s += Ukq[mp + nb * m] * gn[m + nb * n];
        T[mp + nb * n] = s;
      }
    for (int np_ = 0; np_ < nb; np_++)
      for (int mp = 0; mp < nb; mp++) {
        zc s = 0.0;
        for (int n = 0; n < nb; n++) s += T[mp + nb * n] * conj(Uk[np_ + nb * n]);
        gw[mp + nb * np_ + (int64_t)nbb * nu] = s;
      }
  }
  for (int ka = 0; ka < nm; ka++)
    for (int el = 0; el < nbb; el++) {
      zc s = 0.0;
      for (int nu = 0; nu < nm; nu++) s += gw[el + (int64_t)nbb * nu] * sqrt(2.0 * omega[nu]) * conj(e[ka + nm * nu]);
      gt[el + (int64_t)nbb * ka] = s;
    }
  free(T); free(gw);
}

/* ---------------------------------------------------------------------------------------------
 * Energy-window pre-screening: "skipping the calculation of the e-ph matrix elements involving
 * states outside a ... energy window".  A pair (k,q) is KEPT iff the initial state and the final state can both lie in
 * the window: some band of eps_k and some band of eps_{k+q} is in [emin, emax] (closed interval).
 * mask[ik + nk*iq] = 1 (kept) or 0 (skipped; its |g|^2 block is reported as zeros).
 * ------------------------------------------------------------------------------------------- */
void oracle_window_mask(int nb, int64_t nk, int64_t nq, const double *eps_k, const double *eps_kq, double emin,
                        double emax, unsigned char *mask) {
  for (int64_t iq = 0; iq < nq; iq++)
    for (int64_t ik = 0; ik < nk; ik++) {
      int in_k = 0, in_kq = 0;
      for (int b = 0; b < nb; b++) {
        const double e1 = eps_k[b + nb * ik], e2 = eps_kq[b + nb * (ik + nk * iq)];
        if (e1 >= emin && e1 <= emax) in_k = 1;
        if (e2 >= emin && e2 <= emax) in_kq = 1;
      }
      mask[ik + nk * iq] = (unsigned char)(in_k && in_kq);
    }
}

/* ---------------------------------------------------------------------------------------------
 * A consumer of |g|^2.  The paper names the consumers -- "ab initio Boltzmann transport",
 * "electron self-energy" -- but prints no formula for them; [reading, G18] the
 * imaginary part of the Fan-Migdal electron self-energy in its usual double-sum form with Gaussian-broadened energy
 * conservation is taken, per initial state (n,k):
 *   Im Sigma_nk += pi sum_q w_q sum_{m,nu} |g_{mn nu}(k,q)|^2 [ (n_qnu + f_mk+q)     delta_s(e_nk - e_mk+q + w_qnu)
 *                                                           + (n_qnu + 1 - f_mk+q) delta_s(e_nk - e_mk+q - w_qnu) ]
 *   delta_s(x) = exp(-(x/s)^2) / (s sqrt(pi)),  n = 1/(exp(w/kT) - 1),  f = 1/(exp((e - mu)/kT) + 1);
 * modes with w <= 0 are skipped.  out[n + Nb*ik] is ACCUMULATED (+=).  g2 [nq][nk][Nm][Nb(n)][Nb(m)].
 * ------------------------------------------------------------------------------------------- */
void oracle_selfenergy_accumulate(int nb, int nm, int64_t nk, int64_t nq, const double *g2, const double *eps_k,
                                  const double *eps_kq, const double *omega, const double *w_q, double mu, double kT,
                                  double sigma, double *out) {
  const double pi = 3.14159265358979323846;
  for (int64_t iq = 0; iq < nq; iq++)
    for (int64_t ik = 0; ik < nk; ik++)
      for (int n = 0; n < nb; n++) {
        const double e1 = eps_k[n + nb * ik];
        double s = 0.0;
        for (int nu = 0; nu < nm; nu++) {
          const double w = omega[nu + nm * iq];
          if (!(w > 0.0)) continue;
          const double bose = 1.0 / (exp(w / kT) - 1.0);
          for (int m = 0; m < nb; m++) {
            const double e2 = eps_kq[m + nb * (ik + nk * iq)];
            const double f = 1.0 / (exp((e2 - mu) / kT) + 1.0);
            const double xa = (e1 - e2 + w) / sigma, xe = (e1 - e2 - w) / sigma;
            const double da = exp(-xa * xa) / (sigma * sqrt(pi)), de = exp(-xe * xe) / (sigma * sqrt(pi));
            s += g2[m + nb * (n + nb * (nu + nm * (ik + nk * iq)))] * ((bose + f) * da + (bose + 1.0 - f) * de);
          }
        }
        out[n + nb * ik] += pi * (w_q ? w_q[iq] : 1.0) * s;
      }
}

/* ---------------------------------------------------------------------------------------------
 * Bookkeeping helpers pinned by the paper's printed numbers.
 * ------------------------------------------------------------------------------------------- */
/* Table III caption: size of g(Re,Rp) = 16 Nb^2 Nm Ne Np bytes. */
double oracle_g_bytes(double nb, double nm, double ne, double np) { return 16.0 * nb * nb * nm * ne * np; }

/* Eq. 8, PAPER.md:L102 (single loop) and Eq. 11, PAPER.md:L118-122 (nested loop): numbers of complex
 * multiplications AS PRINTED (band rotation counted as 2 Nb^2 Nm, [reading G2]). */
double oracle_nmul_single_loop(double nb, double nm, double ne, double np, double nk, double nq) {
  return (nb * nb * nm * ne * np + nb * nb * nm * ne + 2.0 * nb * nb * nm + nb * nb * nm * nm) * nk * nq;
}
double oracle_nmul_nested_loop(double nb, double nm, double ne, double np, double nk, double nq) {
  return nb * nb * nm * ne * np * nq + (nb * nb * nm * ne + 2.0 * nb * nb * nm + nb * nb * nm * nm) * nk * nq;
}
