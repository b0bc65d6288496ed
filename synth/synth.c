/*
 * synth.c -- seeded, counter-based synthetic input generator (host only).
 *
 * This module holds NONE of the method's arithmetic.  It only produces the
 * random operators H(R), D(R), g(Re,Rp) and the random q-points that stand in
 * for the paper's silicon / MoS2 / stanene data sets (PAPER.md:L241, L251, L265,
 * L321 -- not available offline).  Both the CPU oracle and the CUDA library are
 * fed from here, so that they see bit-identical inputs.
 *
 * Generator: value(seed, stream, index) is a pure function (SplitMix64 finaliser
 * chain -> two uniforms -> Box-Muller), so any slab of the 49 GB config-4 tensor
 * can be regenerated without ever materialising the whole array.
 *
 * Layout of g follows PAPER.md:L501-511 (Fig. 13: column-major A(m,n), the
 * column index n is Rp) and BASELINE.json ([Nb,Nb,Ne,Nm,Np], first index
 * fastest): flat = m' + Nb*(n' + Nb*(ie + Ne*(ka + Nm*ip))).
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

static inline uint64_t mix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}

static inline uint64_t ctr_hash(uint64_t seed, uint64_t stream, uint64_t idx, uint64_t lane) {
  uint64_t h = mix64(seed ^ 0x5851F42D4C957F2DULL);
  h = mix64(h ^ (stream * 0xD1B54A32D192ED03ULL));
  h = mix64(h ^ idx);
  return mix64(h + lane);
}

static inline double u01_open(uint64_t h) { /* (0,1) */
  return ((double)(h >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

/* one complex standard normal: re, im i.i.d. N(0,1) */
static inline void gauss_pair(uint64_t seed, uint64_t stream, uint64_t idx, double *re, double *im) {
  double u1 = u01_open(ctr_hash(seed, stream, idx, 0));
  double u2 = u01_open(ctr_hash(seed, stream, idx, 1));
  double r = sqrt(-2.0 * log(u1));
  double a = 6.283185307179586476925286766559 * u2;
  *re = r * cos(a);
  *im = r * sin(a);
}

/* out[2*i], out[2*i+1] = complex normal number (start+i) of the stream, times scale */
void synth_gauss_complex(uint64_t seed, uint64_t stream, uint64_t start, uint64_t count, double scale,
                         double *out) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < (int64_t)count; i++) {
    double re, im;
    gauss_pair(seed, stream, start + (uint64_t)i, &re, &im);
    out[2 * i] = scale * re;
    out[2 * i + 1] = scale * im;
  }
}

/* out[i] = uniform in (0,1), number (start+i) of the stream */
void synth_uniform(uint64_t seed, uint64_t stream, uint64_t start, uint64_t count, double *out) {
  for (uint64_t i = 0; i < count; i++) out[i] = u01_open(ctr_hash(seed, stream, start + i, 0));
}

/*
 * Slabs ip_start .. ip_start+ip_count-1 of g(Re,Rp):
 *   g[m',n',ie,ka,ip] = amp * exp(-|Re_ie|/lam_e - |Rp_ip|/lam_p) * Z(flat index)
 * re_norm[ne], rp_norm[np] are the Euclidean norms of the integer lattice vectors.
 * out holds ip_count * (nb*nb*ne*nm) complex numbers (interleaved re, im).
 */
void synth_fill_g(uint64_t seed, uint64_t stream, int32_t nb, int32_t nm, int32_t ne, int32_t np,
                  int32_t ip_start, int32_t ip_count, double amp, const double *re_norm,
                  const double *rp_norm, double lam_e, double lam_p, double *out) {
  (void)np;
  const int64_t nbb = (int64_t)nb * nb;
  const int64_t slab = nbb * ne * nm;
#pragma omp parallel for collapse(2) schedule(static)
  for (int32_t dp = 0; dp < ip_count; dp++) {
    for (int64_t row = 0; row < (int64_t)nm * ne; row++) {
      const int32_t ip = ip_start + dp;
      const int32_t ie = (int32_t)(row % ne);
      const double a = amp * exp(-re_norm[ie] / lam_e - rp_norm[ip] / lam_p);
      const uint64_t flat0 = (uint64_t)ip * (uint64_t)slab + (uint64_t)row * (uint64_t)nbb;
      double *o = out + 2 * ((int64_t)dp * slab + row * nbb);
      for (int64_t e = 0; e < nbb; e++) {
        double re, im;
        gauss_pair(seed, stream, flat0 + (uint64_t)e, &re, &im);
        o[2 * e] = a * re;
        o[2 * e + 1] = a * im;
      }
    }
  }
}
