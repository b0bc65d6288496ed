/*
 * epw_interp.h -- C ABI of the B200-native Wannier-to-Bloch interpolation of
 * electron-phonon matrix elements (arxiv/paper_2603_10295, EPW 6.1).
 *
 * The path ("The path"):
 *   S0  phase tables          exp(2 pi i q.Rp), exp(2 pi i k.Re)            PAPER.md:L110, L114, L303 ("x" of Fig. 13)
 *   S1  Rp -> q               g(Re,q) = sum_Rp g(Re,Rp) e^{i q.Rp}          PAPER.md:L110 (Eq. 9), L501-511 (Fig. 13)
 *   S3  operators             H(R)->H(k), H(k+q); D(Rp)->D(q); Hermitian eigensolves -> U, eps, e_q, omega_q
 *                                                                           BASELINE.json north_star stage (3)
 *   S4a mode rotation         g^ = g e_q / sqrt(2 omega_q)   (hoisted onto g(Re,q): it is linear and depends on q only)
 *                                                                           PAPER.md:L114 (u_{ka,nu}(q)), L102 ("Rotation by")
 *   S2  Re -> k               g~(k,q) = sum_Re g^(Re,q) e^{i k.Re}, batched over k as one FP64 tensor (DMMA) contraction
 *                                                                           PAPER.md:L112-114 (Eq. 10), L118 ("FT w.r.t. Re")
 *   S4b band rotation, |g|^2  g_{mn nu} = sum_{m'n'} conj(U_{k+q}[m',m]) g~_{m'n' nu} U_k[n',n];  out = |g_{mn nu}|^2
 *                                                                           PAPER.md:L114 (U_{mm'k+q} U*_{nn'k}), north_star stage (4)
 *
 * Conventions common to every entry point
 *   - Complex numbers are interleaved (re, im) FP64 pairs ("c128"); all arithmetic is FP64.
 *   - "Fortran (a,b,c)" means the FIRST index is fastest in memory.
 *   - k, q are crystal (fractional) coordinates; R vectors are integer triples; phase = 2 pi frac(x.R).
 *   - Matrices are column-major, eigenvectors are the COLUMNS of U / e, eigenvalues ascending.
 *   - Return value: 0 (EPW_OK) or a negative epw_status; nothing is thrown across the ABI.
 *     epw_interp_last_error(h) returns a human-readable message for the last failure on that handle.
 *   - Ownership: the caller owns every buffer passed in; the library copies the operators in
 *     epw_interp_set_wannier_operators and owns that copy and its workspace.
 *   - "device" pointers are CUDA device pointers valid on the handle's device; "host" pointers are CPU memory.
 *   - Calls on one handle must not overlap (a handle is not thread-safe); distinct handles are independent.
 *   - One stream per handle: every call writes the handle's workspace, so the asynchronous calls on a handle are meant to be
 *     issued on ONE stream, which orders them.  A caller that moves a handle to another stream first orders the new stream
 *     behind the old one (event, or epw_interp_sync).  The one thing the library orders by itself is its k-side cache: a
 *     grid call that reuses H(k), U_k, eps_k of an earlier call on a different stream waits on an event recorded behind them.
 *   - There is no CPU fallback: every call fails with EPW_ECUDA if no sm_100 device is usable.
 */
#ifndef EPW_INTERP_H_
#define EPW_INTERP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct epw_interp *epw_interp_t; /* opaque; owned by the library */

typedef enum {
  EPW_OK = 0,
  EPW_EINVAL = -1,        /* bad argument (null pointer, non-positive size, operators not set, ...) */
  EPW_ENOMEM = -2,        /* device or host allocation failed */
  EPW_ECUDA = -3,         /* CUDA runtime error, or no usable sm_100 device */
  EPW_ENOTCONVERGED = -4, /* a Jacobi eigensolve hit the sweep limit (reported by epw_interp_sync) */
  EPW_EUNSUPPORTED = -5   /* shape outside what this build implements (message says which) */
} epw_status;

typedef struct {
  int32_t nbnd;           /* Nb: number of Wannier functions / bands  */
  int32_t nmodes;         /* Nm = 3 Na: number of phonon modes  */
  int32_t ne;             /* Ne: number of electron Wigner-Seitz vectors Re */
  int32_t np;             /* Np: number of phonon Wigner-Seitz vectors Rp */
  int32_t device;         /* CUDA device ordinal */
  int32_t q_batch;        /* q-points contracted per pass over g(Re,Rp) in S1 (1..8); 0 = library default (8); lowered by the
                             library when the [Np][q_batch] phase table would not fit shared memory (Np > 1,760 at 8);
                             Np > 14,080 is EPW_EUNSUPPORTED */
  int32_t path;           /* EPW_PATH_AUTO (0): chosen from Nb, Nm; EPW_PATH_SMALL / EPW_PATH_LARGE force one (tests) */
  int32_t flags;          /* 0: on a uniform grid the library picks the faster form of the last axis pass of S2 + S4b: ONE kernel
                             (g~ never reaches HBM) for Nb <= 8, two kernels (the pass writes g~, rotate_g2 reads it) above;
                             EPW_FLAG_GRID_FUSED / EPW_FLAG_GRID_UNFUSED force the one-kernel (Nb <= 16) / two-kernel form */
  size_t workspace_bytes; /* cap on the library's scratch HBM; 0 = library chooses from free memory */
  double degen_tol;       /* informational (gap below which callers should sum |g|^2 over a subspace); unused inside */
  double omega_min;       /* modes with omega_q,nu <= omega_min give |g|^2 = 0 (acoustic modes at Gamma); default 0;
                             must be >= 0 (create fails with EPW_EINVAL otherwise: soft modes are reported with negative omega) */
} epw_interp_config;

/* Kernel families of the path.  SMALL: a whole (k,q) pair lives in shared memory (Nb <= 16, configs[0..3]).
 * LARGE: S4a, S2 and both halves of S4b are FP64 tensor-path contractions that read their operand in place
 * (any Nb; configs[4], Nb = 192, Nm = 288).  Same results; AUTO picks by size. */
enum { EPW_PATH_AUTO = 0, EPW_PATH_SMALL = 1, EPW_PATH_LARGE = 2 };
enum { EPW_FLAG_GRID_UNFUSED = 1, EPW_FLAG_GRID_FUSED = 2 };

/* Create / destroy a handle.  *out is set to NULL on failure. */
int epw_interp_create(epw_interp_t *out, const epw_interp_config *cfg);
void epw_interp_destroy(epw_interp_t h);

/*
 * Upload the Wannier-representation operators (they stay resident in HBM for the whole interpolation,
 * PAPER.md:L184).  on_device = 0: host pointers, 1: device pointers (copied device-to-device).
 *   H_R   c128 Fortran (i, j, ie)            [Ne][Nb][Nb]      H(Re)_{ij}, H(-R) = H(R)^dagger expected
 *   D_R   c128 Fortran (a, b, ip)            [Np][Nm][Nm]      dynamical matrix, masses absorbed (eV^2)
 *   g_RR  c128 Fortran (m', n', ie, ka, ip)  [Np][Nm][Ne][Nb][Nb]   size 16 Nb^2 Nm Ne Np bytes;
 *         this is Fig. 13's column-major A(m,n) with the Rp index as the column.
 *         May be NULL: then every Rp slab must be supplied with epw_interp_set_g_slabs before interpolating.
 *   Re    int32 [Ne][3], w_e f64 [Ne]   electron lattice vectors and Wigner-Seitz weights (1/ndegen)
 *   Rp    int32 [Np][3], w_p f64 [Np]   phonon lattice vectors and weights
 */
int epw_interp_set_wannier_operators(epw_interp_t h, const void *H_R, const void *D_R, const void *g_RR,
                                     const int32_t *Re, const double *w_e, const int32_t *Rp, const double *w_p,
                                     int on_device);

/* Upload Rp slabs ip_start .. ip_start+ip_count-1 of g_RR (each Nb^2 Ne Nm c128, same layout as above), so that
 * a tensor larger than host memory (Table III) can be streamed in. */
int epw_interp_set_g_slabs(epw_interp_t h, int32_t ip_start, int32_t ip_count, const void *g_slabs, int on_device);

/*
 * The hot path: every (k,q) pair of the two lists.  All pointers are DEVICE pointers.  Asynchronous on `cuda_stream`
 * (a cudaStream_t passed as void*; NULL = legacy default stream): caller buffers are touched only between enqueue
 * and stream completion.
 *   k_list  f64 [nk][3], q_list f64 [nq][3]   crystal coordinates (any values; no grid assumed)
 *   kq_map  NULL, or int32 [nq][nk]: index in k_list of k+q folded onto the list (grid case): then U_{k+q},
 *           eps_{k+q} are looked up instead of eigensolving H(k+q) per pair
 *   eps_k   out f64 [nk][Nb]            eigenvalues of H(k), ascending
 *   eps_kq  out f64 [nq][nk][Nb] or NULL
 *   omega_q out f64 [nq][Nm]            sqrt of the eigenvalues of D(q) (negative = imaginary frequency)
 *   g2      out f64 [nq][nk][Nm][Nb][Nb] = Fortran (m, n, nu, k, q): |g_{mn nu}(k,q)|^2, m (the k+q band) fastest
 * The caller batches q so that g2 (8 Nb^2 Nm nk nq bytes) fits.
 */
int epw_interp_interpolate(epw_interp_t h, const double *k_list, int64_t nk, const double *q_list, int64_t nq,
                           const int32_t *kq_map, double *eps_k, double *eps_kq, double *omega_q, double *g2,
                           void *cuda_stream);

/*
 * Same computation with HOST buffers (pinned or pageable): copies k_list, q_list, kq_map to the device, runs the
 * path, copies eps_k, eps_kq (if non-NULL), omega_q and g2 back, and returns after everything has completed.
 * The g2 / eps_kq slices of each finished q are copied on an internal second stream while the next q is computed
 * (pinned host buffers make that copy asynchronous; pageable ones still work).
 */
int epw_interp_interpolate_host(epw_interp_t h, const double *k_list, int64_t nk, const double *q_list, int64_t nq,
                                const int32_t *kq_map, double *eps_k, double *eps_kq, double *omega_q, double *g2,
                                void *cuda_stream);

/*
 * The same hot path for k-points on a UNIFORM GRID, given by its three sizes instead of a list:
 *     k[(i1*N2 + i2)*N3 + i3] = ((i1 + s1)/N1, (i2 + s2)/N2, (i3 + s3)/N3),   i3 fastest,   nk = N1 N2 N3
 *   k_grid  int32 [3] HOST: N1, N2, N3 (all > 0);   k_shift f64 [3] HOST or NULL (= 0: Gamma-centred grid)
 * Results, layouts and every other argument are those of epw_interp_interpolate called with that k-list (kq_map, if
 * given, indexes the grid in the order above).  On a grid the phase of the Re -> k Fourier sum (PAPER.md:L112-118,
 * Eq. 10) factorises over the crystal axes, so S2 and the H(k), H(k+q) part of S3a are taken one axis at a time
 * (csrc/re_to_k_grid.cu): (L1 L2 N3 L3 + L1 N2 N3 L2 + N1 N2 N3 L1) instead of Nk Ne multiplications per column, with
 * L_d the extents of the bounding box of the Re list -- the same sums re-associated, equal to the list form up to
 * rounding order.  The large-Nb kernel family (one-dimensional grids) expands the grid to a list internally.
 * The k side of the call (H(k), U_k, eps_k) is kept in the handle and reused by the next grid call with the same sizes and
 * shift, until the operators change or a k-list call comes in between: a caller looping over batches of q on one fine
 * k-grid pays for the Nk eigensolves of H(k) once.  A call that returns an error, and an epw_interp_sync that reports
 * EPW_ENOTCONVERGED, drop the kept k side: the next grid call computes it again.
 */
int epw_interp_interpolate_grid(epw_interp_t h, const int32_t *k_grid, const double *k_shift, const double *q_list,
                                int64_t nq, const int32_t *kq_map, double *eps_k, double *eps_kq, double *omega_q,
                                double *g2, void *cuda_stream);
/* Host-buffer form of epw_interp_interpolate_grid (cf. epw_interp_interpolate_host). */
int epw_interp_interpolate_grid_host(epw_interp_t h, const int32_t *k_grid, const double *k_shift, const double *q_list,
                                     int64_t nq, const int32_t *kq_map, double *eps_k, double *eps_kq, double *omega_q,
                                     double *g2, void *cuda_stream);

/*
 * Energy-window pre-screening of the pairs ("skipping the calculation of the e-ph matrix elements
 * involving states outside a 0.3 eV energy window").  While enabled, every following
 * interpolate call keeps a pair (k,q) iff some band of eps_k AND some band of eps_{k+q} lies in the closed interval
 * [emin, emax] (decided on the library's own FP64 eigenvalues, right after the eigensolves); the |g|^2 block of a
 * skipped pair is written as zeros and its S4b work is not done (the one-kernel grid form works on quads of four
 * consecutive i1: a quad is skipped when all four of its pairs are).
 * eps_k, eps_kq and omega_q are still complete.  mask_out: NULL, or a device buffer uint8 [nq][nk] that receives
 * 1 (kept) / 0 (skipped) for every pair of each call.  (To drop k-points altogether, pass the screened k-list.)
 */
int epw_interp_set_energy_window(epw_interp_t h, int enabled, double emin, double emax, uint8_t *mask_out);

/*
 * A consumer of |g|^2 on the device: while enabled, every following interpolate call adds, for
 * each of its pairs, the contribution of that pair to the imaginary part of the Fan-Migdal electron self-energy
 *   Im Sigma_nk += pi w_q sum_{m,nu} |g_{mn nu}(k,q)|^2 [ (n_qnu + f_mk+q) delta_s(e_nk - e_mk+q + w_qnu)
 *                                                      + (n_qnu + 1 - f_mk+q) delta_s(e_nk - e_mk+q - w_qnu) ]
 * (delta_s(x) = exp(-(x/s)^2)/(s sqrt(pi)), Bose n at kT, Fermi f at (mu, kT), modes with omega <= 0 skipped) -- the
 * paper names this consumer without printing it: DESIGN.md reading G18.
 *   w_q      NULL (weight 1) or device f64 [nq of the call]: weight of every q-point of the call
 *   im_sigma device f64 [nk][Nb], ACCUMULATED (+=) by every call: the caller zeroes it and may sum over many calls
 * With the consumer enabled the g2 argument of the interpolate calls (device or host form) may be NULL.  On a uniform grid
 * with Nb <= 8 (the one-kernel form of the last axis pass + S4b) the reduction happens in the epilogue of that kernel,
 * straight from the accumulator registers: no |g|^2 is written anywhere and nothing of size nk nq exists.  In the other
 * kernel routes the library keeps |g|^2 of one q at a time in its own scratch (8 Nb^2 Nm nk bytes) and reduces it with a
 * second kernel.  The sum over (m, nu) runs in a fixed order (deterministic) unless the modes of a pair are split over
 * several tiles of the one-kernel form (large Nb^2 Nm L1: atomic adds, the order of the partial sums then varies).
 */
int epw_interp_set_selfenergy_consumer(epw_interp_t h, int enabled, double mu, double kT, double sigma, const double *w_q,
                                       double *im_sigma);

/*
 * g(Re,Rp) split over several GPUs by Rp (the paper's pool level for operators larger than one GPU's memory,
 * PAPER.md:L186-188, Table III; SURVEY.md 8(e) variant B / 8(f) NEXT-1).  Eq. 9 is a sum over Rp, so each
 * rank contracts its own slabs and the partial g(Re,q) are summed across ranks -- the paper does D2H + mp_sum on the
 * host (L514, L522); here the partial sums stay on the device and the caller all-reduces them on the same stream
 * (NCCL through torch.distributed: the one real exchange step of the path).  After the sum every rank holds the full
 * g(Re,q) and runs the rest of the path on ITS share of the k-points (outputs are disjoint).
 *
 *   epw_interp_set_rp_shard     before uploading g: this handle keeps only slabs [ip_start, ip_start+ip_count) of g_RR
 *                               (H_R, D_R, Re, Rp and the weights are still the complete lists).
 *   epw_interp_rp_to_q_partial  S0 + S1 over the handle's slabs: g1_partial c128 [nq][Nb^2 Nm Ne] (device, caller-owned),
 *                               asynchronous on cuda_stream.  q_list f64 [nq][3] device.
 *   epw_interp_set_gq           the NEXT epw_interp_interpolate / _grid call takes g(Re,q) from g1_reduced (device,
 *                               c128 [nq][Nb^2 Nm Ne], the same nq and q order as that call) instead of running S1;
 *                               NULL restores the normal path.  The buffer must stay valid until that call completes.
 */
int epw_interp_set_rp_shard(epw_interp_t h, int32_t ip_start, int32_t ip_count);
int epw_interp_rp_to_q_partial(epw_interp_t h, const double *q_list, int64_t nq, void *g1_partial, void *cuda_stream);
/*
 * The same exchange step FUSED into the S1 pass (compute + collective in one kernel): S0 + S1 over the handle's slabs,
 * with the partial g(Re,q) of q-point iq ADDED (red.global.add.f64, system scope) to dst[iq] instead of being stored.
 *   dst   HOST array of nq DEVICE pointers, dst[iq] -> c128 [Nb^2 Nm Ne]: the buffer of the rank that owns q-point iq.  It
 *         may be memory of ANOTHER GPU mapped into this process (NVLink peer access, CUDA IPC or symmetric memory): the
 *         sums then cross NVLink row tile by row tile while g(Re,Rp) is still being streamed, and no collective follows.
 * Every rank calls it with the same q_list and its own view of the same buffers; the owners zero their buffers before and
 * all ranks synchronise after (barrier) before epw_interp_set_gq hands dst[own iq] to the rest of the path.  The order of
 * the additions varies from run to run: the sum over ranks is reproducible to rounding only (W terms per element).
 * (The paper: D2H of the partial y, mp_sum on the host.)  Asynchronous on cuda_stream: the table is
 * uploaded on the stream and the host is not made to wait; the dst array may be reused as soon as the call returns.
 * Adding into another GPU's memory needs native atomics over the link between the two devices
 * (cudaDevP2PAttrNativeAtomicSupported: NVLink yes, PCIe peer access no); the call checks every destination that the
 * process knows to be on another device and returns EPW_EUNSUPPORTED if that attribute is 0.
 */
int epw_interp_rp_to_q_scatter_add(epw_interp_t h, const double *q_list, int64_t nq, void *const *dst, void *cuda_stream);
int epw_interp_set_gq(epw_interp_t h, const void *g1_reduced);

/* Wait for the handle's last enqueued work and report deferred device-side status (EPW_ENOTCONVERGED, EPW_ECUDA).
 * The convergence flag is sticky: it is set by any eigensolve of any call enqueued since the last epw_interp_sync and is
 * read and cleared only here, so one sync after several asynchronous calls reports a failure in any of them. */
int epw_interp_sync(epw_interp_t h);

/*
 * Per-stage device times (ms, CUDA events on the caller's stream) accumulated over every interpolate call since
 * stage timing was last enabled:
 *   ms[0] S0 phase tables   ms[1] S1 Rp->q   ms[2] D(q) + phonon eigensolve   ms[3] H(k) + eigensolve
 *   ms[4] S2 Re->k contraction   ms[5] H(k+q) eigensolve   ms[6] S4b rotation + |g|^2   ms[7] total
 *   ms[8] S4a mode rotation (hoisted onto g(Re,q)) incl. building the packed operand of S2
 * Synchronises the stream.  Returns the number of entries written (<= n) or a negative status.
 */
#define EPW_NUM_STAGES 9
int epw_interp_get_stage_times(epw_interp_t h, double *ms, int n);

/* Kernel launches per stage over the same accumulation period as epw_interp_get_stage_times (same indices;
 * counts[7] = all launches).  Returns the number of entries written or a negative status. */
int epw_interp_get_stage_launches(epw_interp_t h, int64_t *counts, int n);

/* Stage timing records two CUDA events per stage invocation; it is off by default.  on != 0 enables it for the
 * following interpolate calls and clears the accumulated times; on == 0 disables it. */
int epw_interp_enable_stage_timing(epw_interp_t h, int on);

/* Plane rotations (matrix-rotations) the register-resident Jacobi eigensolvers executed since stage timing was last
 * enabled: counts[0] H(k), counts[1] H(k+q), counts[2] D(q).  The sweep count of Jacobi is data dependent, so this is
 * what turns the eigensolve time into an FP64 rate (flops per rotation of each kernel).  Zero for the
 * shared-memory / cluster kernels, which do not count.  Synchronises the stream.  Returns entries written. */
int epw_interp_get_eigh_rotations(epw_interp_t h, uint64_t *counts, int n);

/* Number of kernels the library launched during the last interpolate call (for bench.py's gpu_launches). */
int64_t epw_interp_last_launch_count(epw_interp_t h);

/* How the last interpolate call was executed: plan[0] = EPW_PATH_SMALL or EPW_PATH_LARGE, plan[1] = q-points per pass
 * over g(Re,Rp) in S1, plan[2] = k-points per chunk of S2 / S3b / S4b, plan[3] = 0 for the dense k-list contraction, 1 if S2 ran in its
 * factorised uniform-grid form with g~ written to HBM, 2 if its last axis pass was fused with S4b (g~ never leaves
 * the SM; times and launches of that kernel are booked under stage 6).  Returns the number of entries written. */
int epw_interp_last_plan(epw_interp_t h, int64_t *plan, int n);

/*
 * Intermediate results of the LAST q of the last interpolate call, for parity tests (device -> host copy,
 * synchronises).  `bytes` must be at least the size stated; returns bytes written or a negative status.
 *   EPW_DBG_G_REQ   g(Re,q)  c128 Fortran (m', n', ie, ka)            16 Nb^2 Ne Nm
 *   EPW_DBG_G_TILDE g~(k,q) after S4a+S2, c128 [nk][Nm][Nb][Nb]       16 Nb^2 Nm nk  (mode basis, amplitude applied)
 *   EPW_DBG_H_K     H(k)     c128 [nk][Nb][Nb] column-major           16 Nb^2 nk
 *   EPW_DBG_U_K     U_k      c128 [nk][Nb][Nb] columns = eigenvectors 16 Nb^2 nk
 *   EPW_DBG_U_KQ    U_{k+q}  c128 [nk][Nb][Nb] (per-pair solves only) 16 Nb^2 nk
 *   EPW_DBG_E_Q     e_q      c128 [Nm][Nm] columns = mode eigenvectors 16 Nm^2
 */
enum { EPW_DBG_G_REQ = 1, EPW_DBG_G_TILDE = 2, EPW_DBG_H_K = 3, EPW_DBG_U_K = 4, EPW_DBG_U_KQ = 5, EPW_DBG_E_Q = 6 };
int64_t epw_interp_debug_get(epw_interp_t h, int what, void *dst_host, size_t bytes);

const char *epw_interp_last_error(epw_interp_t h); /* h may be NULL: last error of a failed create */

/* -------------------------------------------------------------------------------------------------
 * Stage-level entry points (same kernels the path uses; device pointers; asynchronous on `cuda_stream`).
 * They exist so that each kernel can be parity-tested against the oracle on its own.
 * ----------------------------------------------------------------------------------------------- */

/* S0: P[ix][ir] = w[ir] * exp(2 pi i frac(x_ix . R_ir)), c128 [nx][nr] row-major. */
int epw_phase_table(const double *x_list, int64_t nx, const int32_t *R, const double *w, int32_t nr, void *P_out,
                    void *cuda_stream);

/* S1 (Eq. 9) for a batch of q: g1[iq] = sum_ip g_RR[ip] * Pq[iq][ip];  rows = Nb^2 Ne Nm.
 * g_RR c128 [np][rows], Pq c128 [nq][np] (weights included), g1 c128 [nq][rows].  nq <= 8 per call. */
int epw_rp_to_q(const void *g_RR, int64_t rows, int32_t np, const void *Pq, int32_t nq, void *g1_out,
                void *cuda_stream);

/* S3a: Op(x)[ix] = sum_ir P[ix][ir] Op_R[ir], n x n matrices (column-major), P from epw_phase_table. */
int epw_interp_operator(const void *Op_R, int32_t n, int32_t nr, const void *P, int64_t nx, void *out,
                        void *cuda_stream);

/* S3b: batched Hermitian eigensolve (parallel-order Jacobi).  A c128 [batch] matrices, column-major, matrix b at
 * A + b*stride_a (stride in c128 elements); only its Hermitian part (A + A^dagger)/2 is used.
 * evals f64 [batch][n] ascending; V c128 [batch][n][n], columns = eigenvectors.
 * sqrt_mode != 0 writes omega = sign(lambda) sqrt(|lambda|) instead of lambda.
 * status: int32 device word, set to nonzero if any solve hits the sweep limit (may be NULL). */
int epw_eigh_batched(const void *A, int64_t stride_a, int32_t n, int64_t batch, double *evals, void *V,
                     int sqrt_mode, int32_t *status, void *cuda_stream);
/* The same solve with an explicit kernel choice (parity tests exercise every kernel at every size it supports):
 *   EPW_EIGH_AUTO    what epw_eigh_batched and the path use: for batch >= 2048 THREAD (2 <= n <= 8) or COLS
 *                    (9 <= n <= 16), else WARP
 *   EPW_EIGH_WARP    n <= 32: one warp per matrix in shared memory; n > 32: thread-block cluster / CTA per matrix
 *   EPW_EIGH_THREAD  2 <= n <= 8 only (EPW_EINVAL otherwise): one thread per matrix, matrix and eigenvectors in
 *                    registers, rotation schedule unrolled at compile time
 *   EPW_EIGH_COLS    9 <= n <= 16 only (EPW_EINVAL otherwise): one-sided Jacobi, the columns of 32 matrices spread
 *                    over the warps of a CTA (lane = matrix), odd-even ordering */
enum { EPW_EIGH_AUTO = 0, EPW_EIGH_WARP = 1, EPW_EIGH_THREAD = 2, EPW_EIGH_COLS = 3 };
int epw_eigh_batched_algo(const void *A, int64_t stride_a, int32_t n, int64_t batch, double *evals, void *V,
                          int sqrt_mode, int32_t *status, int algo, void *cuda_stream);

/* Dense complex FP64 contraction on the FP64 tensor path:  C[m][n] = sum_r A[m][r] B[r][n],
 * A c128 [M][K] row-major, B c128 [K][N] row-major, C c128 [M][ldc] row-major (ldc >= N).
 * (Packs both operands into the DMMA fragment layout, then runs the same TMA + DMMA kernel as S2.) */
int epw_zgemm(const void *A, const void *B, void *C, int64_t M, int32_t N, int32_t K, int64_t ldc, void *cuda_stream);

/*
 * epw_zgemm for callers that must not allocate device memory: the same contraction (the K = Ne sum of Eq. 10,
 * PAPER.md:L112-118, as one FP64 tensor-path product), the same three kernels, the same result bit for bit -- but this
 * call never reaches cudaMalloc, cudaFree or any other allocating routine, and it does not synchronise.
 *
 * Meant for: applications that gave all of HBM to their own pool allocator (a library-side cudaMalloc would fail there,
 * or fragment the pool), time-critical / in-situ loops where cudaMalloc and cudaFree are banned because each of them
 * stalls the whole device, and hosts that do not let a loaded library grow the process's device footprint.  epw_zgemm
 * allocates and frees its two packed operands on every call; here they live in a fixed array of
 * EPW_ZGEMM_NOALLOC_SCRATCH_BYTES (16 MiB) that is part of the library image: EVERY GPU on which this function has been
 * called keeps those 16 MiB until the process exits, whether or not the function is called again.
 *
 *   A, B, C, M, N, K, ldc, cuda_stream   exactly as epw_zgemm: device pointers owned by the caller, A c128 [M][K],
 *                                        B c128 [K][N], C c128 [M][ldc] row-major; asynchronous on cuda_stream
 *   errbuf, errbuf_len                   NULL / 0, or a HOST buffer that receives a one-line message when the call fails
 *
 * Limit: ceil(M/128) ceil(K/8) + ceil(N/64) ceil(K/8) <= 1,024 (16 KB per term; e.g. M = 4,096, N = 384, K = 200).
 * Anything larger returns EPW_EUNSUPPORTED, launches nothing and leaves C untouched: split the product over row blocks
 * of A, or call epw_zgemm.
 *
 * First call on each device: it looks up the device address of the array (and makes the CUDA runtime load the library's
 * code on that device, which is when the 16 MiB appear).  Make that first call during start-up, in particular before
 * any stream capture begins; later calls on the device only launch kernels.  The device current at the call must be the
 * one the pointers and the stream belong to.
 *
 * All calls on a device share the one array.  Nothing in it has to be cleared between calls (the packing kernels
 * rewrite every value the product reads, padding included), and calls on ONE stream are ordered by the stream.  Calls
 * whose kernels can overlap on the GPU -- issued by one process on different streams of the same device (from one host
 * thread or several) with no event or synchronise between them -- overwrite each other's packed operands, and the
 * results are then garbage.  Serialise such calls yourself.  (Each process has its own copy of the array.)
 */
#define EPW_ZGEMM_NOALLOC_SCRATCH_BYTES (16u * 1024u * 1024u)
int epw_zgemm_noalloc(const void *A, const void *B, void *C, int64_t M, int32_t N, int32_t K, int64_t ldc,
                      void *cuda_stream, char *errbuf, size_t errbuf_len);

/* The contraction kernel of the large-Nb path (zgemm_strided.cu): `batch` problems C_b = A_b B_b on the FP64 tensor
 * path with the big operand A read in place:
 *   A_b[row][r] at A + b*a_batch + (row / a_rb)*a_bs + (row % a_rb) + r*a_ks      (c128 elements; rows contiguous)
 *   B_b[r][col] at B + bb*b_batch + r*b_sr + col*b_sn, conjugated if b_conj, bb = b_gather ? b_gather[b] : b,
 *               nb_mats matrices are packed (b_gather values must be < nb_mats; nb_mats = batch when b_gather is NULL)
 *   C_b[row][col] at C + b*c_batch + (row / c_rb)*c_bs + (row % c_rb)*c_rs + col*c_cs   as c128, or, if abs2 != 0,
 *               |C_b[row][col]|^2 as f64 (strides then count f64 elements).
 * All device pointers.  Synchronises the stream before returning (temporary packed B). */
int epw_zgemm_strided(const void *A, int64_t a_rb, int64_t a_bs, int64_t a_ks, int64_t a_batch, const void *B,
                      int64_t b_sr, int64_t b_sn, int64_t b_batch, int b_conj, const int32_t *b_gather, int64_t nb_mats,
                      void *C, int64_t c_rb, int64_t c_bs, int64_t c_rs, int64_t c_cs, int64_t c_batch, int abs2,
                      int64_t M, int32_t N, int32_t K, int64_t batch, void *cuda_stream);

/* One axis of the factorised Re -> k sum on a uniform grid (Eq. 10; reading G17) as the FP64
 * tensor-path (DMMA) product of grid_fused.cuh, for nbatch independent blocks:
 *     out[b][j][c][col] = sum_{n < L} P[n][j] T[b][n][c][col],    j < cnt, c < slab, col < ncols
 *   T    c128, block b at T + b*in_bstride, layout [L][slab][ncols];  ncols must be a multiple of nb*nb (the kernel works
 *        on column groups of nb^2, 1 <= nb <= 16), L <= 18
 *   P    c128 [L][cnt]: the phases w e^{2 pi i (j+s) n / N} of this axis
 *   out  c128, block b at out + b*out_bstride, row (j*slab + c) at stride out_stride (>= ncols)
 * All device pointers; asynchronous on cuda_stream.  EPW_EUNSUPPORTED when the shape does not fit the kernel. */
int epw_axis_pass_dmma(const void *T, int64_t slab, int32_t ncols, int32_t L, const void *P, int32_t cnt, int32_t nb,
                       void *out, int64_t out_stride, int32_t nbatch, int64_t in_bstride, int64_t out_bstride,
                       void *cuda_stream);

/* S4b: g2[ik][nu][n][m] = | sum_{m'n'} conj(Ukq[ik][m',m]) gt[ik][nu][n'][m'] Uk[ik][n',n] |^2.
 * gt c128, pair ik at gt + ik*stride_gt (c128 elements); Uk, Ukq c128 [..][Nb][Nb] column-major;
 * kq_idx NULL (Ukq indexed by ik) or int32 [nk] (Ukq indexed by kq_idx[ik]).
 * Small (Nb, Nm): one CTA per pair in shared memory; otherwise two epw_zgemm_strided contractions (needs
 * stride_gt == Nb^2 Nm there; allocates and frees a temporary of the size of gt, synchronising the stream). */
int epw_rotate_g2(const void *gt, int64_t stride_gt, const void *Uk, const void *Ukq, const int32_t *kq_idx,
                  int32_t nb, int32_t nm, int64_t nk, double *g2, void *cuda_stream);

/* -------------------------------------------------------------------------------------------------
 * Eq. 6, the step before the hot path: coarse-grid Bloch representation -> g(Re,Rp).
 * Device pointers; both calls synchronise the stream before returning (temporary workspace).
 * ----------------------------------------------------------------------------------------------- */

/* Gauge part of Eq. 6 for every (k',q') block of a coarse grid:
 *   gt[iq][ik][ka][n'][m'] = sum_{m n nu} Ukq[iq][ik][m',m] g[iq][ik][nu][n][m] conj(Uk[ik][n',n]) sqrt(2 omega[iq][nu]) conj(e[iq][ka,nu])
 * (the inverse of S4a + S4b; paper-U = V^dagger, u = e/sqrt(2 omega): DESIGN.md readings G3, G4).
 *   g_bloch c128 [nqc][nkc][Nm][Nb][Nb] (m fastest), Uk c128 [nkc][Nb][Nb], Ukq c128 [nqc][nkc][Nb][Nb] (column-major,
 *   columns = eigenvectors), e_q c128 [nqc][Nm][Nm] (columns = mode eigenvectors), omega_q f64 [nqc][Nm] (> 0),
 *   gt_out c128 [nqc][nkc][Nm][Nb][Nb] (may not alias g_bloch). */
int epw_eq6_unrotate(const void *g_bloch, const void *Uk, const void *Ukq, const void *e_q, const double *omega_q,
                     int32_t nb, int32_t nm, int64_t nkc, int64_t nqc, void *gt_out, void *cuda_stream);

/* The two inverse Fourier sums of Eq. 6 in the Wannier gauge:
 *   g_RR[ip][ka][ie][n'][m'] = 1/(Ne Np) sum_{iq,ik} gt[iq][ik][ka][n'][m'] exp(-2 pi i (q'_iq . Rp_ip + k'_ik . Re_ie))
 * with the normalisation as printed in the paper (Ne, Np = numbers of lattice vectors; for one vector per residue
 * class of the coarse grids this is the exact inverse of the interpolation).
 *   gt c128 [nqc][nkc][Nm][Nb][Nb], kc f64 [nkc][3], qc f64 [nqc][3] (crystal coordinates), Re int32 [ne][3],
 *   Rp int32 [np][3]; g_RR_out c128 [np][Nm][ne][Nb][Nb] -- the layout epw_interp_set_wannier_operators takes.
 * Runs as two in-place FP64 tensor-path contractions (zgemm_strided.cu) with conjugated phase tables. */
int epw_wannier_from_bloch(const void *gt, const double *kc, int64_t nkc, const double *qc, int64_t nqc, const int32_t *Re,
                           int32_t ne, const int32_t *Rp, int32_t np, int32_t nb, int32_t nm, void *g_RR_out,
                           void *cuda_stream);

/* Roofline denominators measured on this device ("Measurement"): FP64 tensor (DMMA m8n8k4) TFLOP/s,
 * plain DFMA TFLOP/s and HBM read / copy GB/s from tight probe kernels.  out[0..3]; returns 0 or a status. */
int epw_probe_peaks(int32_t device, double *out4);

const char *epw_version(void);

#ifdef __cplusplus
}
#endif
#endif /* EPW_INTERP_H_ */
