/* qe_hpsi.h -- C ABI of libqe_hpsi.so: H|psi> for plane-wave pseudopotential Kohn-Sham on one NVIDIA B200.
 *
 * What the library computes.  The paper (PAPER.md, arXiv:2104.10502) names the operation -- "Hamiltonian
 * builds (i.e. the application of the one-particle Hamiltonian to molecular orbitals and Bloch states)",
 * PAPER.md:L105 section III -- and its three terms -- "local-potential, pseudopotential, kinetic-energy
 * contributions to the Hamiltonian", section III.C -- plus "generation of plane waves and of
 * their mapping to FFT grids", PAPER.md:L176 (vi).  It prints no formula; BASELINE.json's north_star fixes
 *
 *     (H psi)(G) = |k+G|^2 psi(G) + sum_G' V(G-G') psi(G') + sum_a sum_ij beta_ai(G) D^a_ij <beta_aj|psi>
 *
 * in Rydberg atomic units (lengths bohr, energies Ry), with V(G-G') the 3-D DFT coefficient of the supplied
 * real-space array V(r) at the cyclically wrapped index difference.  The library is a
 * self-contained object with a flat API in the sense of PAPER.md:L112/L152/L156, callable as the external
 * H builder of an iterative eigensolver; the caller owns streams and synchronisation
 * (PAPER.md:L134-136).
 *
 * Conventions shared by all calls
 *   - `at[9]`: lattice vectors a_1,a_2,a_3 as rows (row-major 3x3), bohr.  Reciprocal rows b_j, a_i.b_j = 2 pi d_ij.
 *   - `xk[3]`: Cartesian k in bohr^-1.  `nr[3]`: FFT grid N1,N2,N3; every N_j must factor into 2,3,5.
 *   - Miller triple n, G = sum n_j b_j; wrapped index i_j = n_j mod N_j; linear index idx = (i1*N2+i2)*N3+i3.
 *   - The sphere {G : |k+G|^2 <= ecutwfc} (inclusive) is ordered by ASCENDING idx ("canonical order"); psi,
 *     hpsi and beta rows are indexed by position ig in that order.
 *   - complex128 = interleaved (re,im) doubles.  psi/hpsi: band-major [nbands][ld], beta: [nproj][ldbeta].
 *   - psi(r) = sum_G c(G) exp(+i(k+G).r): sphere -> grid uses the un-normalised exp(+) DFT, grid -> sphere the
 *     exp(-) DFT with 1/N.
 *   - "dev" pointers are CUDA device pointers on the current device, "host" pointers ordinary host memory.
 *   - Every function returns 0 (QE_HPSI_OK) or a negative qe_hpsi_status; none throws, aborts or exits.
 *   - There is no CPU fallback: without a CUDA device every compute entry point returns QE_HPSI_ECUDA.
 */
#ifndef QE_HPSI_H
#define QE_HPSI_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qe_hpsi_handle* qe_hpsi_t;

typedef enum {
  QE_HPSI_OK = 0,
  QE_HPSI_EINVAL = -1, /* null pointer, negative size, ld < npw, psi aliases hpsi, bad block table        */
  QE_HPSI_EGRID = -2,  /* N_j has a prime factor other than 2,3,5, exceeds QE_HPSI_MAX_N, or is smaller  */
                       /* than the sphere's index extent along j (the sphere itself would wrap)          */
  QE_HPSI_ENOMEM = -3, /* host or device allocation failed                                               */
  QE_HPSI_ECUDA = -4,  /* CUDA runtime error; the cudaError_t is returned by qe_hpsi_last_cuda_error     */
  QE_HPSI_ESTATE = -5  /* handle is NULL / destroyed                                                     */
} qe_hpsi_status;

/* flags for qe_hpsi_create */
#define QE_HPSI_BORROW_BETA 1u   /* use beta_dev in place (caller keeps it alive and unchanged) instead of copying */
#define QE_HPSI_GENERIC_FFT 2u   /* (testing) use only radices 2,3,4,5 in the FFT passes                           */
#define QE_HPSI_FP64_DMMA   4u   /* projector contractions a6 / a8 on the FP64 tensor pipe (mma.sync DMMA, 3M product) */
                                 /* instead of the default: the FP64 operands are split error-free into S = 6 signed */
                                 /* 8-bit digits (per-row exponent) whose products are summed exactly on the int8    */
                                 /* tensor cores (tcgen05, int32 level sums in TMEM) and recombined in FP64:         */
                                 /* |error| <= ~(S+1) 2^(-8S+1) K max|a| max|b| per contraction (2^-47 = 7e-15);     */
                                 /* costs 3 S bytes per complex entry of beta for a6 and 3 S for a8 (planes Re, Im,  */
                                 /* half sum of the integer 3M forms; 2 S each for small problems).                  */
                                 /* Default only when nproj * npw >= 2^20 (smaller steps are launch-latency bound).  */
                                 /* Env QE_HPSI_OZAKI = 0 | 4..7 forces the digit count (0 = same as this flag).     */
                                 /* Non-finite operands are not propagated by the int8 path (use this flag for them). */

#define QE_HPSI_MAX_N 720        /* largest supported FFT dimension (shared-memory pencil tile)                     */

/* a0, stand-alone (PAPER.md:L176 (vi)).  Canonical sphere for a cell / k / cutoff / grid before any handle
 * exists, so that the caller can lay out psi and beta.  Two-call pattern: with miller_host == NULL only
 * *npw is written; otherwise miller_host[3*npw] (host, int32, triples n1,n2,n3 in canonical order) is filled
 * and must hold at least 3 * (*npw as returned by the first call) entries.  Runs kernel a0 on the current
 * device and synchronises. */
int qe_hpsi_gsphere(const double at[9], const double xk[3], double ecutwfc, const int nr[3],
                    int64_t* npw, int32_t* miller_host);

/* Build a handle (once per k-point / potential update).
 *   vr_dev     [N1][N2][N3] real FP64 local potential V(r) in Ry, i3 contiguous, r = sum (i_j/N_j) a_j.  COPIED
 *              (pre-scaled by 1/N).
 *   nproj      total number of projectors (0 allowed: kinetic + local only; beta/blocks then ignored).
 *   beta_dev   complex128 [nproj][ldbeta], ldbeta >= npw, canonical G order.  Copied unless QE_HPSI_BORROW_BETA.
 *   nblocks, blk_off_host[nblocks+1]   atoms: block a owns projectors blk_off[a] .. blk_off[a+1]-1;
 *              blk_off[0] = 0, strictly increasing, blk_off[nblocks] = nproj.
 *   d_host     the real symmetric D^a blocks packed one after another, block a row-major nh_a x nh_a
 *              (nh_a = blk_off[a+1]-blk_off[a]), Ry.  COPIED.
 *   max_batch  largest number of bands processed as one internal chunk (workspace is sized for it), >= 1.
 *   cuda_stream  cudaStream_t (NULL = default stream) on which create's device work is enqueued; create
 *              synchronises that stream before returning.
 * On failure *out = NULL. */
int qe_hpsi_create(qe_hpsi_t* out, const double at[9], double ecutwfc, const double xk[3], const int nr[3],
                   const double* vr_dev, int nproj, const void* beta_dev, int64_t ldbeta, int nblocks,
                   const int32_t* blk_off_host, const double* d_host, int max_batch, unsigned flags,
                   void* cuda_stream);

/* The hot path (steps a1-a8 of DESIGN.md): hpsi[b][0..npw) = (H psi_b) for b < nbands.
 *   psi_dev  [nbands][ldpsi] complex128 (read only), hpsi_dev [nbands][ldhpsi] complex128 (overwritten, not
 *   accumulated; entries ig >= npw of each row untouched).  ldpsi, ldhpsi >= npw.  The two arrays must not
 *   overlap.  Any nbands >= 0; internally processed in chunks of at most max_batch bands; the result for a
 *   band does not depend on which other bands are in the call.
 * Asynchronous: all work is enqueued on cuda_stream, no host synchronisation, no device->host traffic.  Only
 * argument errors are reported synchronously.  One in-flight apply per handle (the workspace is shared). */
int qe_hpsi_apply(qe_hpsi_t h, const void* psi_dev, int64_t ldpsi, void* hpsi_dev, int64_t ldhpsi, int nbands,
                  void* cuda_stream);

/* End-to-end variant with HOST buffers (pinned memory recommended): per internal chunk copies psi host->device,
 * applies H, copies hpsi device->host, overlapping copies with compute on internal streams.  Returns after
 * the last copy has completed (synchronous).  Same layouts and rules as qe_hpsi_apply. */
int qe_hpsi_apply_host(qe_hpsi_t h, const void* psi_host, int64_t ldpsi, void* hpsi_host, int64_t ldhpsi,
                       int nbands);

/* Frees everything the handle owns.  NULL is a no-op.  The caller must have synchronised every stream that
 * used the handle. */
int qe_hpsi_destroy(qe_hpsi_t h);

/* ---- accessors (needed for the bit-exact map check, the roofline report and diagnostics) ---- */
int64_t qe_hpsi_npw(qe_hpsi_t h);            /* sphere size, or a negative status                               */
int64_t qe_hpsi_nsticks(qe_hpsi_t h);        /* S: (i1,i2) columns holding >= 1 sphere point                    */
int64_t qe_hpsi_nplanes(qe_hpsi_t h);        /* P: i1 planes holding >= 1 sphere point                          */
/* Copies the device-built maps into caller DEVICE arrays (any may be NULL): miller [npw][3] int32,
 * fft_index [npw] int32, g2kin [npw] float64.  Enqueued on cuda_stream. */
int qe_hpsi_get_maps(qe_hpsi_t h, int32_t* miller_dev, int32_t* fftidx_dev, double* g2kin_dev, void* cuda_stream);
/* Stage access for tests: becp = beta^H psi (a6) and dbecp = D becp (a7) of the LAST chunk applied, as
 * complex128 [nproj][nb_last] band-contiguous, into caller DEVICE arrays (either may be NULL). */
int qe_hpsi_get_becp(qe_hpsi_t h, void* becp_dev, void* dbecp_dev, void* cuda_stream);
/* Number of kernel launches qe_hpsi_apply enqueues for nbands bands (for the benchmark's gpu_launches). */
int64_t qe_hpsi_launch_count(qe_hpsi_t h, int nbands);
/* info[0..15]: npw, S, P, fft band chunk, split-K count (FP64 path), workspace bytes, per axis j=0..2 the number of
 * generic FFT passes, K chunk, x split, SM count, two-pass FFT plan in use, then the projector path: [13] digits per
 * FP64 operand of the int8 path (0 = FP64 tensor path), [14] its split-K count of a6, [15] 1 if a6 runs in the
 * integer 3M form, 2 if a8 does too.  For the roofline report and the tests. */
int qe_hpsi_info(qe_hpsi_t h, int64_t info[16]);
const char* qe_hpsi_strerror(int status);
int qe_hpsi_last_cuda_error(qe_hpsi_t h);    /* cudaError_t of the last QE_HPSI_ECUDA (0 if none)               */

/* Stage timing for the roofline report.  mode 0 = off (default; apply records no events), 1 = CUDA events around
 * a6 (slot 0), a7 (slot 1), the whole a1-a5 chain (slot 2) and a8 (slot 3) of every chunk, 2 = additionally
 * around each of the five FFT kernels a1..a5 (slots 4..8; slot 2 is then not recorded).  Events are recorded
 * on the stream passed to apply.  qe_hpsi_profile resets the accumulators; qe_hpsi_profile_read synchronises
 * the pending events and returns, per slot, the summed milliseconds and the number of spans. */
int qe_hpsi_profile(qe_hpsi_t h, int mode);
int qe_hpsi_profile_read(qe_hpsi_t h, double ms[16], int64_t count[16]);

/* Measurement helper (not on the hot path): runs register-resident FP64 DMMA (mma.sync m8n8k4.f64) and DFMA
 * loops on every SM for about `millis` ms each and returns the achieved TFLOP/s.  bench.py uses the DMMA
 * figure as the measured FP64 tensor peak of the box.  Synchronises the device. */
int qe_hpsi_probe_fp64(double millis, double* dmma_tflops, double* dfma_tflops);

/* Stand-alone stage entry points for tests and micro-benchmarks (same kernels the hot path launches):
 *   qe_hpsi_fft_local: hpsi = g2kin*psi + local term only (a1-a5), ignoring projectors.
 *   qe_hpsi_nonlocal:  hpsi += beta D beta^H psi (a6-a8) on top of the caller's hpsi contents. */
int qe_hpsi_fft_local(qe_hpsi_t h, const void* psi_dev, int64_t ldpsi, void* hpsi_dev, int64_t ldhpsi, int nbands,
                      void* cuda_stream);
int qe_hpsi_nonlocal(qe_hpsi_t h, const void* psi_dev, int64_t ldpsi, void* hpsi_dev, int64_t ldhpsi, int nbands,
                     void* cuda_stream);

/* ---- rows SURVEY.md 8(f) marks "next": same kernels and tables as the hot path ---------------------------- */

/* NEXT-2, overlap operator of ultrasoft/PAW pseudopotentials ("application of the overlap operator",
 * PAPER.md:L226): S = 1 + sum_a sum_ij |beta_ai> q^a_ij <beta_aj|.
 * qe_hpsi_set_s stores the real symmetric q^a blocks (packed exactly like d_host of qe_hpsi_create; COPIED;
 * synchronises).  qe_hpsi_apply_hs computes hpsi = H psi and spsi = S psi in one call: becp = beta^H psi (a6) is
 * computed once and shared; spsi[b][0..npw) is overwritten, entries >= npw untouched; spsi must not overlap psi or
 * hpsi.  hpsi_dev may be NULL (S psi only).  Without projectors S = 1.  QE_HPSI_ESTATE if set_s was never called
 * on a handle that has projectors.  Asynchronous on cuda_stream like qe_hpsi_apply. */
int qe_hpsi_set_s(qe_hpsi_t h, const double* q_host);
int qe_hpsi_apply_hs(qe_hpsi_t h, const void* psi_dev, int64_t ldpsi, void* hpsi_dev, int64_t ldhpsi, void* spsi_dev,
                     int64_t ldspsi, int nbands, void* cuda_stream);

/* NEXT-3, reduced matrices of the iterative diagonaliser: out[i][j] = <a_i|b_j> =
 * sum_G conj(a[i][G]) b[j][G] over the npw sphere entries, i < na, j < nb.  a_dev [na][lda], b_dev [nb][ldb]
 * complex128 (may be the same array), out_dev [na][ldo] complex128, ldo >= nb (entries j >= nb untouched).  Runs the
 * split-K DMMA kernel of step a6 with a fixed-order reduction (bit-reproducible).  Asynchronous on cuda_stream. */
int qe_hpsi_overlap(qe_hpsi_t h, const void* a_dev, int64_t lda, int na, const void* b_dev, int64_t ldb, int nb,
                    void* out_dev, int64_t ldo, void* cuda_stream);

/* NEXT-3, the rest of the Davidson step:
 * qe_hpsi_hdiag:   hdiag[G] = |k+G|^2 + vbar + sum_p D_pp |beta_p(G)|^2  (vbar = mean of V(r), supplied by the caller)
 *                  sdiag[G] = 1 + sum_p q_pp |beta_p(G)|^2              (needs qe_hpsi_set_s when there are projectors)
 *                  either output may be NULL; DEVICE arrays of npw doubles.
 * qe_hpsi_precond: r[b][G] /= (1 + x + sqrt(1 + (x-1)^2)) / 2, x = hdiag[G] - e[b] sdiag[G]; e_dev [nb] on the device,
 *                  sdiag_dev NULL means 1.
 * qe_hpsi_rotate:  y[k][G] (+)= sum_j coef[k][j] x[j][G], k < ny, j < nx, over the npw sphere entries; coef_dev complex128
 *                  [ny][ldcoef], ldcoef >= nx; accumulate = 0 overwrites y[k][0..npw).  Runs the DMMA kernel of step a8.
 * All asynchronous on cuda_stream. */
int qe_hpsi_hdiag(qe_hpsi_t h, double vbar, double* hdiag_dev, double* sdiag_dev, void* cuda_stream);
int qe_hpsi_precond(qe_hpsi_t h, void* r_dev, int64_t ldr, int nb, const double* e_dev, const double* hdiag_dev,
                    const double* sdiag_dev, void* cuda_stream);
int qe_hpsi_rotate(qe_hpsi_t h, const void* x_dev, int64_t ldx, int nx, const void* coef_dev, int64_t ldcoef, void* y_dev,
                   int64_t ldy, int ny, int accumulate, void* cuda_stream);

/* NEXT-4, charge density ("charge density generation"):
 *   rho[i1][i2][i3] += scale * sum_b occ[b] |psi_b(r_i)|^2,  psi_b(r_i) = sum_G psi[b][G] exp(+2 pi i n.i/N)
 * using steps a1-a2 of the hot path and the inverse half of a3.  rho_dev is a dense [N1][N2][N3] FP64 DEVICE array
 * that is ACCUMULATED into (zero it first for a fresh density); occ_dev [nbands] FP64 on the device.
 * Asynchronous on cuda_stream; bit-reproducible (each grid point is owned by one thread, bands summed in order). */
int qe_hpsi_density(qe_hpsi_t h, const void* psi_dev, int64_t ldpsi, int nbands, const double* occ_dev, double scale,
                    double* rho_dev, void* cuda_stream);

/* NEXT-1, Gamma-only path ("Gamma-point specific algorithms"): k = 0 and real wavefunctions, so only
 * the half sphere is stored, c(-G) = conj(c(G)).  Half rule: G = n1 b1 + n2 b2 + n3 b3 is kept if n1 > 0, or n1 == 0 and
 * n2 > 0, or n1 == n2 == 0 and n3 >= 0; order = the order those G have in the canonical full sphere (G = 0 first).
 * psi, hpsi and beta are complex128 arrays over the ngw half-sphere entries with Im(x[G=0]) = 0; beta(-G) = conj(beta(G))
 * is implied (projector functions real in real space).  The library transforms two bands per complex FFT and contracts
 * the projectors as real matrices over the 2*ngw real components.  Arguments as qe_hpsi_create / qe_hpsi_apply (no k). */
typedef struct qe_hpsi_gamma_handle* qe_hpsi_gamma_t;
int qe_hpsi_gamma_gsphere(const double at[9], double ecutwfc, const int nr[3], int64_t* ngw, int32_t* miller_host);
int qe_hpsi_gamma_create(qe_hpsi_gamma_t* out, const double at[9], double ecutwfc, const int nr[3], const double* vr_dev,
                         int nproj, const void* beta_dev, int64_t ldbeta, int nblocks, const int32_t* blk_off_host,
                         const double* d_host, int max_batch, unsigned flags, void* cuda_stream);
int qe_hpsi_gamma_apply(qe_hpsi_gamma_t g, const void* psi_dev, int64_t ldpsi, void* hpsi_dev, int64_t ldhpsi, int nbands,
                        void* cuda_stream);
int64_t qe_hpsi_gamma_ngw(qe_hpsi_gamma_t g);
int qe_hpsi_gamma_destroy(qe_hpsi_gamma_t g);

#ifdef __cplusplus
}
#endif
#endif /* QE_HPSI_H */
