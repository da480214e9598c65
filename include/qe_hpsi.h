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
 * This header is the PRODUCT boundary.  Measurement and test helpers (stage entry points, stage timers, the FP64
 * peak probe, launch counts) are exported by the same library but declared in qe_hpsi_test.h.
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
 *   - Arithmetic: FP64 throughout by default.  The only other accuracy class (int8 digit products for the projector
 *     contractions) is an explicit create flag, never chosen by problem size, device or environment.
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
  QE_HPSI_EINVAL = -1, /* null pointer, negative size, ld < npw, psi aliases hpsi, bad block table, bad flags, */
                       /* complex128 array not 16-byte aligned                                            */
  QE_HPSI_EGRID = -2,  /* N_j has a prime factor other than 2,3,5, exceeds QE_HPSI_MAX_N, or is smaller  */
                       /* than the sphere's index extent along j (the sphere itself would wrap)          */
  QE_HPSI_ENOMEM = -3, /* host or device allocation failed (including the digit planes of QE_HPSI_PROJ_INT8) */
  QE_HPSI_ECUDA = -4,  /* CUDA runtime error; the cudaError_t is returned by qe_hpsi_last_error          */
  QE_HPSI_ESTATE = -5  /* handle is NULL / destroyed / not prepared for the call                         */
} qe_hpsi_status;

/* flags for qe_hpsi_create */
#define QE_HPSI_BORROW_BETA 1u   /* use beta_dev in place (caller keeps it alive and unchanged) instead of copying */
#define QE_HPSI_GENERIC_FFT 2u   /* (testing) use only radices 2,3,4,5 in the FFT passes                           */
#define QE_HPSI_FP64_DMMA   4u   /* projector contractions a6 / a8 on the FP64 tensor pipe (mma.sync DMMA, 3M       */
                                 /* product).  THIS IS THE DEFAULT (the flag only names it): every product and sum   */
                                 /* of the path is IEEE FP64, as in the paper's port (cuBLAS FP64 GEMM) */
/* Opt-in accuracy class for a6 / a8: the FP64 operands are split into S signed 8-bit digits under one exponent per
 * row (projector, plane wave or band), the digit products are summed EXACTLY on the int8 tensor cores (tcgen05
 * kind::i8, int32 level sums in TMEM) and recombined in FP64.  This is block fixed point, not FP64: per contraction
 *     |error| <= ~(S+1) 2^(-8S+1) K max|a| max|b|     (K = contraction length; relative to the ROW MAXIMA, not the entry)
 * i.e. 8S-1 bits under the row exponent: S = 7 -> 55 bits, S = 6 -> 47 bits.  Digits: QE_HPSI_PROJ_DIGITS(4..7);
 * 0 = 7.  Costs 3 S bytes per complex entry of beta for a6 and 3 S for a8 of device memory (2 S each for small
 * problems) NEXT TO the FP64 beta: at S = 6 that is 2.25 x the size of beta (56 GB for the 25 GB beta of the
 * largest benchmark workload), 2.6 x at S = 7; in the Gamma-symmetric mode (k = 0, see QE_HPSI_NO_GAMMA_SYM below) the
 * planes hold real forms over the half sphere, 2 S bytes per complex entry of beta in all: 0.75 x the size of beta at
 * S = 6 (19 GB for that workload).  If those planes cannot be allocated qe_hpsi_create FAILS with
 * QE_HPSI_ENOMEM; it never changes the arithmetic silently.  Non-finite operands give NaN for the affected
 * projector / band.  Needs an sm_100 device (tcgen05).
 * QE_HPSI_PROJ_CERTIFY (with QE_HPSI_PROJ_INT8) adds an a-posteriori check of every int8 result and the automatic
 * FP64 re-computation of the bands that fail it: see qe_hpsi_set_proj_tolerance. */
#define QE_HPSI_PROJ_INT8    8u
#define QE_HPSI_PROJ_CERTIFY 16u
#define QE_HPSI_PROJ_DIGITS(s) (((unsigned)(s) & 15u) << 8)
/* integer 3M forms of the int8 contractions (three real digit GEMMs per complex product instead of four).  Default:
 * chosen by size (a6 from 2^26 entries of beta, a8 from 1536 projectors).  The forms differ in rounding only. */
#define QE_HPSI_PROJ_3M_OFF (1u << 12)
#define QE_HPSI_PROJ_3M_A6  (2u << 12)
#define QE_HPSI_PROJ_3M_ALL (3u << 12)

/* At k = 0 the library checks at create, bit for bit, whether every projector obeys beta_p(-G) = +-conj(beta_p(G)) (projector
 * functions real in real space) and D couples equal signs only; if so a6 / a8 contract psi = u + i v as two real-wavefunction
 * problems over the half sphere: 2/3 of the FP64 tensor work and half of the beta traffic, same FP64 arithmetic, results equal
 * to the general path up to rounding order.  The int8 digit path does the same with real-form digit
 * planes over the half sphere (a third of the plane memory).  This flag keeps the general complex contraction. */
#define QE_HPSI_NO_GAMMA_SYM 32u

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
 *   flags      OR of the QE_HPSI_* flags above; unknown bits, QE_HPSI_FP64_DMMA together with QE_HPSI_PROJ_INT8, a digit
 *              count outside 4..7, or QE_HPSI_PROJ_CERTIFY / DIGITS / 3M without QE_HPSI_PROJ_INT8 give QE_HPSI_EINVAL.
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
 * Asynchronous: all work is enqueued on cuda_stream, no host synchronisation, no device->host traffic (also with
 * QE_HPSI_PROJ_CERTIFY: the check and the re-computation are decided on the device).  Only argument errors are
 * reported synchronously.  One in-flight apply per handle (the workspace is shared). */
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

/* ---- accessors -------------------------------------------------------------------------------------------- */
int64_t qe_hpsi_npw(qe_hpsi_t h);            /* sphere size, or a negative status                               */
int64_t qe_hpsi_nsticks(qe_hpsi_t h);        /* S: (i1,i2) columns holding >= 1 sphere point                    */
int64_t qe_hpsi_nplanes(qe_hpsi_t h);        /* P: i1 planes holding >= 1 sphere point                          */
/* Copies the device-built maps into caller DEVICE arrays (any may be NULL): miller [npw][3] int32,
 * fft_index [npw] int32, g2kin [npw] float64.  Enqueued on cuda_stream. */
int qe_hpsi_get_maps(qe_hpsi_t h, int32_t* miller_dev, int32_t* fftidx_dev, double* g2kin_dev, void* cuda_stream);
/* info[0..15]: npw, S, P, fft band chunk, split-K count (FP64 path), workspace bytes, per axis j=0..2 the number of
 * generic FFT passes, K chunk, x split, SM count, [12] bit 0: two-pass FFT plan in use, bit 1: Gamma-symmetric projector mode of
 * the FP64 path in use, bit 2: x stage of the FFT chain with quarter pruning (populated planes within the outer quarters of the
 * axis); then the projector path: [13] digits per
 * FP64 operand of the int8 path (0 = FP64 tensor path), [14] its split-K count of a6, [15] 1 if a6 runs in the
 * integer 3M form, 2 if a8 does too, +4 if QE_HPSI_PROJ_CERTIFY is on. */
int qe_hpsi_info(qe_hpsi_t h, int64_t info[16]);
const char* qe_hpsi_strerror(int status);
int qe_hpsi_last_error(qe_hpsi_t h);         /* cudaError_t of the last QE_HPSI_ECUDA (0 if none); h may be NULL */

/* ---- certified int8 projector path (QE_HPSI_PROJ_INT8 | QE_HPSI_PROJ_CERTIFY) ------------------------------
 * The agreement the paper reports between its CPU and GPU runs is an FP64 statement; the int8
 * digit path is block fixed point and its worst-case bound (above) is far looser than what it delivers on smooth
 * operands.  With QE_HPSI_PROJ_CERTIFY every chunk is checked a posteriori: the nonlocal
 * part v_b = V_NL psi_b computed on the int8 path is kept apart, and for QE_HPSI_NPROBE random sign vectors s_t the
 * identity  sum_G s_t(G) v_b(G) = <y_t|psi_b>,  y_t = V_NL^H s_t  (computed once, in FP64, at create) is tested;
 *     est_b = sqrt( mean_t |sum_G s_t v_b - <y_t|psi_b>|^2 )      estimates ||v_b - V_NL psi_b||_2  (Freivalds / Hutchinson)
 * to within a factor 2 with probability > 0.998 down to the FP64 rounding of the check itself (~1e-15 ||v_b||).
 * Bands with est_b > tol * ||v_b||_2 (or a non-finite value) are re-computed on the FP64 tensor path -- selected, compacted and
 * launched on the device, no host synchronisation -- and the FP64 result is what is added to hpsi.
 * qe_hpsi_set_proj_tolerance: tol >= 0, default 1e-11 (north_star's parity tolerance, demanded of the nonlocal part alone).
 * qe_hpsi_get_proj_check: for the LAST chunk applied, est_b / ||v_b|| per band into rel_dev [nb_last] (FP64, device) and
 *   1 / 0 = re-computed in FP64 / int8 result kept into redo_dev [nb_last] (int32, device); either may be NULL; enqueued
 *   on cuda_stream.  QE_HPSI_ESTATE if the handle was not created with QE_HPSI_PROJ_CERTIFY. */
#define QE_HPSI_NPROBE 8
int qe_hpsi_set_proj_tolerance(qe_hpsi_t h, double tol);
int qe_hpsi_get_proj_check(qe_hpsi_t h, double* rel_dev, int32_t* redo_dev, void* cuda_stream);

/* ---- rows SURVEY.md 8(f) marks "next": same kernels and tables as the hot path ---------------------------- */

/* NEXT-2, overlap operator of ultrasoft/PAW pseudopotentials ("application of the overlap operator",
 * PAPER.md:L226): S = 1 + sum_a sum_ij |beta_ai> q^a_ij <beta_aj|.
 * qe_hpsi_set_s stores the real symmetric q^a blocks (packed exactly like d_host of qe_hpsi_create; COPIED;
 * synchronises).  qe_hpsi_apply_hs computes hpsi = H psi and spsi = S psi in one call: becp = beta^H psi (a6) is
 * computed once and shared; spsi[b][0..npw) is overwritten, entries >= npw untouched; spsi must not overlap psi or
 * hpsi.  hpsi_dev may be NULL (S psi only).  Without projectors S = 1.  QE_HPSI_ESTATE if set_s was never called
 * on a handle that has projectors.  Asynchronous on cuda_stream like qe_hpsi_apply.  (Not certified: with
 * QE_HPSI_PROJ_CERTIFY this call returns QE_HPSI_ESTATE.)  On a QE_HPSI_PROJ_INT8 handle in the Gamma-symmetric mode (k = 0,
 * see QE_HPSI_NO_GAMMA_SYM) the digit planes hold the real forms only, so q must couple projectors of equal parity only
 * (as D does); otherwise qe_hpsi_set_s returns QE_HPSI_EINVAL and the handle should be created with QE_HPSI_NO_GAMMA_SYM. */
int qe_hpsi_set_s(qe_hpsi_t h, const double* q_host);
int qe_hpsi_apply_hs(qe_hpsi_t h, const void* psi_dev, int64_t ldpsi, void* hpsi_dev, int64_t ldhpsi, void* spsi_dev,
                     int64_t ldspsi, int nbands, void* cuda_stream);

/* NEXT-3, reduced matrices of the iterative diagonaliser: out[i][j] = <a_i|b_j> =
 * sum_G conj(a[i][G]) b[j][G] over the npw sphere entries, i < na, j < nb.  a_dev [na][lda], b_dev [nb][ldb]
 * complex128 (may be the same array), out_dev [na][ldo] complex128, ldo >= nb (entries j >= nb untouched).  Runs the
 * split-K DMMA kernel of step a6 with a fixed-order reduction (bit-reproducible).  Asynchronous on cuda_stream: no
 * allocation, no synchronisation (the split-K workspace is part of the handle). */
int qe_hpsi_overlap(qe_hpsi_t h, const void* a_dev, int64_t lda, int na, const void* b_dev, int64_t ldb, int nb,
                    void* out_dev, int64_t ldo, void* cuda_stream);

/* The same reduced matrix for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc): no handle, and neither set-up nor call uses cudaMalloc / cudaFree or an allocating library routine.  The
 * split-K partials live in ONE file-scope device array of 8 MiB (32 slices x 128 x 128 complex128) that every GPU loading the
 * library holds until exit.  Limits: na, nb <= QE_HPSI_OVERLAP_STATIC_MAX, npw < 2^31 - 4096; anything beyond returns
 * QE_HPSI_EINVAL and launches nothing.  a_dev [na][lda], b_dev [nb][ldb], out_dev [na][ldo] as for qe_hpsi_overlap, summed over the
 * leading npw entries of the rows; same K slices, kernel and reduction order, hence the same bits as qe_hpsi_overlap on a handle
 * with that npw.  Asynchronous on cuda_stream.  ALL calls on a device share the array (it keeps the last call's partials;
 * nothing in it has to start at zero): calls that can overlap on the GPU -- different streams, or graph branches -- race; order
 * them.  qe_hpsi_overlap_static_init does the once-per-device set-up (device address of the array, kernel attributes) for the
 * CURRENT device; the call does it on first use, so call init before a stream capture begins. */
#define QE_HPSI_OVERLAP_STATIC_MAX 128
int qe_hpsi_overlap_static_init(void);
int qe_hpsi_overlap_static(const void* a_dev, int64_t lda, int na, const void* b_dev, int64_t ldb, int nb, int64_t npw,
                           void* out_dev, int64_t ldo, void* cuda_stream);

/* NEXT-3, the rest of the Davidson step:
 * qe_hpsi_hdiag:   hdiag[G] = |k+G|^2 + vbar + sum_p D_pp |beta_p(G)|^2  (vbar = mean of V(r), supplied by the caller)
 *                  sdiag[G] = 1 + sum_p q_pp |beta_p(G)|^2              (needs qe_hpsi_set_s when there are projectors)
 *                  either output may be NULL; DEVICE arrays of npw doubles.
 * qe_hpsi_precond: r[b][G] /= (1 + x + sqrt(1 + (x-1)^2)) / 2, x = hdiag[G] - e[b] sdiag[G]; e_dev [nb] on the device,
 *                  sdiag_dev NULL means 1.
 * qe_hpsi_rotate:  y[k][G] (+)= sum_j coef[k][j] x[j][G], k < ny, j < nx, over the npw sphere entries; coef_dev complex128
 *                  [ny][ldcoef], ldcoef >= nx; accumulate = 0 overwrites y[k][0..npw) (store-only epilogue: y is not read).  Runs the DMMA kernel of step a8.
 *                  All arguments are validated before anything is written.
 * qe_hpsi_residual: r[b][G] = hx[b][G] - e[b] sx[b][G] for G < npw (r may be hx or sx), and rnorm2[b] = sum_G |r[b][G]|^2
 *                  (rnorm2_dev [nb] FP64 on the device, may be NULL; fixed summation order, bit-reproducible).
 * qe_hpsi_scale:   x[b][G] *= fac[b] (fac_dev [nb] FP64 on the device), e.g. normalisation of correction vectors.
 * All asynchronous on cuda_stream. */
int qe_hpsi_hdiag(qe_hpsi_t h, double vbar, double* hdiag_dev, double* sdiag_dev, void* cuda_stream);
int qe_hpsi_precond(qe_hpsi_t h, void* r_dev, int64_t ldr, int nb, const double* e_dev, const double* hdiag_dev,
                    const double* sdiag_dev, void* cuda_stream);
int qe_hpsi_rotate(qe_hpsi_t h, const void* x_dev, int64_t ldx, int nx, const void* coef_dev, int64_t ldcoef, void* y_dev,
                   int64_t ldy, int ny, int accumulate, void* cuda_stream);
int qe_hpsi_residual(qe_hpsi_t h, const void* hx_dev, int64_t ldh, const void* sx_dev, int64_t lds, const double* e_dev,
                     void* r_dev, int64_t ldr, int nb, double* rnorm2_dev, void* cuda_stream);
int qe_hpsi_scale(qe_hpsi_t h, void* x_dev, int64_t ldx, int nb, const double* fac_dev, void* cuda_stream);

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
 * the projectors as real matrices over the 2*ngw real components.  Arguments as qe_hpsi_create / qe_hpsi_apply (no k);
 * flags as for qe_hpsi_create except QE_HPSI_PROJ_CERTIFY (QE_HPSI_EINVAL). */
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
