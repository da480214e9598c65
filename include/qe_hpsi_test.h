/* qe_hpsi_test.h -- measurement and test helpers exported by libqe_hpsi.so.  NOT part of the product boundary
 * (include/qe_hpsi.h): nothing here is needed to apply H; tests/, bench.py and __graft_entry__.smoke() use these to look
 * at single stages of the path (the three terms), to time them, and to measure the FP64 peak the
 * roofline is quoted against.  Same conventions as qe_hpsi.h. */
#ifndef QE_HPSI_TEST_H
#define QE_HPSI_TEST_H

#include "qe_hpsi.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Stand-alone stage entry points (the same kernels the hot path launches):
 *   qe_hpsi_fft_local: hpsi = g2kin*psi + local term only (a1-a5), ignoring projectors.
 *   qe_hpsi_nonlocal:  hpsi += beta D beta^H psi (a6-a8) on top of the caller's hpsi contents. */
int qe_hpsi_fft_local(qe_hpsi_t h, const void* psi_dev, int64_t ldpsi, void* hpsi_dev, int64_t ldhpsi, int nbands,
                      void* cuda_stream);
int qe_hpsi_nonlocal(qe_hpsi_t h, const void* psi_dev, int64_t ldpsi, void* hpsi_dev, int64_t ldhpsi, int nbands,
                     void* cuda_stream);
/* becp = beta^H psi (a6) and dbecp = D becp (a7) of the LAST chunk applied, as complex128 [nproj][nb_last]
 * band-contiguous, into caller DEVICE arrays (either may be NULL).  With QE_HPSI_PROJ_CERTIFY: of the int8 pass. */
int qe_hpsi_get_becp(qe_hpsi_t h, void* becp_dev, void* dbecp_dev, void* cuda_stream);
/* Number of kernel launches qe_hpsi_apply enqueues for nbands bands (the benchmark's gpu_launches). */
int64_t qe_hpsi_launch_count(qe_hpsi_t h, int nbands);

/* Stage timing for the roofline report.  mode 0 = off (default; apply records no events), 1 = CUDA events around
 * a6 (slot 0), a7 (slot 1), the whole a1-a5 chain (slot 2) and a8 (slot 3) of every chunk, 2 = additionally
 * around each of the five FFT kernels a1..a5 (slots 4..8; slot 2 is then not recorded); slot 9 = digit kernels of the
 * int8 path, slot 10 = check + FP64 re-computation of QE_HPSI_PROJ_CERTIFY.  Events are recorded on the stream passed
 * to apply.  qe_hpsi_profile resets the accumulators; qe_hpsi_profile_read synchronises the pending events and returns,
 * per slot, the summed milliseconds and the number of spans. */
int qe_hpsi_profile(qe_hpsi_t h, int mode);
int qe_hpsi_profile_read(qe_hpsi_t h, double ms[16], int64_t count[16]);

/* Runs register-resident FP64 DMMA (mma.sync m8n8k4.f64) and DFMA loops on every SM for about `millis` ms each and
 * returns the achieved TFLOP/s.  bench.py uses the DMMA figure as the measured FP64 tensor peak of the box (neither
 * MEASURED_PEAKS.json nor the profiling guide has an FP64 entry).  Synchronises the device. */
int qe_hpsi_probe_fp64(double millis, double* dmma_tflops, double* dfma_tflops);

/* (testing) cap, in reals, on the K range one CTA of the int8 GEMMs sums exactly in int32; 0 = the natural 2^17/S.
 * Read by the next qe_hpsi_create: lowering it makes small cases take the multi-range paths of big ones (a6 split
 * finer, a8 walking its K ranges launch by launch).  Process-wide; not for production use. */
int qe_hpsi_test_set_int8_kmax(int64_t kmax);

/* (testing) smallest nproj * npw from which the Gamma-symmetric projector mode (qe_hpsi.h, QE_HPSI_NO_GAMMA_SYM) is used by
 * handles created from now on; default 2^20 (smaller steps are launch-latency bound; both forms are FP64), negative = default,
 * 0 = always.  Lets the tests run the symmetric kernels on tiny cases the oracle can check with a dense H.  Process-wide. */
int qe_hpsi_test_set_sym_min(int64_t entries);

/* Guard bands (the pool's GPUs do not run compute-sanitizer): every device buffer a handle owns is allocated with a
 * pattern-filled tail of 256..511 bytes.  Synchronises the device and returns the number of buffers whose tail was
 * overwritten (0 = no kernel wrote past the end of a workspace since create), or a negative status. */
int64_t qe_hpsi_test_check_guards(qe_hpsi_t h);

#ifdef __cplusplus
}
#endif
#endif /* QE_HPSI_TEST_H */
