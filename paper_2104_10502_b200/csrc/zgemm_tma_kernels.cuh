// zgemm_tma_kernels.cuh -- the FP64 projector contractions (a6 / a8 of DESIGN.md sections 5.3 and 5.8; "pseudopotential ...
// contributions to the Hamiltonian"; "Gamma-point specific algorithms") with the operand tiles
// brought in by TMA instead of per-thread cp.async.
//
// Same tiles, same DMMA order and same epilogues as k_becp / k_vnl_add of zgemm_kernels.cuh (the results are bit-identical);
// what changes is who moves the data.  There every thread issued 8-12 LDGSTS per K tile with their address arithmetic, in the
// issue slots of the warps that feed the DMMA pipe; here ONE thread issues 4 (a6) or 5 (a8) cp.async.bulk.tensor copies per K
// tile that complete on the stage's `full` mbarrier (expect_tx), and the other 255 threads execute DMMA, LDS and the class swap
// only.  Measured on the symmetric a8 kernel at the cfg-4 shape: 0.898 -> 0.955 of the DMMA peak (profiles/r2j_dmma_pipeline.md).
//
// Forms (template parameter FORM), the arithmetic of each as in zgemm_kernels.cuh:
//   ZF_3M    general complex product, 3 real DMMAs per complex block (k != 0, or projectors without the Gamma symmetry)
//   ZF_GAMMA real wavefunctions over the half sphere (Gamma-only handle, NEXT-1)
//   ZF_SYM   Gamma-symmetric projector mode: psi = u + i v as two real problems, class-1 rows as i beta (section 5.8)
//
// Shared-memory layouts are produced by the box shapes and the swizzle mode:
//   M-contiguous operand (beta of a8): one box of BK rows x (BM + 2) complex, no swizzle -> row pitch BM + 2 complex, the pitch
//     that makes the fragment loads of a quarter warp hit 8 distinct 16-byte bank groups (ZgCfg::LDA_M); the 2 extra columns
//     are read but never used.
//   K-contiguous operand of a8 (coefficients, L2-resident): KSTEPS boxes of 4 complex (64 B) x rows -> [k4 group][row][4]: a
//     quarter warp (2 rows x 4 k) reads 128 contiguous bytes.
//   K-contiguous operands of a6 (beta, psi; rows megabytes apart): 2 boxes of 8 complex (128 B) x rows in SWIZZLE_128B mode
//     (16-byte chunk c of row r sits at chunk c ^ (r & 7)), half as many row segments as 64-byte boxes (which made a6 slower
//     than cp.async).  The two rows a quarter warp reads are made to differ in bit 2 (fragment row f -> tile row
//     (f >> 1) | ((f & 1) << 2)), so that their four chunks fall into different 64-byte halves of a 128-byte bank line:
//     conflict-free.  The C fragment carries the same permutation of rows and columns into the epilogue.
// Out-of-range parts of a box (K tail, row tail, columns beyond the sphere) are zero-filled by the TMA unit and count towards
// the transaction bytes, so there is no edge code in the K loop.  Rows of the workspaces beyond the call's band count may hold
// older data: they only reach accumulators of columns the epilogue does not store.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include "zgemm_kernels.cuh"

namespace qehpsi {

enum ZgForm { ZF_3M = 0, ZF_GAMMA = 1, ZF_SYM = 2 };

__device__ __forceinline__ void mb_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("{\n\t.reg .b64 t;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 t, [%0], %1;\n\t}" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_2d(unsigned dst, const CUtensorMap* tm, int c0, int c1, unsigned bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
               "l"(tm), "r"(c0), "r"(c1), "r"(bar)
               : "memory");
}
// full[s] (1 arrival: the issuing thread's expect_tx) at mb0 + 8 s, empty[s] (one arrival per warp) at mb0 + 8 (NSTAGE + s)
template <int NSTAGE, int NT>
__device__ __forceinline__ unsigned mb_setup_tma(unsigned long long* mbar) {
  const unsigned mb0 = static_cast<unsigned>(__cvta_generic_to_shared(mbar));
  if (threadIdx.x == 0) {
    for (int s = 0; s < NSTAGE; ++s) {
      mb_init(mb0 + 8 * s, 1);
      mb_init(mb0 + 8 * (NSTAGE + s), NT / 32);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  return mb0;
}

// a6: partial[ks][p][c] = sum over the K slice ks of conj(A[p][k]) B[c][k] in the arithmetic of FORM (k_becp).
//   tmA: beta as FP64 [nproj][2 npw], tmB: psi (ZF_3M, ZF_GAMMA) or U = (u', v') columns of k_sym_merge (ZF_SYM) as FP64
//   [nb][2 npw]; boxes of 16 doubles x BM / BN rows, SWIZZLE_128B.  npw = entries of the contraction (ZF_SYM: sym_m).
//   Dynamic shared memory: Cfg::SMEM_BECP + 1024 (the swizzle pattern is tied to address bits 7..9).
template <class Cfg, int FORM>
__global__ void __launch_bounds__(Cfg::NT, 1)
    k_becp_tma(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, int nproj, int nb, int npw,
               int kchunk, double2* __restrict__ partial, int ldc, const unsigned char* __restrict__ cls,
               const int* __restrict__ nb_dev, int dead0, int dead1) {
  constexpr int BM = Cfg::BM, BN = Cfg::BN, WM = Cfg::WM, WN = Cfg::WN, BK = Cfg::BK, NSTAGE = Cfg::NSTAGE;
  constexpr int NT = Cfg::NT, TM = Cfg::TM, TN = Cfg::TN, KSTEPS = Cfg::KSTEPS;
  constexpr int STAGE = (BM + BN) * BK;  // complex elements per stage
  static_assert(BK == 16 && (BM * 128) % 1024 == 0 && (BN * 128) % 1024 == 0, "two 128-byte halves per row, 1024-byte aligned boxes");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* sm = reinterpret_cast<double2*>(smem_raw + ((1024u - (static_cast<unsigned>(__cvta_generic_to_shared(smem_raw)) & 1023u)) & 1023u));
  __shared__ __align__(8) unsigned long long mbar[2 * NSTAGE];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm0 = (warp / WN) * (BM / WM), wn0 = (warp % WN) * (BN / WN);
  const int ntn = (nb + BN - 1) / BN;  // the grid was sized for the host-side nb
  const int m0 = (blockIdx.x / ntn) * BM, n0 = (blockIdx.x % ntn) * BN;
  if (nb_dev) {  // QE_HPSI_PROJ_CERTIFY: the band count is decided on the device; tiles beyond it retire at once (see k_becp)
    nb = min(nb, *nb_dev);
    if (n0 >= nb) return;
  }
  const int ks = blockIdx.y;
  const int kb = ks * kchunk, ke = min(npw, kb + kchunk);  // kchunk is a multiple of BK: only the last slice has a ragged tile
  // K tiles [dead0, dead1) (in units of BK entries) hold zeros in B (ZF_SYM: rows of the other half sphere, see k_vnl_tma): the
  // slice walks [t0, ta) and [tb, t1) only.  Adding their exact zeros would not change a bit of the sums.
  const int t0 = kb / BK, t1 = (ke + BK - 1) / BK;
  const int ta = min(t1, max(t0, dead0)), tb = max(t0, min(t1, max(dead1, dead0)));
  const int nk1 = ta - t0, nkt = nk1 + (t1 - tb);
  const unsigned mb0 = mb_setup_tma<NSTAGE, NT>(mbar);
  const unsigned sm0 = static_cast<unsigned>(__cvta_generic_to_shared(sm));

  auto load_stage = [&](int kt, int st) {  // thread 0 only
    if (kt >= NSTAGE) mb_wait(mb0 + 8 * (NSTAGE + st), ((kt / NSTAGE) - 1) & 1);  // every warp is done with the stage's last tile
    const unsigned full = mb0 + 8 * st;
    const unsigned dst = sm0 + (unsigned)(st * STAGE * 16);
    mb_expect_tx(full, STAGE * 16);
    const int k0 = 2 * BK * (kt < nk1 ? t0 + kt : tb + (kt - nk1));
#pragma unroll
    for (int hf = 0; hf < 2; ++hf) {
      tma_load_2d(dst + (unsigned)(hf * BM * 128), &tmA, k0 + 16 * hf, m0, full);
      tma_load_2d(dst + (unsigned)(BM * BK * 16 + hf * BN * 128), &tmB, k0 + 16 * hf, n0, full);
    }
  };

  double P[TM][TN][2], Q[TM][TN][2], R[TM][TN][2];  // R: ZF_3M only
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j)
#pragma unroll
      for (int e = 0; e < 2; ++e) P[i][j][e] = Q[i][j][e] = R[i][j][e] = 0.0;
  if (tid == 0)
    for (int s = 0; s < Cfg::DIST; ++s)
      if (s < nkt) load_stage(s, s);
  const int fr = lane >> 2, fk = lane & 3;
  const int pr = (fr >> 1) | ((fr & 1) << 2);  // tile row (and column) of fragment row fr
  // element (row, k) of a tile [half][rows][8]: chunk (k & 7) ^ (row & 7) of that row in half k >> 3;  row & 7 = pr
  auto at = [&](int nrows, int row, int k) { return (k >> 3) * nrows * 8 + row * 8 + ((k & 7) ^ pr); };
  bool swp[TM];  // ZF_SYM: class 1 rows enter as i beta: fragment swapped to (a_i, a_r), sign in the epilogue (see k_becp)
#pragma unroll
  for (int i = 0; i < TM; ++i) {
    const int p = m0 + wm0 + i * 8 + pr;
    swp[i] = FORM == ZF_SYM && p < nproj && cls[p] != 0;
  }
  int st_c = 0, st_l = Cfg::DIST;
  for (int kt = 0; kt < nkt; ++kt) {
    mb_wait(mb0 + 8 * st_c, (kt / NSTAGE) & 1);
    const double2* As = sm + st_c * STAGE;
    const double2* Bs = As + BM * BK;
    double2 af[2][TM], bf[2][TN];
#pragma unroll
    for (int i = 0; i < TM; ++i) af[0][i] = As[at(BM, wm0 + i * 8 + pr, fk)];
#pragma unroll
    for (int j = 0; j < TN; ++j) bf[0][j] = Bs[at(BN, wn0 + j * 8 + pr, fk)];
#pragma unroll
    for (int kk = 0; kk < KSTEPS; ++kk) {
      if (kk + 1 < KSTEPS) {
#pragma unroll
        for (int i = 0; i < TM; ++i) af[(kk + 1) & 1][i] = As[at(BM, wm0 + i * 8 + pr, (kk + 1) * 4 + fk)];
#pragma unroll
        for (int j = 0; j < TN; ++j) bf[(kk + 1) & 1][j] = Bs[at(BN, wn0 + j * 8 + pr, (kk + 1) * 4 + fk)];
      }
      if constexpr (FORM == ZF_3M) {
        mma3m<TM, TN, true>(P, Q, R, af[kk & 1], bf[kk & 1]);
      } else {
        if constexpr (FORM == ZF_SYM) {
#pragma unroll
          for (int i = 0; i < TM; ++i)
            if (swp[i]) af[kk & 1][i] = make_double2(af[kk & 1][i].y, af[kk & 1][i].x);
        }
        mma2r<TM, TN, true>(P, Q, af[kk & 1], bf[kk & 1]);
      }
      if (kk == 0 && tid == 0 && kt + Cfg::DIST < nkt) load_stage(kt + Cfg::DIST, st_l);
    }
    __syncwarp();
    if (lane == 0) mb_arrive(mb0 + 8 * (NSTAGE + st_c));  // this warp has read the stage
    st_c = (st_c + 1 == NSTAGE) ? 0 : st_c + 1;
    st_l = (st_l + 1 == NSTAGE) ? 0 : st_l + 1;
  }
  double2* out = partial + (size_t)ks * nproj * ldc;
#pragma unroll
  for (int i = 0; i < TM; ++i) {
    const int p = m0 + wm0 + i * 8 + pr;
    if (p >= nproj) continue;
#pragma unroll
    for (int j = 0; j < TN; ++j)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int b = n0 + wn0 + j * 8 + fk + 4 * e;  // fragment column 2 fk + e -> tile column fk | e << 2
        if (b >= nb) continue;
        if constexpr (FORM == ZF_3M)  // conj(a) b = (P + Q) + i (R - P + Q)
          out[(size_t)p * ldc + b] = make_double2(P[i][j][e] + Q[i][j][e], (R[i][j][e] - P[i][j][e]) + Q[i][j][e]);
        else
          out[(size_t)p * ldc + b] = make_double2(swp[i] ? Q[i][j][e] - P[i][j][e] : P[i][j][e] + Q[i][j][e], 0.0);
      }
  }
}

// a8: hpsi[b][g] (+)= sum_p A[p][g] B[b][p] in the arithmetic of FORM (k_vnl_add).
//   tmA: beta as FP64 [nproj][2 npw] (box BK rows x (BM + 2) complex), tmB: coefficient rows as FP64 [nb][2 nproj] (KSTEPS boxes
//   of 4 complex x BN rows): dbT of k_dmul (ZF_3M, ZF_GAMMA: real d in the first slot) or E = (e, +-e) of k_sym_coef (ZF_SYM;
//   then nb = number of real columns = 2 x bands and the epilogue also updates hpsi(-G), see k_vnl_add).
//   overwrite != 0 (ZF_3M): hpsi = product, nothing is read in the epilogue.
template <class Cfg, int FORM>
__global__ void __launch_bounds__(Cfg::NT, 1)
    k_vnl_tma(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, int nproj, int npw, int nb,
              double2* __restrict__ hpsi, long long ldh, const int* __restrict__ nb_dev, const unsigned* __restrict__ cmask,
              const int* __restrict__ minus, int overwrite, const int* __restrict__ live = nullptr, int live0 = 0) {
  static_assert(FORM != ZF_SYM || Cfg::BK == 16, "cmask holds one 16-bit class mask per K tile of 16 projectors");
  constexpr int BM = Cfg::BM, BN = Cfg::BN, WM = Cfg::WM, WN = Cfg::WN, BK = Cfg::BK, NSTAGE = Cfg::NSTAGE;
  constexpr int NT = Cfg::NT, TM = Cfg::TM, TN = Cfg::TN, KSTEPS = Cfg::KSTEPS, LDA = Cfg::LDA_M;
  constexpr int STAGE = BK * LDA + BN * BK;
  static_assert((STAGE * 16) % 128 == 0 && (BK * LDA * 16) % 128 == 0 && (BN * 64) % 128 == 0, "TMA destinations are 128-byte aligned");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* sm = reinterpret_cast<double2*>(smem_raw);
  __shared__ __align__(8) unsigned long long mbar[2 * NSTAGE];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm0 = (warp / WN) * (BM / WM), wn0 = (warp % WN) * (BN / WN);
  const int ntn = (nb + BN - 1) / BN;
  // row tile live0 + blockIdx.x / ntn, taken from the list of tiles that have something to store when there is one (ZF_SYM)
  const int mtile = live0 + (int)(blockIdx.x / ntn);
  const int m0 = (live ? live[mtile] : mtile) * BM, n0 = (blockIdx.x % ntn) * BN;
  if (nb_dev) {  // see k_becp
    nb = min(nb, *nb_dev);
    if (n0 >= nb) return;
  }
  if (FORM == ZF_SYM && live == nullptr) {
    // Row tiles whose entries all belong to the other half of the sphere (minus = -1: most of the n1 = 0, n2 < 0 half plane, a
    // contiguous run in canonical order) would compute X, Y and store nothing: they retire here (or are not launched at all
    // when the host passes the list of live tiles).  cfg 4: 98 of 6 074 tiles, which takes the launch from 41.04 waves of
    // 148 CTAs to 40.4, i.e. one round less.
    const int r = m0 + (tid & (BM - 1));
    const bool dead = tid >= BM || r >= npw || minus[r] == -1;
    if (__syncthreads_and(dead)) return;
  }
  const int nkt = (nproj + BK - 1) / BK;
  const unsigned mb0 = mb_setup_tma<NSTAGE, NT>(mbar);
  const unsigned sm0 = static_cast<unsigned>(__cvta_generic_to_shared(sm));

  auto load_stage = [&](int kt, int st) {  // thread 0 only
    if (kt >= NSTAGE) mb_wait(mb0 + 8 * (NSTAGE + st), ((kt / NSTAGE) - 1) & 1);
    const unsigned full = mb0 + 8 * st;
    const unsigned dst = sm0 + (unsigned)(st * STAGE * 16);
    mb_expect_tx(full, STAGE * 16);
    tma_load_2d(dst, &tmA, 2 * m0, kt * BK, full);
#pragma unroll
    for (int q = 0; q < KSTEPS; ++q) tma_load_2d(dst + (unsigned)(BK * LDA * 16 + q * BN * 64), &tmB, 2 * (kt * BK + 4 * q), n0, full);
  };

  double P[TM][TN][2], Q[TM][TN][2], R[TM][TN][2];  // R: ZF_3M only
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j)
#pragma unroll
      for (int e = 0; e < 2; ++e) P[i][j][e] = Q[i][j][e] = R[i][j][e] = 0.0;
  if (tid == 0)
    for (int s = 0; s < Cfg::DIST; ++s)
      if (s < nkt) load_stage(s, s);
  const int fr = lane >> 2, fk = lane & 3;
  int st_c = 0, st_l = Cfg::DIST;
  for (int kt = 0; kt < nkt; ++kt) {
    mb_wait(mb0 + 8 * st_c, (kt / NSTAGE) & 1);
    const double2* As = sm + st_c * STAGE;
    const double2* Bs = As + BK * LDA;
    double2 af[2][TM], bf[2][TN];
    unsigned cm = 0;
    if constexpr (FORM == ZF_SYM) cm = __ldg(&cmask[kt]);
#pragma unroll
    for (int i = 0; i < TM; ++i) af[0][i] = As[fk * LDA + wm0 + i * 8 + fr];
#pragma unroll
    for (int j = 0; j < TN; ++j) bf[0][j] = Bs[(wn0 + j * 8 + fr) * 4 + fk];
#pragma unroll
    for (int kk = 0; kk < KSTEPS; ++kk) {
      if (kk + 1 < KSTEPS) {
#pragma unroll
        for (int i = 0; i < TM; ++i) af[(kk + 1) & 1][i] = As[((kk + 1) * 4 + fk) * LDA + wm0 + i * 8 + fr];
#pragma unroll
        for (int j = 0; j < TN; ++j) bf[(kk + 1) & 1][j] = Bs[(kk + 1) * BN * 4 + (wn0 + j * 8 + fr) * 4 + fk];
      }
      if constexpr (FORM == ZF_SYM) {
        // projector kt*BK + kk*4 + fk of class 1: i*beta = (-a_i, a_r); fragment swapped, sign in the B operand (e, -e)
        if ((cm >> (kk * 4 + fk)) & 1u) {
#pragma unroll
          for (int i = 0; i < TM; ++i) af[kk & 1][i] = make_double2(af[kk & 1][i].y, af[kk & 1][i].x);
        }
#pragma unroll
        for (int i = 0; i < TM; ++i)
#pragma unroll
          for (int j = 0; j < TN; ++j) dmma884(P[i][j][0], P[i][j][1], af[kk & 1][i].x, bf[kk & 1][j].y);
#pragma unroll
        for (int i = 0; i < TM; ++i)
#pragma unroll
          for (int j = 0; j < TN; ++j) dmma884(Q[i][j][0], Q[i][j][1], af[kk & 1][i].y, bf[kk & 1][j].x);
      } else if constexpr (FORM == ZF_GAMMA) {
        mma2r<TM, TN, false>(P, Q, af[kk & 1], bf[kk & 1]);
      } else {
        mma3m<TM, TN, false>(P, Q, R, af[kk & 1], bf[kk & 1]);
      }
      if (kk == 0 && tid == 0 && kt + Cfg::DIST < nkt) load_stage(kt + Cfg::DIST, st_l);
    }
    __syncwarp();
    if (lane == 0) mb_arrive(mb0 + 8 * (NSTAGE + st_c));
    st_c = (st_c + 1 == NSTAGE) ? 0 : st_c + 1;
    st_l = (st_l + 1 == NSTAGE) ? 0 : st_l + 1;
  }
  if constexpr (FORM == ZF_SYM) {
    // columns 2 fk, 2 fk + 1 of an 8-column block are (X, Y) of one band; loads of a row block before its stores (see k_vnl_add)
#pragma unroll
    for (int i = 0; i < TM; ++i) {
      const int gg = m0 + wm0 + i * 8 + fr;
      if (gg >= npw) continue;
      const int mg = minus[gg];
      if (mg == -1) continue;
      double2 v[TN], w[TN];
#pragma unroll
      for (int j = 0; j < TN; ++j) {
        const int col = n0 + wn0 + j * 8 + 2 * fk;
        v[j] = w[j] = make_double2(0.0, 0.0);
        if (col < nb) {
          v[j] = hpsi[(size_t)(col >> 1) * ldh + gg];
          if (mg >= 0) w[j] = hpsi[(size_t)(col >> 1) * ldh + mg];
        }
      }
#pragma unroll
      for (int j = 0; j < TN; ++j) {
        const int col = n0 + wn0 + j * 8 + 2 * fk;
        if (col >= nb) continue;
        const double xr = P[i][j][0], xi = Q[i][j][0], yr = P[i][j][1], yi = Q[i][j][1];
        hpsi[(size_t)(col >> 1) * ldh + gg] = make_double2(v[j].x + (xr - yi), v[j].y + (xi + yr));
        if (mg >= 0) hpsi[(size_t)(col >> 1) * ldh + mg] = make_double2(w[j].x + (xr + yi), w[j].y + (yr - xi));
      }
    }
  } else {
    // a b = (P - Q) + i (R - P - Q) (ZF_3M) or (P, Q) (ZF_GAMMA); loads of a row block before its stores (see k_vnl_add)
#pragma unroll
    for (int i = 0; i < TM; ++i) {
      const int gg = m0 + wm0 + i * 8 + fr;
      if (gg >= npw) continue;
      double2 v[TN][2];
#pragma unroll
      for (int j = 0; j < TN; ++j)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int b = n0 + wn0 + j * 8 + 2 * fk + e;
          v[j][e] = (b < nb && !overwrite) ? hpsi[(size_t)b * ldh + gg] : make_double2(0.0, 0.0);
        }
#pragma unroll
      for (int j = 0; j < TN; ++j)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int b = n0 + wn0 + j * 8 + 2 * fk + e;
          if (b >= nb) continue;
          double2 t = v[j][e];
          if constexpr (FORM == ZF_GAMMA) {
            t.x += P[i][j][e];
            t.y += Q[i][j][e];
          } else {
            t.x += P[i][j][e] - Q[i][j][e];
            t.y += (R[i][j][e] - P[i][j][e]) - Q[i][j][e];
          }
          hpsi[(size_t)b * ldh + gg] = t;
        }
    }
  }
}

}  // namespace qehpsi
