// zgemm_kernels.cuh -- the nonlocal (pseudopotential) term as FP64 tensor-core contractions (steps a6-a8 of
// DESIGN.md section 5; "pseudopotential ... contributions to the Hamiltonian", done with GEMM
// in the paper's port).
//   a6 k_becp     : partial[ks][p][b] = sum_{ig in K-slice ks} conj(beta[p][ig]) psi[b][ig]     (split-K ZGEMM)
//   a7 k_becp_reduce / k_dmul : becp = sum_ks partial (fixed order); dbecpT[b][p] = sum_j D^a_ij becp[a,j][b]
//   a8 k_vnl_add  : hpsi[b][ig] += sum_p beta[p][ig] dbecpT[b][p]                                 (ZGEMM)
// FP64 tensor math on sm_100a exists only as warp-level mma.sync (DMMA.8x8x4 in SASS; there is no tcgen05 /
// TMEM path for f64), so the tiles are fed by cp.async multi-stage pipelines into bank-conflict-free shared
// memory layouts.
//
// Complex product = "3M" (Karatsuba) form: with P = sum ar*br, Q = sum ai*bi, R = sum (ar+ai)*(br+bi),
//   sum a*b       = (P - Q) + i (R - P - Q)
//   sum conj(a)*b = (P + Q) + i (R' - P + Q),   R' = sum (ar-ai)*(br+bi)
// i.e. three real DMMAs per complex 8x8x4 block instead of four; the fragment sums cost one DADD per loaded
// element.  Normwise error stays O(eps*sqrt(K)) (tolerance).
#pragma once
#include <cuda_runtime.h>

namespace qehpsi {

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
      : "+d"(c0), "+d"(c1)
      : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, bool valid) {
  const unsigned s = static_cast<unsigned>(__cvta_generic_to_shared(smem));
  const int sz = valid ? 16 : 0;  // src-size 0 => 16 zero bytes are written, nothing is read
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gmem), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N));
}

// mbarrier pipeline of the DMMA kernels: every stage has a `full` barrier (all NT threads arrive through
// cp.async.mbarrier.arrive.noinc once their own copies of the stage have landed) and an `empty` barrier (one arrive per warp
// after its last fragment load of the stage).  No CTA-wide barrier in the K loop: a warp waits for DATA only, and may run up to
// NSTAGE - 2 tiles ahead of the slowest one (the refill of a stage is issued two tiles after the stage was consumed).  Against
// __syncthreads per tile: 0.83 -> 0.90 of the DMMA peak on the symmetric a8 kernel, same bits (profiles/r2j_dmma_pipeline.md).
__device__ __forceinline__ void mb_init(unsigned bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mb_wait(unsigned bar, unsigned parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tMBW_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@!p bra MBW_%=;\n\t}" ::"r"(bar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void mb_arrive(unsigned bar) {
  asm volatile("{\n\t.reg .b64 t;\n\tmbarrier.arrive.shared::cta.b64 t, [%0];\n\t}" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mb_cp_arrive(unsigned bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}
// full[s] at mb0 + 8 s, empty[s] at mb0 + 8 (NSTAGE + s); ends with a CTA barrier
template <int NSTAGE, int NT>
__device__ __forceinline__ unsigned mb_setup(unsigned long long* mbar) {
  const unsigned mb0 = static_cast<unsigned>(__cvta_generic_to_shared(mbar));
  if (threadIdx.x == 0) {
    for (int s = 0; s < NSTAGE; ++s) {
      mb_init(mb0 + 8 * s, NT);
      mb_init(mb0 + 8 * (NSTAGE + s), NT / 32);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  return mb0;
}

// K-contiguous operand tile: rows of BK complex; 16-byte column kc of odd rows is XOR-ed with 4 so that a
// fragment load (quarter warp = 2 rows x 4 k) touches 8 distinct 16-byte bank groups.
template <int BK>
__device__ __forceinline__ int swz_k(int row, int kc) {
  return row * BK + (kc ^ ((row & 1) << 2));
}

template <int BM_, int BN_, int WM_, int WN_, int BK_, int NSTAGE_>
struct ZgCfg {
  static constexpr int BM = BM_, BN = BN_, WM = WM_, WN = WN_, BK = BK_, NSTAGE = NSTAGE_;
  static constexpr int NT = WM * WN * 32;
  static constexpr int TM = BM / WM / 8;  // 8-row blocks per warp along M
  static constexpr int TN = BN / WN / 8;
  static constexpr int KSTEPS = BK / 4;
  static constexpr int LDA_M = BM + 2;  // row stride of an M-contiguous [k][m] tile: (2k + m) mod 8 distinct per quarter warp
  static constexpr size_t SMEM_BECP = (size_t)NSTAGE * (BM + BN) * BK * sizeof(double2);
  static constexpr size_t SMEM_VNL = (size_t)NSTAGE * (BK * LDA_M + BN * BK) * sizeof(double2);
  static constexpr int DIST = NSTAGE - 2;  // tiles in flight ahead of the one being consumed (mbarrier pipeline above)
  static_assert(BM % (WM * 8) == 0 && BN % (WN * 8) == 0 && BK % 4 == 0 && BK >= 8 && NSTAGE >= 3, "tile shape");
};

// one k4 step of the 3M product on a TM x TN grid of 8x8 blocks
template <int TM, int TN, bool CONJ_A>
__device__ __forceinline__ void mma3m(double (&P)[TM][TN][2], double (&Q)[TM][TN][2], double (&R)[TM][TN][2],
                                      const double2 (&af)[TM], const double2 (&bf)[TN]) {
  double as[TM], bs[TN];
#pragma unroll
  for (int i = 0; i < TM; ++i) as[i] = CONJ_A ? af[i].x - af[i].y : af[i].x + af[i].y;
#pragma unroll
  for (int j = 0; j < TN; ++j) bs[j] = bf[j].x + bf[j].y;
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) dmma884(P[i][j][0], P[i][j][1], af[i].x, bf[j].x);
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) dmma884(Q[i][j][0], Q[i][j][1], af[i].y, bf[j].y);
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) dmma884(R[i][j][0], R[i][j][1], as[i], bs[j]);
}

// Gamma-only variants (NEXT-1: real wavefunctions, c(-G) = conj c(G), half sphere).  A complex element is read as
// two consecutive reals, so the contraction over the 2*ngw real components needs two real DMMAs per block:
//   becp (real)  : sum_k (ar*br + ai*bi)            -> P += ar*br, Q += ai*bi, result P + Q
//   vnl_add      : out.re += sum_p ar*d, out.im += sum_p ai*d with real d = B.re -> P += ar*br, Q += ai*br
template <int TM, int TN, bool B_IMAG>
__device__ __forceinline__ void mma2r(double (&P)[TM][TN][2], double (&Q)[TM][TN][2], const double2 (&af)[TM],
                                      const double2 (&bf)[TN]) {
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) dmma884(P[i][j][0], P[i][j][1], af[i].x, bf[j].x);
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) dmma884(Q[i][j][0], Q[i][j][1], af[i].y, B_IMAG ? bf[j].y : bf[j].x);
}

// a6 ------------------------------------------------------------------------------------------------------
// C[p][b] = sum_k conj(A[p][k]) B[b][k] over k in [ks*kchunk, min(npw,(ks+1)*kchunk)); A = beta, B = psi.
template <class Cfg, bool GAMMA = false>
__global__ void __launch_bounds__(Cfg::NT, 1)
    k_becp(const double2* __restrict__ beta, long long ldb, int nproj, const double2* __restrict__ psi, long long ldpsi,
           int nb, int npw, int kchunk, double2* __restrict__ partial, int ldc, const int* __restrict__ nb_dev = nullptr,
           const unsigned char* __restrict__ cls = nullptr) {
  constexpr int BM = Cfg::BM, BN = Cfg::BN, WM = Cfg::WM, WN = Cfg::WN, BK = Cfg::BK, NSTAGE = Cfg::NSTAGE;
  constexpr int NT = Cfg::NT, TM = Cfg::TM, TN = Cfg::TN, KSTEPS = Cfg::KSTEPS;
  constexpr int STAGE = (BM + BN) * BK;  // complex elements per stage
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* sm = reinterpret_cast<double2*>(smem_raw);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm0 = (warp / WN) * (BM / WM), wn0 = (warp % WN) * (BN / WN);
  const int ntn = (nb + BN - 1) / BN;  // the grid was sized for the host-side nb
  const int m0 = (blockIdx.x / ntn) * BM, n0 = (blockIdx.x % ntn) * BN;
  // nb_dev (QE_HPSI_PROJ_CERTIFY): the number of bands to process is decided on the device; tiles beyond it retire at once
  if (nb_dev) {
    nb = min(nb, *nb_dev);
    if (n0 >= nb) return;
  }
  __shared__ __align__(8) unsigned long long mbar[2 * NSTAGE];
  const unsigned mb0 = mb_setup<NSTAGE, NT>(mbar);
  const int ks = blockIdx.y;
  const int kb = ks * kchunk, ke = min(npw, kb + kchunk);
  const int nkt = (ke - kb + BK - 1) / BK;

  // Per-thread copy plan, fixed for the whole K loop: thread owns 16-byte column kc of rows r0, r0+RPT, ...
  // (A rows first, then B rows); only the k offset advances, so a stage costs one compare plus the cp.asyncs.
  constexpr int RPT = NT / BK, NA = BM / RPT, NB = BN / RPT;
  static_assert(NT % BK == 0 && BM % RPT == 0 && BN % RPT == 0 && RPT % 2 == 0, "copy plan");
  const int ckc = tid % BK, cr0 = tid / BK;
  const double2* asrc[NA];
  const double2* bsrc[NB];
  unsigned rowok = 0;
#pragma unroll
  for (int n = 0; n < NA; ++n) {
    const int p = m0 + cr0 + n * RPT;
    const bool ok = p < nproj;
    rowok |= ok ? (1u << n) : 0u;
    asrc[n] = beta + (size_t)(ok ? p : 0) * ldb + kb + ckc;
  }
#pragma unroll
  for (int n = 0; n < NB; ++n) {
    const int b = n0 + cr0 + n * RPT;
    const bool ok = b < nb;
    rowok |= ok ? (1u << (NA + n)) : 0u;
    bsrc[n] = psi + (size_t)(ok ? b : 0) * ldpsi + kb + ckc;
  }
  const unsigned cdst = static_cast<unsigned>(__cvta_generic_to_shared(sm + swz_k<BK>(cr0, ckc)));
  auto load_stage = [&](int kt, int st) {
    if (kt >= NSTAGE) mb_wait(mb0 + 8 * (NSTAGE + st), ((kt / NSTAGE) - 1) & 1);  // every warp is done with the stage's last tile
    const int koff = kt * BK;
    const bool kok = (kb + koff + ckc) < ke;
    const unsigned d0 = cdst + (unsigned)(st * STAGE * (int)sizeof(double2));
#pragma unroll
    for (int n = 0; n < NA; ++n) {
      const int sz = (kok && ((rowok >> n) & 1u)) ? 16 : 0;
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d0 + (unsigned)(n * RPT * BK * 16)),
                   "l"(asrc[n] + koff), "r"(sz));
    }
#pragma unroll
    for (int n = 0; n < NB; ++n) {
      const int sz = (kok && ((rowok >> (NA + n)) & 1u)) ? 16 : 0;
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d0 + (unsigned)((BM + n * RPT) * BK * 16)),
                   "l"(bsrc[n] + koff), "r"(sz));
    }
    mb_cp_arrive(mb0 + 8 * st);
  };

  double P[TM][TN][2], Q[TM][TN][2], R[TM][TN][2];
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j)
#pragma unroll
      for (int e = 0; e < 2; ++e) P[i][j][e] = Q[i][j][e] = R[i][j][e] = 0.0;

#pragma unroll
  for (int s = 0; s < Cfg::DIST; ++s)
    if (s < nkt) load_stage(s, s);
  const int fr = lane >> 2, fk = lane & 3;
  // Gamma-symmetric projector mode (cls != nullptr, GAMMA form): rows of class 1 (beta(-G) = -conj beta(G)) enter as i*beta =
  // (-a_i, a_r), so that every row is Hermitian and the real form applies; the fragment is only swapped to (a_i, a_r) and the
  // sign goes into the epilogue (Q - P instead of P + Q): no FP64 instruction is spent on it
  bool swp[TM];
#pragma unroll
  for (int i = 0; i < TM; ++i) {
    const int p = m0 + wm0 + i * 8 + fr;
    swp[i] = GAMMA && cls != nullptr && p < nproj && cls[p] != 0;
  }
  int st_c = 0, st_l = Cfg::DIST;  // stage being consumed / stage being refilled
  for (int kt = 0; kt < nkt; ++kt) {
    mb_wait(mb0 + 8 * st_c, (kt / NSTAGE) & 1);  // the tile has landed (copies of all threads)
    const double2* As = sm + st_c * STAGE;
    const double2* Bs = As + BM * BK;
    double2 af[2][TM], bf[2][TN];
#pragma unroll
    for (int i = 0; i < TM; ++i) af[0][i] = As[swz_k<BK>(wm0 + i * 8 + fr, fk)];
#pragma unroll
    for (int j = 0; j < TN; ++j) bf[0][j] = Bs[swz_k<BK>(wn0 + j * 8 + fr, fk)];
#pragma unroll
    for (int kk = 0; kk < KSTEPS; ++kk) {
      if (kk + 1 < KSTEPS) {
#pragma unroll
        for (int i = 0; i < TM; ++i) af[(kk + 1) & 1][i] = As[swz_k<BK>(wm0 + i * 8 + fr, (kk + 1) * 4 + fk)];
#pragma unroll
        for (int j = 0; j < TN; ++j) bf[(kk + 1) & 1][j] = Bs[swz_k<BK>(wn0 + j * 8 + fr, (kk + 1) * 4 + fk)];
      }
      if constexpr (GAMMA) {
#pragma unroll
        for (int i = 0; i < TM; ++i)
          if (swp[i]) af[kk & 1][i] = make_double2(af[kk & 1][i].y, af[kk & 1][i].x);  // (a_i, a_r): P = sum a_i b_r, Q = sum a_r b_i
        mma2r<TM, TN, true>(P, Q, af[kk & 1], bf[kk & 1]);
      } else
        mma3m<TM, TN, true>(P, Q, R, af[kk & 1], bf[kk & 1]);
      if (kk == 0) {  // refill the stage consumed two tiles ago, behind the first batch of DMMAs
        if (kt + Cfg::DIST < nkt) load_stage(kt + Cfg::DIST, st_l);
      }
    }
    __syncwarp();
    if (lane == 0) mb_arrive(mb0 + 8 * (NSTAGE + st_c));  // this warp has read the stage
    st_c = (st_c + 1 == NSTAGE) ? 0 : st_c + 1;
    st_l = (st_l + 1 == NSTAGE) ? 0 : st_l + 1;
  }
  // C fragment: row = lane/4, columns 2*(lane%4) + {0,1};  conj(a) b = (P + Q) + i (R - P + Q)
  double2* out = partial + (size_t)ks * nproj * ldc;
#pragma unroll
  for (int i = 0; i < TM; ++i) {
    const int p = m0 + wm0 + i * 8 + fr;
    if (p >= nproj) continue;
#pragma unroll
    for (int j = 0; j < TN; ++j) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int b = n0 + wn0 + j * 8 + 2 * fk + e;
        if (b < nb)
          out[(size_t)p * ldc + b] = GAMMA ? make_double2(swp[i] ? Q[i][j][e] - P[i][j][e] : P[i][j][e] + Q[i][j][e], 0.0)
                                           : make_double2(P[i][j][e] + Q[i][j][e], (R[i][j][e] - P[i][j][e]) + Q[i][j][e]);
      }
    }
  }
}

// a7 ------------------------------------------------------------------------------------------------------
// becp[p][b] = sum_ks partial[ks][p][b], ks ascending (deterministic, independent of the batch composition)
__global__ void k_becp_reduce(const double2* __restrict__ partial, int nsplit, int nproj, int ldc, int nb,
                              double2* __restrict__ becp, const int* __restrict__ nb_dev = nullptr) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  const int p = blockIdx.y;
  if (nb_dev) nb = min(nb, *nb_dev);
  if (b >= nb) return;
  double re = 0.0, im = 0.0;
  for (int ks = 0; ks < nsplit; ++ks) {
    const double2 v = partial[((size_t)ks * nproj + p) * ldc + b];
    re += v.x;
    im += v.y;
  }
  becp[(size_t)p * ldc + b] = make_double2(re, im);
}
// Gamma-only a7: becp[p][b] = 2 * sum_ks partial[ks][p][b].re - beta[p][0].re * psi[b][0].re  (the G = 0 term of the
// half sphere must count once, not twice; real result stored as (re, 0))
__global__ void k_becp_reduce_gamma(const double2* __restrict__ partial, int nsplit, int nproj, int ldc, int nb,
                                    const double2* __restrict__ beta, long long ldb, const double2* __restrict__ psi,
                                    long long ldpsi, double2* __restrict__ becp) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  const int p = blockIdx.y;
  if (b >= nb) return;
  double re = 0.0;
  for (int ks = 0; ks < nsplit; ++ks) re += partial[((size_t)ks * nproj + p) * ldc + b].x;
  const double2 b0 = beta[(size_t)p * ldb], c0 = psi[(size_t)b * ldpsi];
  becp[(size_t)p * ldc + b] = make_double2(2.0 * re - (b0.x * c0.x + b0.y * c0.y), 0.0);
}
// NEXT-3 (Davidson step): preconditioner diagonals and the preconditioner itself.
// diag[g] = base[g] (or 1) + shift + sum_p w[p] |beta[p][g]|^2, w[p] = diagonal entry of projector p's D (or q) block
__global__ void k_proj_diag(const double2* __restrict__ beta, long long ldb, int nproj, int npw,
                            const long long* __restrict__ proj_doff, const int* __restrict__ proj_blk0,
                            const int* __restrict__ proj_nh, const double* __restrict__ dpk,
                            const double* __restrict__ base, double shift, double* __restrict__ out) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= npw) return;
  double acc = 0.0;
  for (int p = 0; p < nproj; ++p) {
    const double w = __ldg(&dpk[proj_doff[p] + (p - proj_blk0[p])]);  // row (p - q0), column (p - q0) of the block
    const double2 b = beta[(size_t)p * ldb + g];
    acc += w * (b.x * b.x + b.y * b.y);
  }
  out[g] = (base ? base[g] : 1.0) + shift + acc;
}
// r[b][g] /= (1 + x + sqrt(1 + (x-1)^2)) / 2,  x = hdiag[g] - e[b] * sdiag[g]  (sdiag == nullptr: 1)
__global__ void k_precond(double2* __restrict__ r, long long ldr, int nb, int npw, const double* __restrict__ e,
                          const double* __restrict__ hdiag, const double* __restrict__ sdiag) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  const int b = blockIdx.y;
  if (g >= npw) return;
  const double x = hdiag[g] - e[b] * (sdiag ? sdiag[g] : 1.0);
  const double den = 0.5 * (1.0 + x + sqrt(1.0 + (x - 1.0) * (x - 1.0)));
  double2 v = r[(size_t)b * ldr + g];
  r[(size_t)b * ldr + g] = make_double2(v.x / den, v.y / den);
}
// NEXT-3 (reduced matrices <a_i|b_j>): out[i][j] = sum_ks partial[ks][i][j], ks ascending, with its own row stride
__global__ void k_ovl_reduce(const double2* __restrict__ partial, int nsplit, int na, int ldc, int nb,
                             double2* __restrict__ out, long long ldo) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  const int p = blockIdx.y;
  if (b >= nb) return;
  double re = 0.0, im = 0.0;
  for (int ks = 0; ks < nsplit; ++ks) {
    const double2 v = partial[((size_t)ks * na + p) * ldc + b];
    re += v.x;
    im += v.y;
  }
  out[(size_t)p * ldo + b] = make_double2(re, im);
}
// dbecp[p][b] = sum_j D[p][j] becp[blk_start(p)+j][b]; written both as dbecp[p][b] and transposed dbT[b][p]
__global__ void k_dmul(const double2* __restrict__ becp, int nproj, int ldc, int nb, const int* __restrict__ proj_blk0,
                       const int* __restrict__ proj_nh, const long long* __restrict__ proj_doff,
                       const double* __restrict__ dpk, double2* __restrict__ dbecp, double2* __restrict__ dbT, int ldp,
                       const int* __restrict__ nb_dev = nullptr) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  const int p = blockIdx.y;
  if (nb_dev) nb = min(nb, *nb_dev);
  if (b >= nb) return;
  const int q0 = proj_blk0[p], nh = proj_nh[p];
  const double* drow = dpk + proj_doff[p];  // row (p - q0) of the block
  double re = 0.0, im = 0.0;
  for (int j = 0; j < nh; ++j) {
    const double d = __ldg(&drow[j]);
    const double2 v = becp[(size_t)(q0 + j) * ldc + b];
    re += d * v.x;
    im += d * v.y;
  }
  dbecp[(size_t)p * ldc + b] = make_double2(re, im);
  dbT[(size_t)b * ldp + p] = make_double2(re, im);
}

// a8 ------------------------------------------------------------------------------------------------------
// hpsi[b][g] += sum_p A[p][g] B[b][p];  A = beta ([p][g], g contiguous: "M-major"), B = dbT ([b][p], p contiguous)
// SYM (Gamma-symmetric projector mode of a complex handle; needs GAMMA): rows g run over the leading
// `npw` = M sphere entries (n1 >= 0), columns come in pairs (2b, 2b+1) = real coefficient vectors (Re e, Im e) of band b, rows p of
// class 1 enter as i*beta; with X, Y the two complex sums of a pair the epilogue adds X + iY to hpsi[b][g] and conj(X) + i conj(Y)
// to hpsi[b][minus[g]] (minus[g] = position of -G; -1: g is not in the half sphere, skip; -2: G = 0, no partner).
template <class Cfg, bool GAMMA = false, bool SYM = false>
__global__ void __launch_bounds__(Cfg::NT, 1)
    k_vnl_add(const double2* __restrict__ beta, long long ldb, int nproj, int npw, const double2* __restrict__ dbT,
              int ldp, int nb, double2* __restrict__ hpsi, long long ldh, const int* __restrict__ nb_dev = nullptr,
              const unsigned* __restrict__ cmask = nullptr, const int* __restrict__ minus = nullptr, int overwrite = 0) {
  // overwrite != 0 (general form only; qe_hpsi_rotate without accumulation): hpsi = product, nothing is read in the epilogue
  static_assert(!SYM || GAMMA, "the symmetric mode is a real form");
  static_assert(!SYM || Cfg::BK == 16, "cmask holds one 16-bit class mask per K tile of 16 projectors");
  constexpr int BM = Cfg::BM, BN = Cfg::BN, WM = Cfg::WM, WN = Cfg::WN, BK = Cfg::BK, NSTAGE = Cfg::NSTAGE;
  constexpr int NT = Cfg::NT, TM = Cfg::TM, TN = Cfg::TN, KSTEPS = Cfg::KSTEPS, LDA = Cfg::LDA_M;
  constexpr int STAGE = BK * LDA + BN * BK;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* sm = reinterpret_cast<double2*>(smem_raw);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm0 = (warp / WN) * (BM / WM), wn0 = (warp % WN) * (BN / WN);
  const int ntn = (nb + BN - 1) / BN;
  const int m0 = (blockIdx.x / ntn) * BM, n0 = (blockIdx.x % ntn) * BN;
  if (nb_dev) {  // see k_becp
    nb = min(nb, *nb_dev);
    if (n0 >= nb) return;
  }
  if constexpr (SYM) {  // row tiles with nothing to store retire at once (see k_vnl_tma)
    const int r = m0 + (tid & (BM - 1));
    const bool dead = tid >= BM || r >= npw || minus[r] == -1;
    if (__syncthreads_and(dead)) return;
  }
  const int nkt = (nproj + BK - 1) / BK;
  __shared__ __align__(8) unsigned long long mbar[2 * NSTAGE];
  const unsigned mb0 = mb_setup<NSTAGE, NT>(mbar);

  // Per-thread copy plan (see k_becp).  A tile [BK][LDA]: thread owns column gc of rows ra, ra+RPA, ...; B tile
  // [BN][BK]: column ckc of rows cr0, cr0+RPT, ...
  constexpr int RPA = NT / BM, NA = BK / RPA, RPT = NT / BK, NB = BN / RPT;
  static_assert(NT % BM == 0 && BK % RPA == 0 && NT % BK == 0 && BN % RPT == 0 && RPT % 2 == 0, "copy plan");
  const int gc = tid % BM, ra = tid / BM;
  const bool gok = (m0 + gc) < npw;
  const double2* asrc = beta + (size_t)ra * ldb + (gok ? m0 + gc : 0);
  const size_t astep = (size_t)RPA * ldb;
  const unsigned adst = static_cast<unsigned>(__cvta_generic_to_shared(sm + ra * LDA + gc));
  const int ckc = tid % BK, cr0 = tid / BK;
  const double2* bsrc[NB];
  unsigned rowok = 0;
#pragma unroll
  for (int n = 0; n < NB; ++n) {
    const int b = n0 + cr0 + n * RPT;
    const bool ok = b < nb;
    rowok |= ok ? (1u << n) : 0u;
    bsrc[n] = dbT + (size_t)(ok ? b : 0) * ldp + ckc;
  }
  const unsigned bdst = static_cast<unsigned>(__cvta_generic_to_shared(sm + BK * LDA + swz_k<BK>(cr0, ckc)));
  auto load_stage = [&](int kt, int st) {
    if (kt >= NSTAGE) mb_wait(mb0 + 8 * (NSTAGE + st), ((kt / NSTAGE) - 1) & 1);  // every warp is done with the stage's last tile
    const int k0 = kt * BK;
    const unsigned soff = (unsigned)(st * STAGE * (int)sizeof(double2));
    const double2* ap = asrc + (size_t)k0 * ldb;
#pragma unroll
    for (int n = 0; n < NA; ++n) {
      const bool ok = gok && (k0 + ra + n * RPA) < nproj;
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(adst + soff + (unsigned)(n * RPA * LDA * 16)),
                   "l"(ok ? ap : beta), "r"(ok ? 16 : 0));
      ap += astep;
    }
    const bool kok = (k0 + ckc) < nproj;
#pragma unroll
    for (int n = 0; n < NB; ++n) {
      const int sz = (kok && ((rowok >> n) & 1u)) ? 16 : 0;
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(bdst + soff + (unsigned)(n * RPT * BK * 16)),
                   "l"(bsrc[n] + k0), "r"(sz));
    }
    mb_cp_arrive(mb0 + 8 * st);
  };

  double P[TM][TN][2], Q[TM][TN][2], R[TM][TN][2];
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j)
#pragma unroll
      for (int e = 0; e < 2; ++e) P[i][j][e] = Q[i][j][e] = R[i][j][e] = 0.0;

#pragma unroll
  for (int s = 0; s < Cfg::DIST; ++s)
    if (s < nkt) load_stage(s, s);
  const int fr = lane >> 2, fk = lane & 3;
  int st_c = 0, st_l = Cfg::DIST;  // stage being consumed / stage being refilled
  for (int kt = 0; kt < nkt; ++kt) {
    mb_wait(mb0 + 8 * st_c, (kt / NSTAGE) & 1);  // the tile has landed (copies of all threads)
    const double2* As = sm + st_c * STAGE;
    const double2* Bs = As + BK * LDA;
    double2 af[2][TM], bf[2][TN];
    unsigned cm = 0;
    if constexpr (SYM) cm = __ldg(&cmask[kt]);
#pragma unroll
    for (int i = 0; i < TM; ++i) af[0][i] = As[fk * LDA + wm0 + i * 8 + fr];
#pragma unroll
    for (int j = 0; j < TN; ++j) bf[0][j] = Bs[swz_k<BK>(wn0 + j * 8 + fr, fk)];
#pragma unroll
    for (int kk = 0; kk < KSTEPS; ++kk) {
      if (kk + 1 < KSTEPS) {
#pragma unroll
        for (int i = 0; i < TM; ++i) af[(kk + 1) & 1][i] = As[((kk + 1) * 4 + fk) * LDA + wm0 + i * 8 + fr];
#pragma unroll
        for (int j = 0; j < TN; ++j) bf[(kk + 1) & 1][j] = Bs[swz_k<BK>(wn0 + j * 8 + fr, (kk + 1) * 4 + fk)];
      }
      if constexpr (GAMMA) {
        if constexpr (SYM) {  // the k row of this fragment is projector kt*BK + kk*4 + fk: bit kk*4 + fk of the tile's class mask
          // class 1: i*beta = (-a_i, a_r); the fragment is swapped to (a_i, a_r) and the sign sits in the B operand, whose rows
          // hold (e, e) for class 0 and (e, -e) for class 1 projectors (k_sym_coef): P += a'.x * b.y, Q += a'.y * b.x
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
        } else
          mma2r<TM, TN, false>(P, Q, af[kk & 1], bf[kk & 1]);
      } else
        mma3m<TM, TN, false>(P, Q, R, af[kk & 1], bf[kk & 1]);
      if (kk == 0) {  // refill the stage consumed two tiles ago, behind the first batch of DMMAs
        if (kt + Cfg::DIST < nkt) load_stage(kt + Cfg::DIST, st_l);
      }
    }
    __syncwarp();
    if (lane == 0) mb_arrive(mb0 + 8 * (NSTAGE + st_c));  // this warp has read the stage
    st_c = (st_c + 1 == NSTAGE) ? 0 : st_c + 1;
    st_l = (st_l + 1 == NSTAGE) ? 0 : st_l + 1;
  }
  if constexpr (SYM) {
    // columns 2 fk, 2 fk + 1 of an 8-column block are (X, Y) of one band: X = (P, Q)[0], Y = (P, Q)[1].
    // All loads of a row block are issued before its first store: the compiler cannot prove that hpsi[.][g] and hpsi[.][-g] do
    // not alias, so interleaved read-modify-writes would serialise into one global round trip per entry.
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
        if (col < nb) {  // nb = number of columns = 2 x bands
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
    // a b = (P - Q) + i (R - P - Q); loads of a row block before its stores (see above)
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
          if (b < nb) {
            double2 t = v[j][e];
            if constexpr (GAMMA) {
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
}

}  // namespace qehpsi
