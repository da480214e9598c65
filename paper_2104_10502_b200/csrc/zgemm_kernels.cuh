// zgemm_kernels.cuh -- the nonlocal (pseudopotential) term as FP64 tensor-core contractions (steps a6-a8 of
// DESIGN.md section 2; "pseudopotential ... contributions to the Hamiltonian", done with GEMM
// in the paper's port).
//   a6 k_becp     : partial[ks][p][b] = sum_{ig in K-slice ks} conj(beta[p][ig]) psi[b][ig]     (split-K ZGEMM)
//   a7 k_becp_reduce / k_dmul : becp = sum_ks partial (fixed order); dbecpT[b][p] = sum_j D^a_ij becp[a,j][b]
//   a8 k_vnl_add  : hpsi[b][ig] += sum_p beta[p][ig] dbecpT[b][p]                                 (ZGEMM)
// FP64 tensor math on sm_100a exists only as warp-level mma.sync (DMMA.8x8x4 in SASS; there is no tcgen05 /
// TMEM path for f64), so the tiles are fed by cp.async multi-stage pipelines into bank-conflict-free shared
// memory layouts and each warp owns a 32x32 complex accumulator tile (4 real DMMAs per complex 8x8x4 block).
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

constexpr int ZG_BK = 8;  // complex k per pipeline stage (two DMMA k-steps)

// rows of 8 complex (128 B), K contiguous; the two 64-byte halves of odd rows are swapped so that the fragment
// load (8 lanes = 2 rows x 4 k) touches 8 distinct 16-byte bank groups.
__device__ __forceinline__ int swz_k8(int row, int kc) { return row * 8 + (kc ^ ((row & 1) << 2)); }

template <int BM, int BN, int WM, int WN, int NSTAGE>
struct ZgCfg {
  static constexpr int NT = WM * WN * 32;
  static constexpr int TM = BM / WM / 8;  // 8-row blocks per warp along M
  static constexpr int TN = BN / WN / 8;
  static_assert(BM % (WM * 8) == 0 && BN % (WN * 8) == 0, "tile shape");
};

// a6 ------------------------------------------------------------------------------------------------------
// C[p][b] = sum_k conj(A[p][k]) B[b][k] over k in [ks*kchunk, min(npw,(ks+1)*kchunk)); A = beta, B = psi.
template <int BM, int BN, int WM, int WN, int NSTAGE>
__global__ void __launch_bounds__(WM* WN * 32, 1)
    k_becp(const double2* __restrict__ beta, long long ldb, int nproj, const double2* __restrict__ psi, long long ldpsi,
           int nb, int npw, int kchunk, double2* __restrict__ partial, int ldc) {
  using Cfg = ZgCfg<BM, BN, WM, WN, NSTAGE>;
  constexpr int NT = Cfg::NT, TM = Cfg::TM, TN = Cfg::TN;
  constexpr int STAGE = (BM + BN) * ZG_BK;  // complex elements per stage
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double2* sm = reinterpret_cast<double2*>(smem_raw);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm0 = (warp / WN) * (BM / WM), wn0 = (warp % WN) * (BN / WN);
  const int ntn = (nb + BN - 1) / BN;
  const int m0 = (blockIdx.x / ntn) * BM, n0 = (blockIdx.x % ntn) * BN;
  const int ks = blockIdx.y;
  const int kb = ks * kchunk, ke = min(npw, kb + kchunk);
  const int nkt = (ke - kb + ZG_BK - 1) / ZG_BK;

  auto load_stage = [&](int kt, int st) {
    double2* As = sm + st * STAGE;
    double2* Bs = As + BM * ZG_BK;
    const int k0 = kb + kt * ZG_BK;
    for (int id = tid; id < (BM + BN) * ZG_BK; id += NT) {
      const int kc = id & 7;
      const int r = id >> 3;
      const bool kok = (k0 + kc) < ke;
      if (r < BM) {
        const int p = m0 + r;
        const bool ok = kok && p < nproj;
        cp_async16(&As[swz_k8(r, kc)], ok ? &beta[(size_t)p * ldb + k0 + kc] : beta, ok);
      } else {
        const int rb = r - BM, b = n0 + rb;
        const bool ok = kok && b < nb;
        cp_async16(&Bs[swz_k8(rb, kc)], ok ? &psi[(size_t)b * ldpsi + k0 + kc] : psi, ok);
      }
    }
  };

  double cre[TM][TN][2], cim[TM][TN][2];
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) cre[i][j][0] = cre[i][j][1] = cim[i][j][0] = cim[i][j][1] = 0.0;

#pragma unroll
  for (int s = 0; s < NSTAGE - 1; ++s) {
    if (s < nkt) load_stage(s, s);
    cp_async_commit();
  }
  const int fr = lane >> 2, fk = lane & 3;
  for (int kt = 0; kt < nkt; ++kt) {
    cp_async_wait<NSTAGE - 2>();
    __syncthreads();
    if (kt + NSTAGE - 1 < nkt) load_stage(kt + NSTAGE - 1, (kt + NSTAGE - 1) % NSTAGE);
    cp_async_commit();
    const double2* As = sm + (kt % NSTAGE) * STAGE;
    const double2* Bs = As + BM * ZG_BK;
#pragma unroll
    for (int kk = 0; kk < 2; ++kk) {
      double2 af[TM], bf[TN];
#pragma unroll
      for (int i = 0; i < TM; ++i) af[i] = As[swz_k8(wm0 + i * 8 + fr, kk * 4 + fk)];
#pragma unroll
      for (int j = 0; j < TN; ++j) bf[j] = Bs[swz_k8(wn0 + j * 8 + fr, kk * 4 + fk)];
#pragma unroll
      for (int i = 0; i < TM; ++i) {
        const double ar = af[i].x, ai = af[i].y, nai = -af[i].y;
#pragma unroll
        for (int j = 0; j < TN; ++j) {
          // conj(a) b = (ar br + ai bi) + i (ar bi - ai br)
          dmma884(cre[i][j][0], cre[i][j][1], ar, bf[j].x);
          dmma884(cim[i][j][0], cim[i][j][1], ar, bf[j].y);
          dmma884(cre[i][j][0], cre[i][j][1], ai, bf[j].y);
          dmma884(cim[i][j][0], cim[i][j][1], nai, bf[j].x);
        }
      }
    }
  }
  cp_async_wait<0>();
  // C fragment: row = lane/4, columns 2*(lane%4) + {0,1}
  double2* out = partial + (size_t)ks * nproj * ldc;
#pragma unroll
  for (int i = 0; i < TM; ++i) {
    const int p = m0 + wm0 + i * 8 + fr;
    if (p >= nproj) continue;
#pragma unroll
    for (int j = 0; j < TN; ++j) {
      const int b = n0 + wn0 + j * 8 + 2 * fk;
      if (b < nb) out[(size_t)p * ldc + b] = make_double2(cre[i][j][0], cim[i][j][0]);
      if (b + 1 < nb) out[(size_t)p * ldc + b + 1] = make_double2(cre[i][j][1], cim[i][j][1]);
    }
  }
}

// a7 ------------------------------------------------------------------------------------------------------
// becp[p][b] = sum_ks partial[ks][p][b], ks ascending (deterministic, independent of the batch composition)
__global__ void k_becp_reduce(const double2* __restrict__ partial, int nsplit, int nproj, int ldc, int nb,
                              double2* __restrict__ becp) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  const int p = blockIdx.y;
  if (b >= nb) return;
  double re = 0.0, im = 0.0;
  for (int ks = 0; ks < nsplit; ++ks) {
    const double2 v = partial[((size_t)ks * nproj + p) * ldc + b];
    re += v.x;
    im += v.y;
  }
  becp[(size_t)p * ldc + b] = make_double2(re, im);
}
// dbecp[p][b] = sum_j D[p][j] becp[blk_start(p)+j][b]; written both as dbecp[p][b] and transposed dbT[b][p]
__global__ void k_dmul(const double2* __restrict__ becp, int nproj, int ldc, int nb, const int* __restrict__ proj_blk0,
                       const int* __restrict__ proj_nh, const long long* __restrict__ proj_doff,
                       const double* __restrict__ dpk, double2* __restrict__ dbecp, double2* __restrict__ dbT, int ldp) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  const int p = blockIdx.y;
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
template <int BM, int BN, int WM, int WN, int NSTAGE>
__global__ void __launch_bounds__(WM* WN * 32, 1)
    k_vnl_add(const double2* __restrict__ beta, long long ldb, int nproj, int npw, const double2* __restrict__ dbT,
              int ldp, int nb, double2* __restrict__ hpsi, long long ldh) {
  using Cfg = ZgCfg<BM, BN, WM, WN, NSTAGE>;
  constexpr int NT = Cfg::NT, TM = Cfg::TM, TN = Cfg::TN;
  constexpr int LDA = BM + 2;  // row stride (complex) of the [k][g] tile: (2k + g) mod 8 distinct in a fragment load
  constexpr int STAGE = ZG_BK * LDA + BN * ZG_BK;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double2* sm = reinterpret_cast<double2*>(smem_raw);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm0 = (warp / WN) * (BM / WM), wn0 = (warp % WN) * (BN / WN);
  const int ntn = (nb + BN - 1) / BN;
  const int m0 = (blockIdx.x / ntn) * BM, n0 = (blockIdx.x % ntn) * BN;
  const int nkt = (nproj + ZG_BK - 1) / ZG_BK;

  auto load_stage = [&](int kt, int st) {
    double2* As = sm + st * STAGE;
    double2* Bs = As + ZG_BK * LDA;
    const int k0 = kt * ZG_BK;
    for (int id = tid; id < ZG_BK * BM; id += NT) {
      const int gc = id % BM, r = id / BM;
      const int p = k0 + r, gg = m0 + gc;
      const bool ok = p < nproj && gg < npw;
      cp_async16(&As[r * LDA + gc], ok ? &beta[(size_t)p * ldb + gg] : beta, ok);
    }
    for (int id = tid; id < BN * ZG_BK; id += NT) {
      const int kc = id & 7, r = id >> 3;
      const int b = n0 + r;
      const bool ok = b < nb && (k0 + kc) < nproj;
      cp_async16(&Bs[swz_k8(r, kc)], ok ? &dbT[(size_t)b * ldp + k0 + kc] : dbT, ok);
    }
  };

  double cre[TM][TN][2], cim[TM][TN][2];
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) cre[i][j][0] = cre[i][j][1] = cim[i][j][0] = cim[i][j][1] = 0.0;

#pragma unroll
  for (int s = 0; s < NSTAGE - 1; ++s) {
    if (s < nkt) load_stage(s, s);
    cp_async_commit();
  }
  const int fr = lane >> 2, fk = lane & 3;
  for (int kt = 0; kt < nkt; ++kt) {
    cp_async_wait<NSTAGE - 2>();
    __syncthreads();
    if (kt + NSTAGE - 1 < nkt) load_stage(kt + NSTAGE - 1, (kt + NSTAGE - 1) % NSTAGE);
    cp_async_commit();
    const double2* As = sm + (kt % NSTAGE) * STAGE;
    const double2* Bs = As + ZG_BK * LDA;
#pragma unroll
    for (int kk = 0; kk < 2; ++kk) {
      double2 af[TM], bf[TN];
#pragma unroll
      for (int i = 0; i < TM; ++i) af[i] = As[(kk * 4 + fk) * LDA + wm0 + i * 8 + fr];
#pragma unroll
      for (int j = 0; j < TN; ++j) bf[j] = Bs[swz_k8(wn0 + j * 8 + fr, kk * 4 + fk)];
#pragma unroll
      for (int j = 0; j < TN; ++j) {
        const double br = bf[j].x, bi = bf[j].y, nbi = -bf[j].y;
#pragma unroll
        for (int i = 0; i < TM; ++i) {
          // a b = (ar br - ai bi) + i (ar bi + ai br)
          dmma884(cre[i][j][0], cre[i][j][1], af[i].x, br);
          dmma884(cim[i][j][0], cim[i][j][1], af[i].x, bi);
          dmma884(cre[i][j][0], cre[i][j][1], af[i].y, nbi);
          dmma884(cim[i][j][0], cim[i][j][1], af[i].y, br);
        }
      }
    }
  }
  cp_async_wait<0>();
#pragma unroll
  for (int i = 0; i < TM; ++i) {
    const int gg = m0 + wm0 + i * 8 + fr;
    if (gg >= npw) continue;
#pragma unroll
    for (int j = 0; j < TN; ++j) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int b = n0 + wn0 + j * 8 + 2 * fk + e;
        if (b < nb) {
          double2* h = &hpsi[(size_t)b * ldh + gg];
          double2 v = *h;
          v.x += cre[i][j][e];
          v.y += cim[i][j][e];
          *h = v;
        }
      }
    }
  }
}

}  // namespace qehpsi
