// Projector contractions a6 / a8 on the 5th-generation tensor cores (tcgen05, kind::i8, s32 accumulators in TMEM) through an
// error-free split of the FP64 operands into signed 8-bit digits (the "Ozaki scheme"): SURVEY.md section 8(a) rows a6 and a8,
// DESIGN.md section 5.6.  tcgen05 has no f64 kind; int8 x int8 -> int32 products are exact, so with the balanced radix-256
// digits x_i in [-128, 127] of X = rint(x 2^(8S-1-e)) (e = exponent of the row maximum, |x| 2^-e <= 0.99, so |x_0| <= 127)
//
//   x = 2^e * sum_{i<S} x_i 2^-(7+8i) + O(2^(e-8S)),
//   sum_k a_k b_k = 2^(ea+eb-14) * sum_{L<S} 2^-8L * sum_{i+j=L} sum_k a_ik b_jk   + O((S+1) 2^(-8S+1) |a|max |b|max K)
//
// Both contractions are brought to the one form D[m][n] = sum_k A[m][k] B[n][k] over REAL k (a complex number is two
// consecutive reals), A and B stored as S planes of int8, K contiguous:
//   a6  becp[p][b]   : A row p  = (beta_r, beta_i)[p][g]      k = 2g+c        B row 2b = (psi_r, psi_i), row 2b+1 = (psi_i, -psi_r)
//   a8  hpsi[b][g] += : A row g  = (beta_r, beta_i)[p][g]      k = 2p+c        B row 2b = (d_r, -d_i),    row 2b+1 = (d_i, d_r)
// (Gamma-only handles: real forms, one B row / D column per band: a6 with B row b = (psi_r, psi_i); a8 with A row 2g+c =
//  component c of beta[.][g], k = p, and B row b = Re dbecp.)
// One CTA owns a 128 x 64 tile of D for one K range: S level accumulators of 64 TMEM columns each (level L = i+j), operands
// staged by TMA (SWIZZLE_64B, 64 bytes of K per stage) on a full/empty mbarrier ring, one thread issuing the MMAs, four
// warps converting the S int32 levels to FP64 in the epilogue.  Integer sums are exact, so results are bit-reproducible and do
// not depend on the batch composition (each band carries its own exponent).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>

namespace qehpsi {
namespace oz {

constexpr int BM = 128, BN = 64, KB = 64, NT = 192;
constexpr int A_BYTES = BM * KB, B_BYTES = BN * KB;
constexpr int MAX_STAGES = 4;
// (L+1) * Kc * 128 * 128 < 2^31 for every level L < S: Kc <= 2^17 / S reals per CTA
__host__ __device__ constexpr long long max_k_per_cta(int S) { return ((1LL << 17) / S) / KB * KB - KB; }
constexpr int E_BAD = -(1 << 28);  // exponent sentinel of a row with a non-finite entry
// 2^(ea+eb-14) d, or NaN when either operand row was non-finite
__device__ __forceinline__ double oz_scale(double d, int ea, int eb) {
  if (ea == E_BAD || eb == E_BAD) return __longlong_as_double(0x7ff8000000000000LL);
  return scalbn(d, ea + eb - 14);
}
__device__ __forceinline__ bool not_finite(double2 v) { return !(fabs(v.x) <= 1.7976931348623157e308) || !(fabs(v.y) <= 1.7976931348623157e308); }

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t n) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(n) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n.reg .pred p;\nWAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t sdst, const CUtensorMap* tm, int c0, int c1, int c2, uint64_t* bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(sdst),
               "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
               : "memory");
}
// K-major operand tile, rows of 64 bytes, SWIZZLE_64B: 8-row groups 512 bytes apart
__device__ __forceinline__ uint64_t desc_sw64(uint32_t saddr) {
  return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)1 << 16) | ((uint64_t)(512 >> 4) << 32) | ((uint64_t)1 << 46) |
         ((uint64_t)4 << 61);
}
__device__ __forceinline__ void mma_i8(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n}" ::"r"(tmem_d),
      "l"(da), "l"(db), "r"(idesc), "r"(acc)
      : "memory");
}
__device__ __forceinline__ void mma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// s8 x s8 -> s32, both operands K-major, M = 128, N = n (a multiple of 16, at most 256)
__host__ __device__ constexpr uint32_t idesc_n(int n) {
  return (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
}
// Digit products of one K block of 32: A_i x B_j accumulates into level i + j = TMEM columns [(i + j) BN, (i + j + 1) BN).  The B
// slices j = 0..S-1 of a stage are adjacent in shared memory (64 rows x 64 B each, 8-row groups 512 B apart), so B_j0..B_j0+w-1 is
// ONE K-major operand of w * 64 rows, and its product with A_i lands in the w consecutive levels i + j0 ..: one tcgen05.mma of
// N = 64 w (w <= 4) instead of w of N = 64.  A 128 x 64 x 32 instruction reads 6 KB of shared memory for 0.52 Mop, more than the
// 128 B / clk port delivers at the tensor rate (ncu: tensor pipe 50 % active, shared-memory operand cycles 61 %); at N = 256 it
// reads 12 KB for 2.1 Mop.  S (S + 1) / 2 instructions per K block become about S (S + 7) / 8: 21 -> 8 at S = 6, 28 -> 11 at S = 7.
template <int S>
__device__ __forceinline__ void mma_digits(uint32_t tm, uint32_t sb, int kk, uint32_t first) {
#pragma unroll
  for (int i = 0; i < S; ++i) {
    const uint64_t da = desc_sw64(sb + i * A_BYTES) + 2 * kk;
#pragma unroll
    for (int j0 = 0; j0 < S - i; j0 += 4) {
      const int w = (S - i - j0) < 4 ? (S - i - j0) : 4;
      const uint64_t db = desc_sw64(sb + S * A_BYTES + j0 * B_BYTES) + 2 * kk;
      mma_i8(tm + (uint32_t)(i + j0) * BN, da, db, idesc_n(w * BN), (first | (uint32_t)i) ? 1u : 0u);
    }
  }
}

// MODE 0 (a6): out = partial[split][m][ldo] complex, written; MODE 1 (a8): out = hpsi[b][ldo] complex at column m, accumulated.
// Gamma-only (real) forms, one column per band: MODE 2 (a6): partial[split][m][b] = (value, 0); MODE 3 (a8): row m = 2g + c
// of the transposed planar digits of beta, component c of hpsi[b][g] accumulated.
// MODE 4 (a8 of the Gamma-symmetric mode of a complex handle, sym_kernels.cuh): rows m = 2g + c over the leading sphere entries,
// columns 2b = X, 2b+1 = Y (real coefficient vectors Re e, Im e of band b); hpsi[b][g] += X + iY and hpsi[b][minus[g]] +=
// conj(X) + i conj(Y): lane pairs (c = 0, 1) exchange their components by shuffle, each lane updates component c of both entries.
template <int S, int MODE>
__global__ void __launch_bounds__(NT, 1)
k_oz_gemm(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, int nstages, int nkb, int kchunk,
          const int* __restrict__ ea, const int* __restrict__ eb, long long mvalid, int nb, double2* __restrict__ out,
          long long ldo, long long split_stride, int ks_base, const int* __restrict__ minus = nullptr) {
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ uint64_t full[MAX_STAGES], empty[MAX_STAGES], done;
  __shared__ uint32_t tmem_base;
  constexpr uint32_t STAGE = S * (A_BYTES + B_BYTES);
  constexpr uint32_t TCOLS = S * BN <= 256 ? 256 : 512;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int q = blockIdx.x, mt = blockIdx.y, ks = ks_base + blockIdx.z;  // ks_base: a8 walks its K ranges launch by launch
  const int kb0 = ks * kchunk;
  const int nit = max(0, min(nkb, kb0 + kchunk) - kb0);
  if constexpr (MODE == 4) {
    // row tiles whose plane waves all belong to the other half of the sphere (minus = -1) have nothing to store: retire before
    // any TMEM or pipeline set-up (see k_vnl_tma)
    const long long r = (long long)mt * BM + threadIdx.x;
    const bool dead = threadIdx.x >= BM || r >= mvalid || minus[r >> 1] == -1;
    if (__syncthreads_and(dead)) return;
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base)), "r"(TCOLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (threadIdx.x == 32) {
    for (int i = 0; i < MAX_STAGES; ++i) {
      mbar_init(&full[i], 1);
      mbar_init(&empty[i], 1);
    }
    mbar_init(&done, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tm = tmem_base;
  // the swizzle pattern is a function of the address: align the ring explicitly (the launch asks for 1 KB more than it uses)
  const uint32_t sbase0 = (smem_u32(smem) + 1023u) & ~1023u;

  if (warp == 0 && lane == 0) {
    // ---- TMA producer ----
    for (int it = 0; it < nit; ++it) {
      const int st = it % nstages;
      const uint32_t ph = (uint32_t)(it / nstages) & 1u;
      mbar_wait(&empty[st], ph ^ 1u);
      mbar_expect_tx(&full[st], STAGE);
      const uint32_t sb = sbase0 + (uint32_t)st * STAGE;
      const int kx = (kb0 + it) * KB;
#pragma unroll
      for (int i = 0; i < S; ++i) tma_load_3d(sb + i * A_BYTES, &tmA, kx, mt * BM, i, &full[st]);
#pragma unroll
      for (int j = 0; j < S; ++j) tma_load_3d(sb + S * A_BYTES + j * B_BYTES, &tmB, kx, q * BN, j, &full[st]);
    }
  } else if (warp == 1 && lane == 0) {
    // ---- MMA issuer: level L = i + j accumulates into TMEM columns [L*64, L*64+64) ----
    for (int it = 0; it < nit; ++it) {
      const int st = it % nstages;
      const uint32_t ph = (uint32_t)(it / nstages) & 1u;
      mbar_wait(&full[st], ph);
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      const uint32_t sb = sbase0 + (uint32_t)st * STAGE;
#pragma unroll
      for (int kk = 0; kk < KB / 32; ++kk) {
        mma_digits<S>(tm, sb, kk, (uint32_t)(it | kk));
      }
      mma_commit(&empty[st]);
    }
    mma_commit(&done);
  } else if (warp >= 2) {
    // ---- epilogue: warp w reads TMEM lanes 32 (w % 4) .. +31; thread = row of the tile ----
    const int wq = warp & 3;
    const long long m = (long long)mt * BM + wq * 32 + lane;
    // the accumulating forms (MODE 1, 3, 4) fetch the hpsi entries this thread will update into registers NOW, while the MMAs run
    // and these warps have nothing else to do: the epilogue below is then TMEM reads, FP64 recombination and stores, without a
    // global round trip per column group.  Only this thread writes these entries (each (row, band) has one owner; K ranges are
    // separate launches).
    double pre[(MODE == 1 || MODE == 3) ? BN : 1];  // MODE 1: (re, im) of hpsi[b][m] for the BN / 2 bands; MODE 3: component m of the BN bands
    if constexpr (MODE == 1) {
#pragma unroll
      for (int jj = 0; jj < BN / 2; ++jj) {
        const int b = q * (BN / 2) + jj;
        const double2 v = (m < mvalid && b < nb) ? out[(size_t)b * ldo + m] : make_double2(0.0, 0.0);
        pre[2 * jj] = v.x;
        pre[2 * jj + 1] = v.y;
      }
    } else if constexpr (MODE == 3) {
#pragma unroll
      for (int j = 0; j < BN; ++j) {
        const int b = q * BN + j;
        pre[j] = (m < mvalid && b < nb) ? reinterpret_cast<const double*>(out + (size_t)b * ldo)[m] : 0.0;
      }
    }
    // MODE 4: component c of row g and of row -G, one pair per band of the tile
    double pg[MODE == 4 ? BN / 2 : 1], pm[MODE == 4 ? BN / 2 : 1];
    if constexpr (MODE == 4) {
      const bool ok = m < mvalid;
      const long long g = m >> 1;
      const int c = (int)(m & 1);
      const int mg = ok ? minus[g] : -1;
#pragma unroll
      for (int jp = 0; jp < BN / 2; ++jp) {
        const int col = q * BN + 2 * jp;
        pg[jp] = pm[jp] = 0.0;
        if (ok && col < nb && mg != -1) {
          const double* row = reinterpret_cast<const double*>(out + (size_t)(col >> 1) * ldo);
          pg[jp] = row[2 * g + c];
          if (mg >= 0) pm[jp] = row[2 * (long long)mg + c];
        }
      }
    }
    mbar_wait(&done, 0);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const int em = (m < mvalid) ? ea[MODE >= 3 ? (m >> 1) : m] : 0;  // MODE 3, 4: rows 2g, 2g+1 share the exponent of plane wave g
#pragma unroll(MODE == 1 || MODE >= 3 ? BN / 8 : 1)
    for (int n0 = 0; n0 < BN; n0 += 8) {
      double d[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) d[j] = 0.0;
      if (nit > 0) {
        uint32_t v[S][8];
#pragma unroll
        for (int L = 0; L < S; ++L) {
          const uint32_t ta = tm + ((uint32_t)(wq * 32) << 16) + (uint32_t)(L * BN + n0);
          asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                       : "=r"(v[L][0]), "=r"(v[L][1]), "=r"(v[L][2]), "=r"(v[L][3]), "=r"(v[L][4]), "=r"(v[L][5]), "=r"(v[L][6]),
                         "=r"(v[L][7])
                       : "r"(ta));
        }
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
        for (int L = S - 1; L >= 0; --L) {  // smallest contributions first
          const double w = 1.0 / (double)(1ULL << (8 * L));
#pragma unroll
          for (int j = 0; j < 8; ++j) d[j] = fma((double)(int)v[L][j], w, d[j]);
        }
      }
      if (MODE == 4) {
        const bool ok = m < mvalid;
        const long long g = m >> 1;
        const int c = (int)(m & 1);
        const int mg = ok ? minus[g] : -1;
        double og[4], om[4], vg[4], vm[4];
        bool wr[4];
#pragma unroll
        for (int jp = 0; jp < 4; ++jp) {
          const int col = q * BN + n0 + 2 * jp;  // X column of band col / 2; nb = number of columns (even)
          const bool cok = col < nb;
          const double x = oz_scale(d[2 * jp], em, cok ? eb[col] : 0), y = oz_scale(d[2 * jp + 1], em, cok ? eb[col + 1] : 0);
          const double yo = __shfl_xor_sync(0xffffffffu, y, 1);  // the other component of Y (lanes 2k, 2k+1 hold rows 2g, 2g+1)
          // c = 0: Re(G) += X_r - Y_i, Re(-G) += X_r + Y_i;   c = 1: Im(G) += X_i + Y_r, Im(-G) += Y_r - X_i
          vg[jp] = c == 0 ? x - yo : x + yo;
          vm[jp] = c == 0 ? x + yo : yo - x;
          wr[jp] = ok && cok && mg != -1;
          og[jp] = pg[n0 / 2 + jp];  // fetched before the wait (see above)
          om[jp] = pm[n0 / 2 + jp];
        }
#pragma unroll
        for (int jp = 0; jp < 4; ++jp) {
          if (wr[jp]) {
            double* row = reinterpret_cast<double*>(out + (size_t)((q * BN + n0 + 2 * jp) >> 1) * ldo);
            row[2 * g + c] = og[jp] + vg[jp];
            if (mg >= 0) row[2 * (long long)mg + c] = om[jp] + vm[jp];
          }
        }
      } else if (MODE >= 2) {  // real forms of the Gamma-only handle: one column per band
        if (m < mvalid) {
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const int b = q * BN + n0 + j;
            if (b < nb) {
              const double val = oz_scale(d[j], em, eb[b]);
              if (MODE == 2)
                out[(size_t)ks * split_stride + (size_t)m * ldo + b] = make_double2(val, 0.0);
              else
                reinterpret_cast<double*>(out + (size_t)b * ldo)[m] = pre[MODE == 3 ? n0 + j : 0] + val;  // m = 2g + c: component c of hpsi[b][g]
            }
          }
        }
      } else if (m < mvalid) {
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
          const int b = (q * BN + n0) / 2 + jj;
          if (b < nb) {
            const double re = oz_scale(d[2 * jj], em, eb[b]), im = oz_scale(d[2 * jj + 1], em, eb[b]);
            if (MODE == 0)
              out[(size_t)ks * split_stride + (size_t)m * ldo + b] = make_double2(re, im);
            else
              out[(size_t)b * ldo + m] = make_double2(pre[MODE == 1 ? n0 + 2 * jj : 0] + re, pre[MODE == 1 ? n0 + 2 * jj + 1 : 0] + im);
          }
        }
      }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) {
    __syncwarp();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tm), "r"(TCOLS) : "memory");
  }
}

// ---- exponents: smallest e with max |component| 2^-e <= 0.99 (0 for an all-zero row): the leading digit then fits an int8 ----
// A row holding a NaN or an infinity gets the sentinel E_BAD: its digits are meaningless, and every epilogue writes NaN for
// the outputs that depend on it (oz_scale), which is what the FP64 contraction would give.
__device__ __forceinline__ int exp_of(double mx, bool bad) {
  if (bad) return E_BAD;
  if (!(mx > 0.0)) return 0;
  int e = ilogb(mx) + 1;
  if (scalbn(mx, -e) > 0.99) ++e;
  return e;
}

// one CTA per row of a complex matrix X[rows][ldx], n entries per row
__global__ void __launch_bounds__(256) k_oz_rowexp(const double2* __restrict__ X, long long ldx, long long n, int* __restrict__ e) {
  __shared__ double red[256];
  __shared__ int anybad;
  if (threadIdx.x == 0) anybad = 0;
  const double2* x = X + (size_t)blockIdx.x * ldx;
  double mx = 0.0;
  bool bad = false;
  for (long long i = threadIdx.x; i < n; i += 256) {
    const double2 v = x[i];
    bad |= not_finite(v);
    mx = fmax(mx, fmax(fabs(v.x), fabs(v.y)));
  }
  red[threadIdx.x] = mx;
  __syncthreads();
  if (bad) anybad = 1;
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) red[threadIdx.x] = fmax(red[threadIdx.x], red[threadIdx.x + s]);
    __syncthreads();
  }
  if (threadIdx.x == 0) e[blockIdx.x] = exp_of(red[0], anybad != 0);
}
// one thread per column g of X[rows][ldx]
__global__ void __launch_bounds__(128) k_oz_colexp(const double2* __restrict__ X, long long ldx, int rows, long long n, int* __restrict__ e) {
  const long long g = (long long)blockIdx.x * 128 + threadIdx.x;
  if (g >= n) return;
  double mx = 0.0;
  bool bad = false;
  for (int p = 0; p < rows; ++p) {
    const double2 v = X[(size_t)p * ldx + g];
    bad |= not_finite(v);
    mx = fmax(mx, fmax(fabs(v.x), fabs(v.y)));
  }
  e[g] = exp_of(mx, bad);
}

// 16 reals -> S x 16 int8 (one 16-byte store per slice); r[] already scaled to [-0.99, 0.99].  Balanced radix-256 digits of the
// integer X = rint(r 2^(8S-1)), least significant first: d = ((X + 128) mod 256) - 128, X <- (X - d) / 256.  Exact for S <= 7.
template <int S>
__device__ __forceinline__ void slice16(double (&r)[16], uint4 (&o)[S]) {
  static_assert(S >= 2 && S <= 7, "8S-1 bits must fit an int64");
  uint32_t w[S][4];
#pragma unroll
  for (int sl = 0; sl < S; ++sl) w[sl][0] = w[sl][1] = w[sl][2] = w[sl][3] = 0u;
#pragma unroll
  for (int t = 0; t < 16; ++t) {
    long long X = __double2ll_rn(r[t] * (double)(1ULL << (8 * S - 1)));
#pragma unroll
    for (int sl = S - 1; sl >= 0; --sl) {
      const long long d = ((X + 128) & 255) - 128;
      X = (X - d) >> 8;
      w[sl][t >> 2] |= ((uint32_t)d & 0xFFu) << (8 * (t & 3));
    }
  }
#pragma unroll
  for (int sl = 0; sl < S; ++sl) o[sl] = make_uint4(w[sl][0], w[sl][1], w[sl][2], w[sl][3]);
}

// rows of X (complex, n per row) -> int8 planes out[sl][orow][kpad], k = 2g + c.
// mode 0: orow = r: (re, im).  mode 1: orow = 2r: (re, im), 2r+1: (im, -re).  mode 2: orow = 2r: (re, -im), 2r+1: (im, re).
// (real parts only, k = g: k_oz_slice_re below)
template <int S>
__global__ void __launch_bounds__(128)
k_oz_slice(const double2* __restrict__ X, long long ldx, long long n, const int* __restrict__ e, int8_t* __restrict__ out,
           long long kpad, long long slice_stride, int mode, const unsigned char* __restrict__ cls = nullptr) {
  const long long g0 = ((long long)blockIdx.x * 128 + threadIdx.x) * 8;
  if (g0 * 2 >= kpad) return;
  const int r = blockIdx.y;
  const int ex = -e[r];
  const bool rot = cls != nullptr && cls[r] != 0;  // Gamma-symmetric mode: a class-1 row is sliced as i * x = (-im, re)
  double a[16], b2[16];
#pragma unroll
  for (int t = 0; t < 8; ++t) {
    double2 v = make_double2(0.0, 0.0);
    if (g0 + t < n) v = X[(size_t)r * ldx + g0 + t];
    if (rot) v = make_double2(-v.y, v.x);
    const double re = scalbn(v.x, ex), im = scalbn(v.y, ex);
    if (mode == 2) {
      a[2 * t] = re, a[2 * t + 1] = -im;
      b2[2 * t] = im, b2[2 * t + 1] = re;
    } else {
      a[2 * t] = re, a[2 * t + 1] = im;
      b2[2 * t] = im, b2[2 * t + 1] = -re;
    }
  }
  uint4 o[S];
  slice16<S>(a, o);
  const long long orow = mode == 0 ? r : 2LL * r;
#pragma unroll
  for (int sl = 0; sl < S; ++sl) *reinterpret_cast<uint4*>(out + (size_t)sl * slice_stride + (size_t)orow * kpad + 2 * g0) = o[sl];
  if (mode != 0) {
    slice16<S>(b2, o);
#pragma unroll
    for (int sl = 0; sl < S; ++sl)
      *reinterpret_cast<uint4*>(out + (size_t)sl * slice_stride + (size_t)(orow + 1) * kpad + 2 * g0) = o[sl];
  }
}

// transpose-and-slice: X[rows = p][ldx] -> out[sl][g][kpad], k = 2p + c, row g scaled by 2^-e[g]; 8 rows p per thread
template <int S>
__global__ void __launch_bounds__(128)
k_oz_slice_t(const double2* __restrict__ X, long long ldx, int rows, long long n, const int* __restrict__ e,
             int8_t* __restrict__ out, long long kpad, long long slice_stride) {
  const long long g = (long long)blockIdx.x * 128 + threadIdx.x;
  if (g >= n) return;
  const int p0 = blockIdx.y * 8;
  const int ex = -e[g];
  double a[16];
#pragma unroll
  for (int t = 0; t < 8; ++t) {
    double2 v = make_double2(0.0, 0.0);
    if (p0 + t < rows) v = X[(size_t)(p0 + t) * ldx + g];
    a[2 * t] = scalbn(v.x, ex);
    a[2 * t + 1] = scalbn(v.y, ex);
  }
  uint4 o[S];
  slice16<S>(a, o);
#pragma unroll
  for (int sl = 0; sl < S; ++sl) *reinterpret_cast<uint4*>(out + (size_t)sl * slice_stride + (size_t)g * kpad + 2 * p0) = o[sl];
}

// Gamma-only a8, B operand: rows of X (complex with zero imaginary part, n per row) -> out[sl][r][kpad], k = g, value Re x
template <int S>
__global__ void __launch_bounds__(128)
k_oz_slice_re(const double2* __restrict__ X, long long ldx, long long n, const int* __restrict__ e, int8_t* __restrict__ out,
              long long kpad, long long slice_stride) {
  const long long g0 = ((long long)blockIdx.x * 128 + threadIdx.x) * 16;
  if (g0 >= kpad) return;
  const int r = blockIdx.y;
  const int ex = -e[r];
  double a[16];
#pragma unroll
  for (int t = 0; t < 16; ++t) a[t] = g0 + t < n ? scalbn(X[(size_t)r * ldx + g0 + t].x, ex) : 0.0;
  uint4 o[S];
  slice16<S>(a, o);
#pragma unroll
  for (int sl = 0; sl < S; ++sl) *reinterpret_cast<uint4*>(out + (size_t)sl * slice_stride + (size_t)r * kpad + g0) = o[sl];
}
// Gamma-only a8, A operand: X[rows = p][ldx] -> out[sl][2g + c][kpad], k = p, rows 2g and 2g+1 scaled by 2^-e[g]; 16 rows p per thread
template <int S>
__global__ void __launch_bounds__(128)
k_oz_slice_tp(const double2* __restrict__ X, long long ldx, int rows, long long n, const int* __restrict__ e,
              int8_t* __restrict__ out, long long kpad, long long slice_stride, const unsigned char* __restrict__ cls = nullptr) {
  const long long g = (long long)blockIdx.x * 128 + threadIdx.x;
  if (g >= n) return;
  const int p0 = blockIdx.y * 16;
  const int ex = -e[g];
  double re[16], im[16];
#pragma unroll
  for (int t = 0; t < 16; ++t) {
    double2 v = make_double2(0.0, 0.0);
    if (p0 + t < rows) {
      v = X[(size_t)(p0 + t) * ldx + g];
      if (cls != nullptr && cls[p0 + t] != 0) v = make_double2(-v.y, v.x);  // Gamma-symmetric mode: class-1 projector enters as i * beta
    }
    re[t] = scalbn(v.x, ex);
    im[t] = scalbn(v.y, ex);
  }
  uint4 o[S];
  slice16<S>(re, o);
#pragma unroll
  for (int sl = 0; sl < S; ++sl) *reinterpret_cast<uint4*>(out + (size_t)sl * slice_stride + (size_t)(2 * g) * kpad + p0) = o[sl];
  slice16<S>(im, o);
#pragma unroll
  for (int sl = 0; sl < S; ++sl) *reinterpret_cast<uint4*>(out + (size_t)sl * slice_stride + (size_t)(2 * g + 1) * kpad + p0) = o[sl];
}

// ---- integer 3M form of a6 (complex handles): conj(beta) psi from three real products over the complex index g --------------
// planes 0, 1, 2 of a row x: Re x, Im x, (Re x + sgn Im x) / 2   (sgn = -1 for beta: the conjugate; +1 for psi), so that with
// Q1 = sum beta_r psi_r, Q2 = sum beta_i psi_i, Q3 = sum plane2(beta) plane2(psi):  becp = (Q1 + Q2) + i (4 Q3 - Q1 + Q2).
// out[sl][plane][row][kpad], k = g; 16 complex entries per thread.
template <int S>
__global__ void __launch_bounds__(128)
k_oz_slice3(const double2* __restrict__ X, long long ldx, long long n, const int* __restrict__ e, int8_t* __restrict__ out,
            long long kpad, long long plane_stride, long long slice_stride, double sgn) {
  const long long g0 = ((long long)blockIdx.x * 128 + threadIdx.x) * 16;
  if (g0 >= kpad) return;
  const int r = blockIdx.y;
  const int ex = -e[r];
  double re[16], im[16], sm[16];
#pragma unroll
  for (int t = 0; t < 16; ++t) {
    double2 v = make_double2(0.0, 0.0);
    if (g0 + t < n) v = X[(size_t)r * ldx + g0 + t];
    re[t] = scalbn(v.x, ex);
    im[t] = scalbn(v.y, ex);
    sm[t] = 0.5 * (re[t] + sgn * im[t]);
  }
  uint4 o[S];
  int8_t* base = out + (size_t)r * kpad + g0;
  slice16<S>(re, o);
#pragma unroll
  for (int sl = 0; sl < S; ++sl) *reinterpret_cast<uint4*>(base + (size_t)sl * slice_stride) = o[sl];
  slice16<S>(im, o);
#pragma unroll
  for (int sl = 0; sl < S; ++sl) *reinterpret_cast<uint4*>(base + (size_t)sl * slice_stride + plane_stride) = o[sl];
  slice16<S>(sm, o);
#pragma unroll
  for (int sl = 0; sl < S; ++sl) *reinterpret_cast<uint4*>(base + (size_t)sl * slice_stride + 2 * plane_stride) = o[sl];
}
// a7 front end of the 3M form: partial[plane][split][p][ldc].x summed over the splits in ascending order, then combined
__global__ void k_oz_reduce3(const double2* __restrict__ partial, int nsplit, int nproj, int ldc, int nb, double2* __restrict__ becp) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  const int p = blockIdx.y;
  if (b >= nb) return;
  double q[3];
#pragma unroll
  for (int pl = 0; pl < 3; ++pl) {
    double acc = 0.0;
    for (int ks = 0; ks < nsplit; ++ks) acc += partial[(((size_t)pl * nsplit + ks) * nproj + p) * ldc + b].x;
    q[pl] = acc;
  }
  becp[(size_t)p * ldc + b] = make_double2(q[0] + q[1], (4.0 * q[2] - q[0]) + q[1]);
}

// ---- integer 3M form of a8 (complex handles): hpsi[b][g] += sum_p beta[p][g] d[p][b] from three real products over p ---------
// A planes (k_oz_slice_t3): rows g, k = p: beta_r, beta_i, (beta_r + beta_i) / 2;  B planes (k_oz_slice3, sgn = +1): d_r, d_i, half sum.
// Q1 = sum beta_r d_r, Q2 = sum beta_i d_i, Q3 = sum of the half-sum planes:  Re = Q1 - Q2,  Im = 4 Q3 - Q1 - Q2.
// One CTA runs the three planes back to back for its 128 x 64 (rows g x bands) tile: the TMA ring and the MMA issue never stop;
// after each plane the epilogue warps pull the S levels out of TMEM into 64 FP64 registers per thread, hand TMEM back, and add
// (cr, ci) * Q to hpsi while the next plane is being multiplied.  K = nproj is not split (needs 128-padded nproj <= max_k_per_cta).
template <int S>
__global__ void __launch_bounds__(NT, 1)
k_oz_vnl3(const __grid_constant__ CUtensorMap tmA0, const __grid_constant__ CUtensorMap tmA1, const __grid_constant__ CUtensorMap tmA2,
          const __grid_constant__ CUtensorMap tmB0, const __grid_constant__ CUtensorMap tmB1, const __grid_constant__ CUtensorMap tmB2,
          int nstages, int nkb, const int* __restrict__ ea, const int* __restrict__ eb, long long mvalid, int nb,
          double2* __restrict__ out, long long ldo) {
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ uint64_t full[MAX_STAGES], empty[MAX_STAGES], done, tfree;
  __shared__ uint32_t tmem_base;
  constexpr uint32_t STAGE = S * (A_BYTES + B_BYTES);
  constexpr uint32_t TCOLS = S * BN <= 256 ? 256 : 512;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int q = blockIdx.x, mt = blockIdx.y;
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base)), "r"(TCOLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (threadIdx.x == 32) {
    for (int i = 0; i < MAX_STAGES; ++i) {
      mbar_init(&full[i], 1);
      mbar_init(&empty[i], 1);
    }
    mbar_init(&done, 1);
    mbar_init(&tfree, 128);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tm = tmem_base;
  const uint32_t sbase0 = (smem_u32(smem) + 1023u) & ~1023u;

  if (warp == 0 && lane == 0) {
    // ---- TMA producer: planes 0, 1, 2 back to back through one ring ----
    int n = 0;
    for (int pl = 0; pl < 3; ++pl) {
      const CUtensorMap* ta = pl == 0 ? &tmA0 : pl == 1 ? &tmA1 : &tmA2;
      const CUtensorMap* tb = pl == 0 ? &tmB0 : pl == 1 ? &tmB1 : &tmB2;
      for (int it = 0; it < nkb; ++it, ++n) {
        const int st = n % nstages;
        const uint32_t ph = (uint32_t)(n / nstages) & 1u;
        mbar_wait(&empty[st], ph ^ 1u);
        mbar_expect_tx(&full[st], STAGE);
        const uint32_t sb = sbase0 + (uint32_t)st * STAGE;
#pragma unroll
        for (int i = 0; i < S; ++i) tma_load_3d(sb + i * A_BYTES, ta, it * KB, mt * BM, i, &full[st]);
#pragma unroll
        for (int j = 0; j < S; ++j) tma_load_3d(sb + S * A_BYTES + j * B_BYTES, tb, it * KB, q * BN, j, &full[st]);
      }
    }
  } else if (warp == 1 && lane == 0) {
    // ---- MMA issuer ----
    int n = 0;
    for (int pl = 0; pl < 3; ++pl) {
      if (pl > 0) {  // the epilogue warps have read plane pl-1 out of TMEM
        mbar_wait(&tfree, (uint32_t)(pl - 1) & 1u);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      }
      for (int it = 0; it < nkb; ++it, ++n) {
        const int st = n % nstages;
        const uint32_t ph = (uint32_t)(n / nstages) & 1u;
        mbar_wait(&full[st], ph);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const uint32_t sb = sbase0 + (uint32_t)st * STAGE;
#pragma unroll
        for (int kk = 0; kk < KB / 32; ++kk) {
          mma_digits<S>(tm, sb, kk, (uint32_t)(it | kk));
        }
        mma_commit(&empty[st]);
      }
      mma_commit(&done);
    }
  } else if (warp >= 2) {
    // ---- epilogue warps: thread = row g of the tile ----
    const int wq = warp & 3;
    const long long m = (long long)mt * BM + wq * 32 + lane;
    const bool row_ok = m < mvalid;
    const int em = row_ok ? ea[m] : 0;
    if (row_ok)
      for (int j = 0; j < BN; ++j)
        if (q * BN + j < nb) asm volatile("prefetch.global.L2 [%0];" ::"l"(out + (size_t)(q * BN + j) * ldo + m));
    for (int pl = 0; pl < 3; ++pl) {
      mbar_wait(&done, (uint32_t)pl & 1u);
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      double val[BN];
#pragma unroll
      for (int n0 = 0; n0 < BN; n0 += 8) {
        uint32_t v[S][8];
#pragma unroll
        for (int L = 0; L < S; ++L) {
          const uint32_t ta = tm + ((uint32_t)(wq * 32) << 16) + (uint32_t)(L * BN + n0);
          asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                       : "=r"(v[L][0]), "=r"(v[L][1]), "=r"(v[L][2]), "=r"(v[L][3]), "=r"(v[L][4]), "=r"(v[L][5]), "=r"(v[L][6]),
                         "=r"(v[L][7])
                       : "r"(ta));
        }
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
        for (int j = 0; j < 8; ++j) val[n0 + j] = 0.0;
#pragma unroll
        for (int L = S - 1; L >= 0; --L) {
          const double w = 1.0 / (double)(1ULL << (8 * L));
#pragma unroll
          for (int j = 0; j < 8; ++j) val[n0 + j] = fma((double)(int)v[L][j], w, val[n0 + j]);
        }
      }
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&tfree)) : "memory");
      const double cr = pl == 0 ? 1.0 : pl == 1 ? -1.0 : 0.0, ci = pl == 2 ? 4.0 : -1.0;
      if (row_ok) {
        // four loads in flight before their stores (the compiler cannot prove the entries distinct: interleaved
        // read-modify-writes would cost one global round trip each)
#pragma unroll
        for (int j0 = 0; j0 < BN; j0 += 4) {
          double2 t[4];
#pragma unroll
          for (int jj = 0; jj < 4; ++jj) {
            const int b = q * BN + j0 + jj;
            t[jj] = b < nb ? out[(size_t)b * ldo + m] : make_double2(0.0, 0.0);
          }
#pragma unroll
          for (int jj = 0; jj < 4; ++jj) {
            const int b = q * BN + j0 + jj;
            if (b < nb) {
              const double x = oz_scale(val[j0 + jj], em, eb[b]);
              out[(size_t)b * ldo + m] = make_double2(fma(cr, x, t[jj].x), fma(ci, x, t[jj].y));
            }
          }
        }
      }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) {
    __syncwarp();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tm), "r"(TCOLS) : "memory");
  }
}
// A operand of k_oz_vnl3: X[rows = p][ldx] -> out[sl][plane][g][kpad], k = p, row g scaled by 2^-e[g]; 16 rows p per thread
template <int S>
__global__ void __launch_bounds__(128)
k_oz_slice_t3(const double2* __restrict__ X, long long ldx, int rows, long long n, const int* __restrict__ e,
              int8_t* __restrict__ out, long long kpad, long long plane_stride, long long slice_stride) {
  const long long g = (long long)blockIdx.x * 128 + threadIdx.x;
  if (g >= n) return;
  const int p0 = blockIdx.y * 16;
  const int ex = -e[g];
  double re[16], im[16], sm[16];
#pragma unroll
  for (int t = 0; t < 16; ++t) {
    double2 v = make_double2(0.0, 0.0);
    if (p0 + t < rows) v = X[(size_t)(p0 + t) * ldx + g];
    re[t] = scalbn(v.x, ex);
    im[t] = scalbn(v.y, ex);
    sm[t] = 0.5 * (re[t] + im[t]);
  }
  uint4 o[S];
  int8_t* base = out + (size_t)g * kpad + p0;
  slice16<S>(re, o);
#pragma unroll
  for (int sl = 0; sl < S; ++sl) *reinterpret_cast<uint4*>(base + (size_t)sl * slice_stride) = o[sl];
  slice16<S>(im, o);
#pragma unroll
  for (int sl = 0; sl < S; ++sl) *reinterpret_cast<uint4*>(base + (size_t)sl * slice_stride + plane_stride) = o[sl];
  slice16<S>(sm, o);
#pragma unroll
  for (int sl = 0; sl < S; ++sl) *reinterpret_cast<uint4*>(base + (size_t)sl * slice_stride + 2 * plane_stride) = o[sl];
}

}  // namespace oz
}  // namespace qehpsi
