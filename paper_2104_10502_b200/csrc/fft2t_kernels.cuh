// fft2t_kernels.cuh -- TMA-staged x stage (step a3) of the two-pass fast path.
// Same arithmetic as k2p_x_vmul (fft2p_kernels.cuh): inverse FFT along i1 over the P populated planes, * V(r)/N, forward
// FFT, keep the populated planes.  What changes is how the [P][8-column] tile of W2 moves: one elected thread issues a
// single 3-D tensor-map bulk copy (cp.async.bulk.tensor, box = 1 band x P planes x 128 bytes) per band into a shared
// staging buffer, completion on an mbarrier, and one bulk tensor store of the result from a second staging buffer; the
// compute threads only touch shared memory.  The load of band b+1 and the store of band b-1 overlap the butterflies of
// band b, which the register-starved radix-16 kernel (two 4-warp CTAs per SM) could not do with its own loads and
// strided 16-byte stores: 43.8 -> 32.2 us per band at 192^3 (profiles/r1e_capture.md).  The twiddles tw[q*j] of both
// passes depend on the thread only and live in registers.  PAPER.md:L215 (1-D FFT stages), L224-226 (local potential).
#pragma once
#include <cuda.h>

#include "fft3p_kernels.cuh"

namespace qehpsi {

__device__ __forceinline__ unsigned smem_u32(const void* p) { return static_cast<unsigned>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n.reg .pred p;\nWAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}

// dynamic shared memory: tiles [2][N][FFT_C] (the two-pass kernel uses one), input stage [P][FFT_C], output stage [P][FFT_C],
// one mbarrier, and (two-pass kernel) the twiddle table tw[q*j] as [RA][RA+1] (RA <= 16)
// (the mbarrier of the two-pass kernel lives in the unused [0][0] entry of its twiddle table; the three-pass kernel has no table)
inline size_t fft2t_smem(int n, int P, bool two_pass, bool one_tile) {
  return (one_tile ? 1 : 2) * (size_t)n * FFT_C * sizeof(double2) + 2 * (size_t)(P + (two_pass ? 1 : 0)) * FFT_C * sizeof(double2) +
         (two_pass ? 16 * 17 * sizeof(double2) : 64);
}

// Radix-R DFT (R = 4 Q) whose inputs Q .. 3Q - 1 are zero: the first stage of Dft<R> (4-point DFTs over v[b], v[Q + b], v[2Q + b],
// v[3Q + b]) sees (t0, 0, 0, t3) and needs 4 complex additions instead of 8; the rest is Dft<R>.  Used by the x stage when the
// populated planes lie in the outer quarters of the axis (HALF below): same sums as Dft<R> on zero-padded inputs up to the sign of
// an exact zero.
template <int R, int DIR>
struct DftHalfIn {
  static constexpr int Q = R / 4;
  static_assert(R % 4 == 0, "quarter pruning needs a radix-4 first stage");
  __device__ __forceinline__ static void run(double2 (&v)[R]) {
    double2 y[Q][4];
    static_for<Q>([&](auto b_) {
      constexpr int b = decltype(b_)::value;
      const double2 t0 = v[b], t3 = v[3 * Q + b];
      const double2 d = cmul_i<DIR>(make_double2(-t3.x, -t3.y));
      double2 t[4] = {cadd(t0, t3), cadd(t0, d), csub(t0, t3), csub(t0, d)};
      static_for<4>([&](auto c_) {
        constexpr int c = decltype(c_)::value;
        y[b][c] = cmul_tw<b * c, R, DIR>(t[c]);
      });
    });
    static_for<4>([&](auto c_) {
      constexpr int c = decltype(c_)::value;
      double2 u[Q];
      static_for<Q>([&](auto b_) {
        constexpr int b = decltype(b_)::value;
        u[b] = y[b][c];
      });
      Dft<Q, DIR>::run(u);
      static_for<Q>([&](auto d_) {
        constexpr int d = decltype(d_)::value;
        v[c + 4 * d] = u[d];
      });
    });
  }
};

// tmap: W2 viewed as FP64 [nb][P][N2*ldz*2], box {16, P, 1}
// Register diet (round 2): the second-pass twiddles tw[q*j] sit in a padded shared table instead of 64 registers, and the
// populated-plane index comes from the wrapped-interval rule of Fft2pGeom (x_hi, x_lo) instead of a 16-entry register array:
// 222 -> under 168 registers, three CTAs per SM instead of two, so the FP64 pipe has 12 warps to pick from across the
// three barriers of a band (the stage is bound by FP64 issue, not HBM: DESIGN.md section 6).
// HALF (RA = 4 QA): every populated plane has i1 < QA RB or i1 >= 3 QA RB, i.e. the inputs q in [QA, 3 QA) of every radix-RA
// transform of the inverse pass are zero and the same outputs of the forward pass are not kept (true whenever the grid holds the
// sphere twice over, x_hi < N / 4: the density-grid rule; checked on the host).  Those 2 QA of 4 QA shared-memory reads and
// writes per thread are not made at all, the inverse butterfly is DftHalfIn, and the unused outputs of the forward butterfly
// fall to dead-code elimination: the stage is bound by shared-memory traffic and FP64 issue, not by HBM.
template <int RA, int RB, bool HALF = false>
__global__ void __launch_bounds__(RA* FFT_C, 3)
k2t_x_vmul(FftGeom g, Fft2pGeom t, const __grid_constant__ CUtensorMap tmap, int nb, int one_tile) {
  static_assert(RB > 1, "single-pass lengths use k2p_x_vmul");
  static_assert(!HALF || RA % 4 == 0, "quarter pruning");
  constexpr int QA = RA / 4;
  static_assert(RA >= RB && RA <= 16, "twiddle table is [RA][RA+1]");
  constexpr int N = RA * RB, NT = RA * FFT_C, NW = (NT + 31) / 32, TWP = RA + 1;
  constexpr unsigned ROWB = FFT_C * sizeof(double2);  // 128 bytes per plane row of the tile
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* tile1 = reinterpret_cast<double2*>(smem_raw);
  // one_tile: the tile is reused between the passes (two more barriers per band, 24 KB less per CTA at N = 192)
  double2* tile2 = one_tile ? tile1 : tile1 + N * FFT_C;
  // both stages carry one extra row P: a zero row in the input stage (what an unpopulated plane reads) and a sink row in the
  // output stage (what it writes), so the loads and stores of the radix-RA passes are unconditional: no branches around them
  double2* inb = tile2 + N * FFT_C;
  const int P = g.P;
  double2* outb = inb + (size_t)(P + 1) * FFT_C;
  double2* twt = outb + (size_t)(P + 1) * FFT_C;
  unsigned long long* full = reinterpret_cast<unsigned long long*>(twt);  // entry [0][0] (tw = 1) is never read: the mbarrier lives there  // [RA][TWP]: tw[(q*j) % N] at j*TWP + q (odd pitch: 4 rows per warp, no conflicts)
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const bool io_thread = tid == (NW - 1) * 32;  // first lane of the last warp (idle in the radix-RA passes when RA > RB)
  const int i2 = blockIdx.x / g.ntz;
  const int z0 = (blockIdx.x - i2 * g.ntz) * FFT_C;
  double vv[RB];
#pragma unroll
  for (int q = 0; q < RB; ++q) vv[q] = __ldg(&g.vs[((size_t)(j + q * RA) * g.n2 + i2) * g.ldz + z0 + c]);
  for (int idx = tid; idx < RA * RA; idx += NT) {
    const int jj = idx / RA, q = idx - jj * RA;
    if (q > 0) twt[jj * TWP + q] = __ldg(&g.ax1.tw[(q * jj) % N]);
  }
  const int xhi = t.x_hi, xlo0 = N - t.x_lo, xsh = N - P;  // plane index of i1: i1 <= xhi ? i1 : (i1 >= xlo0 ? i1 - xsh : row P)
  const double2* twj = twt + j * TWP;
  if (tid < FFT_C) inb[(size_t)P * FFT_C + tid] = make_double2(0.0, 0.0);
  if (tid == 0) {
    mbar_init(full, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int cx = (i2 * g.ldz + z0) * 2;  // innermost tensor coordinate, in doubles
  auto issue_load = [&](int b) {
    mbar_expect_tx(full, (unsigned)P * ROWB);
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
                     smem_u32(inb)),
                 "l"(&tmap), "r"(cx), "r"(0), "r"(b), "r"(smem_u32(full))
                 : "memory");
  };
  auto issue_store = [&](int b) {
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%1, %2, %3}], [%4];" ::"l"(&tmap), "r"(cx), "r"(0),
                 "r"(b), "r"(smem_u32(outb))
                 : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
  };
  const int b0 = blockIdx.y, bstep = gridDim.y;
  if (io_thread && b0 < nb) issue_load(b0);
  int it = 0;
  for (int b = b0; b < nb; b += bstep, ++it) {
    if (j < RB) {
      mbar_wait(full, it & 1);
      double2 v[RA];
      const double2* in = inb + c;
#pragma unroll
      for (int q = 0; q < RA; ++q) {
        if (HALF && q >= QA && q < 3 * QA) continue;  // known zero
        const int i1 = j + q * RB;
        const int p = i1 <= xhi ? i1 : (i1 >= xlo0 ? i1 - xsh : P);
        v[q] = in[p * FFT_C];
      }
      if constexpr (HALF) {
        DftHalfIn<RA, +1>::run(v);
#pragma unroll
        for (int q = 0; q < RA; ++q) tile1[fft_phys(j * RA + q, c)] = v[q];
      } else
        pass_a_store<RA, +1>(v, tile1, j, c);
    }
    __syncthreads();
    if (io_thread) {
      if (b + bstep < nb) issue_load(b + bstep);  // the input stage was consumed before this barrier
      if (it > 0) issue_store(b - bstep);          // written by the previous iteration's last pass, fenced by its writers
    }
    {
      double2 u[RB];
#pragma unroll
      for (int q = 0; q < RB; ++q) u[q] = tile1[fft_phys(j + q * RA, c)];
#pragma unroll
      for (int q = 1; q < RB; ++q) u[q] = cmul(u[q], twj[q]);
      Dft<RB, +1>::run(u);
#pragma unroll
      for (int q = 0; q < RB; ++q) u[q] = make_double2(u[q].x * vv[q], u[q].y * vv[q]);
      Dft<RB, -1>::run(u);  // forward pass 1 = radix RB on the inputs j + q*RA this thread already holds
      if (one_tile) __syncthreads();  // every thread has read its tile1 entries: the tile can take the pass output
#pragma unroll
      for (int q = 0; q < RB; ++q) tile2[fft_phys(j * RB + q, c)] = u[q];
    }
    if (io_thread) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");  // output stage free before it is rewritten
    __syncthreads();
    double2 v[RA];
    if (j < RB) {
#pragma unroll
      for (int q = 0; q < RA; ++q) v[q] = tile2[fft_phys(j + q * RB, c)];
    }
    if (one_tile) __syncthreads();  // the tile has been read: the next band's first pass may overwrite it
    if (j < RB) {
#pragma unroll
      for (int q = 1; q < RA; ++q) v[q] = cmulc(v[q], twj[q]);
      Dft<RA, -1>::run(v);
      double2* out = outb + c;
#pragma unroll
      for (int q = 0; q < RA; ++q) {
        if (HALF && q >= QA && q < 3 * QA) continue;  // not a populated plane: never computed
        const int i1 = j + q * RB;
        const int p = i1 <= xhi ? i1 : (i1 >= xlo0 ? i1 - xsh : P);
        out[p * FFT_C] = v[q];
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy writes -> visible to the bulk store
    }
  }
  __syncthreads();
  if (io_thread && it > 0) {
    issue_store(b0 + (it - 1) * bstep);
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");  // shared memory must outlive the store's reads
  }
}


// NEXT-4 (charge density) with the same staging: inverse FFT along i1 as the first half of k2t_x_vmul, the tile of W2
// arriving by one TMA load per band (double-buffered: two input stages, loads issued one band ahead), then
// rho[i1][i2][i3] += scale * sum_b occ[b] |psi_b(r)|^2.  One CTA owns its (i2, i3 tile) pencils for all bands of the launch
// (gridDim.y must be 1): no atomics, bands summed in order, bit-reproducible.  Shared memory: fft2t_smem(n, P, true, true) + one stage.
inline size_t fft2t_smem_rho(int n, int P) {
  return (size_t)n * FFT_C * sizeof(double2) + 2 * (size_t)(P + 1) * FFT_C * sizeof(double2) + 16 * 17 * sizeof(double2) + 64;
}
template <int RA, int RB, bool HALF = false>
__global__ void __launch_bounds__(RA* FFT_C, 3)
k2t_x_rho(FftGeom g, Fft2pGeom t, const __grid_constant__ CUtensorMap tmap, int nb, const double* __restrict__ occ, double scale,
          double* __restrict__ rho) {
  static_assert(RB > 1 && RA >= RB && RA <= 16, "two-pass lengths with a [RA][RA+1] twiddle table");
  constexpr int N = RA * RB, NT = RA * FFT_C, NW = (NT + 31) / 32, TWP = RA + 1;
  constexpr unsigned ROWB = FFT_C * sizeof(double2);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* tile1 = reinterpret_cast<double2*>(smem_raw);
  const int P = g.P;
  double2* inb0 = tile1 + N * FFT_C;                   // two input stages of P + 1 rows (row P: zeros)
  double2* inb1 = inb0 + (size_t)(P + 1) * FFT_C;
  double2* twt = inb1 + (size_t)(P + 1) * FFT_C;
  unsigned long long* full = reinterpret_cast<unsigned long long*>(twt + RA * TWP);  // two mbarriers
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const bool io_thread = tid == (NW - 1) * 32;
  const int i2 = blockIdx.x / g.ntz;
  const int z0 = (blockIdx.x - i2 * g.ntz) * FFT_C;
  for (int idx = tid; idx < RA * RA; idx += NT) {
    const int jj = idx / RA, q = idx - jj * RA;
    twt[jj * TWP + q] = __ldg(&g.ax1.tw[(q * jj) % N]);
  }
  if (tid < 2 * FFT_C) (tid < FFT_C ? inb0 : inb1)[(size_t)P * FFT_C + (tid & (FFT_C - 1))] = make_double2(0.0, 0.0);
  const int xhi = t.x_hi, xlo0 = N - t.x_lo, xsh = N - P;
  const double2* twj = twt + j * TWP;
  if (tid == 0) {
    mbar_init(&full[0], 1);
    mbar_init(&full[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int cx = (i2 * g.ldz + z0) * 2;
  auto issue_load = [&](int b) {
    mbar_expect_tx(&full[b & 1], (unsigned)P * ROWB);
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
                     smem_u32((b & 1) ? inb1 : inb0)),
                 "l"(&tmap), "r"(cx), "r"(0), "r"(b), "r"(smem_u32(&full[b & 1]))
                 : "memory");
  };
  if (io_thread) {
    if (nb > 0) issue_load(0);
    if (nb > 1) issue_load(1);
  }
  double acc[RB];
#pragma unroll
  for (int q = 0; q < RB; ++q) acc[q] = 0.0;
  for (int b = 0; b < nb; ++b) {
    const double f = __ldg(&occ[b]);
    if (j < RB) {
      mbar_wait(&full[b & 1], (unsigned)(b >> 1) & 1u);
      double2 v[RA];
      const double2* in = ((b & 1) ? inb1 : inb0) + c;
#pragma unroll
      for (int q = 0; q < RA; ++q) {
        if (HALF && q >= RA / 4 && q < 3 * (RA / 4)) continue;  // known zero (quarter pruning, see k2t_x_vmul)
        const int i1 = j + q * RB;
        const int p = i1 <= xhi ? i1 : (i1 >= xlo0 ? i1 - xsh : P);
        v[q] = in[p * FFT_C];
      }
      if constexpr (HALF) {
        DftHalfIn<RA, +1>::run(v);
#pragma unroll
        for (int q = 0; q < RA; ++q) tile1[fft_phys(j * RA + q, c)] = v[q];
      } else
        pass_a_store<RA, +1>(v, tile1, j, c);
    }
    __syncthreads();  // tile complete; the input stage of band b has been read by everybody
    if (io_thread && b + 2 < nb) issue_load(b + 2);
    double2 u[RB];
#pragma unroll
    for (int q = 0; q < RB; ++q) u[q] = tile1[fft_phys(j + q * RA, c)];
#pragma unroll
    for (int q = 1; q < RB; ++q) u[q] = cmul(u[q], twj[q]);
    Dft<RB, +1>::run(u);
#pragma unroll
    for (int q = 0; q < RB; ++q) acc[q] += f * (u[q].x * u[q].x + u[q].y * u[q].y);
    __syncthreads();  // the next band's first pass overwrites tile1
  }
  const int z = z0 + c;
  if (z < g.n3) {
#pragma unroll
    for (int q = 0; q < RB; ++q) {
      double* r = rho + ((size_t)(j + q * RA) * g.n2 + i2) * g.n3 + z;
      *r += scale * acc[q];
    }
  }
}

// three-pass variant (lengths of fft3p_kernels.cuh): same staging, arithmetic of k3p_x_vmul
template <int R1, int R2, int R3>
__global__ void __launch_bounds__(P3<R1, R2, R3>::NT) k3t_x_vmul(FftGeom g, Fft2pGeom t, const __grid_constant__ CUtensorMap tmap,
                                                                int nb, int /*one_tile: two-pass kernel only*/) {
  using PP = P3<R1, R2, R3>;
  constexpr int N = PP::N, NT = PP::NT, NW = (NT + 31) / 32;
  constexpr unsigned ROWB = FFT_C * sizeof(double2);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* tA = reinterpret_cast<double2*>(smem_raw);
  double2* tB = tA + N * FFT_C;
  double2* inb = tB + N * FFT_C;
  const int P = g.P;
  double2* outb = inb + (size_t)P * FFT_C;
  unsigned long long* full = reinterpret_cast<unsigned long long*>(outb + (size_t)P * FFT_C);
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const bool io_thread = tid == (NW - 1) * 32;
  const int i2 = blockIdx.x / g.ntz;
  const int z0 = (blockIdx.x - i2 * g.ntz) * FFT_C;
  const double2 zero = make_double2(0.0, 0.0);
  double vv[R3];
  if (j < PP::T3) {
#pragma unroll
    for (int q = 0; q < R3; ++q) vv[q] = __ldg(&g.vs[((size_t)(j + q * PP::T3) * g.n2 + i2) * g.ldz + z0 + c]);
  }
  int pl[R1];
  if (j < PP::T1) {
#pragma unroll
    for (int q = 0; q < R1; ++q) pl[q] = __ldg(&t.plane_of[j + q * PP::T1]);
  }
  if (tid == 0) {
    mbar_init(full, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int cx = (i2 * g.ldz + z0) * 2;
  auto issue_load = [&](int b) {
    mbar_expect_tx(full, (unsigned)P * ROWB);
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
                     smem_u32(inb)),
                 "l"(&tmap), "r"(cx), "r"(0), "r"(b), "r"(smem_u32(full))
                 : "memory");
  };
  auto issue_store = [&](int b) {
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%1, %2, %3}], [%4];" ::"l"(&tmap), "r"(cx), "r"(0),
                 "r"(b), "r"(smem_u32(outb))
                 : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
  };
  const int b0 = blockIdx.y, bstep = gridDim.y;
  if (io_thread && b0 < nb) issue_load(b0);
  int it = 0;
  for (int b = b0; b < nb; b += bstep, ++it) {
    if (j < PP::T1) {
      mbar_wait(full, it & 1);
      double2 v[R1];
      const double2* in = inb + c;
#pragma unroll
      for (int q = 0; q < R1; ++q) v[q] = pl[q] >= 0 ? in[pl[q] * FFT_C] : zero;
      pass_a_store<R1, +1>(v, tA, j, c);
    }
    __syncthreads();
    if (io_thread) {
      if (b + bstep < nb) issue_load(b + bstep);
      if (it > 0) issue_store(b - bstep);
    }
    if (j < PP::T2) pass_mid<R2, +1>(tA, tB, g.ax1.tw, N, R1, j, c);
    __syncthreads();
    if (j < PP::T3) {
      double2 u[R3];
      pass_b_load<PP::T3, R3, +1>(tB, g.ax1.tw, j, c, u);
#pragma unroll
      for (int q = 0; q < R3; ++q) u[q] = make_double2(u[q].x * vv[q], u[q].y * vv[q]);
      pass_a_store<R3, -1>(u, tA, j, c);
    }
    __syncthreads();
    if (j < PP::T2) pass_mid<R2, -1>(tA, tB, g.ax1.tw, N, R3, j, c);
    if (io_thread) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    __syncthreads();
    if (j < PP::T1) {
      double2 v[R1];
      pass_b_load<PP::T1, R1, -1>(tB, g.ax1.tw, j, c, v);
      double2* out = outb + c;
#pragma unroll
      for (int q = 0; q < R1; ++q)
        if (pl[q] >= 0) out[pl[q] * FFT_C] = v[q];
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
  }
  __syncthreads();
  if (io_thread && it > 0) {
    issue_store(b0 + (it - 1) * bstep);
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
  }
}


// ---------------------------------------------------------------------------------------------------------
// z stages (a1, a5) with bulk-copy staging of the W1 side: the 8 sticks of a tile are 8 contiguous rows of W1, so the tile
// moves as eight 1-D bulk copies of N*16 bytes instead of 16-byte accesses at a row stride (lanes run across sticks).
// Stage layout [stick c][N + 1] complex (odd pitch: the 8 lanes of a quarter warp hit 8 different 16-byte bank groups).
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void bulk_s2g(void* gdst, const void* ssrc, unsigned bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(ssrc)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* sdst, const void* gsrc, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(sdst)),
               "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
inline size_t fft2t_smem_z(int n) { return ((size_t)n * FFT_C + (size_t)FFT_C * (n + 1)) * sizeof(double2) + 64; }

// a1: psi(G) -> z sticks, inverse FFT along i3 -> W1 (bulk stores)
template <int RA, int RB>
__global__ void __launch_bounds__(RA* FFT_C) k2t_scatter_zinv(FftGeom g, Fft2pGeom t, const double2* __restrict__ psi,
                                                              long long ldpsi, double2* __restrict__ w1) {
  static_assert(RB > 1, "single-pass lengths use k2p_scatter_zinv");
  constexpr int N = RA * RB, PITCH = N + 1;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* tile = reinterpret_cast<double2*>(smem_raw);
  double2* stage = tile + N * FFT_C;  // [FFT_C][PITCH]
  unsigned long long* full = reinterpret_cast<unsigned long long*>(stage + FFT_C * PITCH);
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const int b = blockIdx.y;
  const int s0 = blockIdx.x * FFT_C, s = s0 + c;
  const bool sok = s < g.S;
  const double2 zero = make_double2(0.0, 0.0);
  // the sphere entries of the tile's sticks are one contiguous chunk of psi (canonical order): one bulk load
  const int base = g.stick_start[s0], cnt = g.stick_start[min(s0 + FFT_C, g.S)] - base;
  if (tid == 0) {
    mbar_init(full, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if (cnt > 0) {
      mbar_expect_tx(full, (unsigned)(cnt * sizeof(double2)));
      bulk_g2s(stage, psi + (size_t)b * ldpsi + base, (unsigned)(cnt * sizeof(double2)), full);
    }
  }
  __syncthreads();
  if (j < RB) {
    double2 v[RA];
    if (sok) {
      const int start = g.stick_start[s] - base, lo = t.stick_lo[s], hi = t.stick_hi[s];
      if (cnt > 0) mbar_wait(full, 0);
#pragma unroll
      for (int q = 0; q < RA; ++q) {
        const int pos = stick_pos(start, lo, hi, j + q * RB, N);
        v[q] = pos >= 0 ? stage[pos] : zero;
      }
    } else {
#pragma unroll
      for (int q = 0; q < RA; ++q) v[q] = zero;
    }
    pass_a_store<RA, +1>(v, tile, j, c);
  }
  __syncthreads();
  {
    double2 u[RB];
    pass_b_load<RA, RB, +1>(tile, g.ax3.tw, j, c, u);
    double2* out = stage + c * PITCH + j;
#pragma unroll
    for (int q = 0; q < RB; ++q) out[q * RA] = u[q];
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  if (tid < FFT_C && s0 + tid < g.S) {
    bulk_s2g(w1 + ((size_t)b * g.S + s0 + tid) * g.ldz, stage + tid * PITCH, (unsigned)(N * sizeof(double2)));
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");  // shared memory must outlive the store's reads
  }
}

// a5: W1 (bulk loads) -> forward FFT along i3, gather the sphere, add g2kin*psi -> hpsi
template <int RA, int RB>
__global__ void __launch_bounds__(RA* FFT_C) k2t_zfwd_gather(FftGeom g, Fft2pGeom t, const double2* __restrict__ w1,
                                                             const double2* __restrict__ psi, long long ldpsi,
                                                             double2* __restrict__ hpsi, long long ldh) {
  static_assert(RB > 1, "single-pass lengths use k2p_zfwd_gather");
  constexpr int N = RA * RB, PITCH = N + 1;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* tile = reinterpret_cast<double2*>(smem_raw);
  double2* stage = tile + N * FFT_C;
  unsigned long long* full = reinterpret_cast<unsigned long long*>(stage + FFT_C * PITCH);
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const int b = blockIdx.y;
  const int s0 = blockIdx.x * FFT_C, s = s0 + c;
  const int nst = min(FFT_C, g.S - s0);
  const bool sok = s < g.S;
  const double2 zero = make_double2(0.0, 0.0);
  if (tid == 0) {
    mbar_init(full, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0) mbar_expect_tx(full, (unsigned)(nst * N * sizeof(double2)));
  __syncthreads();
  if (tid < nst) bulk_g2s(stage + tid * PITCH, w1 + ((size_t)b * g.S + s0 + tid) * g.ldz, (unsigned)(N * sizeof(double2)), full);
  int start = 0, lo = 1, hi = 0;
  if (sok) {
    start = g.stick_start[s];
    lo = t.stick_lo[s];
    hi = t.stick_hi[s];
  }
  const double2* pb = psi + (size_t)b * ldpsi;
  double2* hb = hpsi + (size_t)b * ldh;
  {
    // the sphere entries of the tile's sticks are one contiguous chunk of psi / g2kin (canonical order): pull it towards L2 now,
    // while the W1 rows are in flight, so that the kinetic-term reads after the transform do not pay a second DRAM latency
    const int base = g.stick_start[s0], cnt = g.stick_start[min(s0 + FFT_C, g.S)] - base;
    for (int i = tid * 8; i < cnt; i += RA * FFT_C * 8) {
      asm volatile("prefetch.global.L2 [%0];" ::"l"(pb + base + i));
      if ((i & 8) == 0) asm volatile("prefetch.global.L2 [%0];" ::"l"(g.g2kin + base + i));
    }
  }
  if (j < RB) {
    mbar_wait(full, 0);
    double2 v[RA];
    const double2* in = stage + c * PITCH;
#pragma unroll
    for (int q = 0; q < RA; ++q) v[q] = sok ? in[j + q * RB] : zero;
    pass_a_store<RA, -1>(v, tile, j, c);
  }
  __syncthreads();
  {
    double2 u[RB];
    pass_b_load<RA, RB, -1>(tile, g.ax3.tw, j, c, u);
#pragma unroll
    for (int q = 0; q < RB; ++q) {
      const int pos = stick_pos(start, lo, hi, j + q * RA, N);
      if (pos >= 0) {
        const double2 cpsi = pb[pos];
        const double k2 = __ldg(&g.g2kin[pos]);
        hb[pos] = make_double2(u[q].x + k2 * cpsi.x, u[q].y + k2 * cpsi.y);
      }
    }
  }
}

using K2tX = void (*)(FftGeom, Fft2pGeom, const CUtensorMap, int, int);

using K2tRho = void (*)(FftGeom, Fft2pGeom, const CUtensorMap, int, const double*, double, double*);
template <int RA, int RB>
constexpr K2tRho rho_half_kernel() {
  if constexpr (RA % 4 == 0)
    return k2t_x_rho<RA, RB, true>;
  else
    return nullptr;
}
template <int RA, int RB>
constexpr K2tX x_half_kernel() {
  if constexpr (RA % 4 == 0)
    return k2t_x_vmul<RA, RB, true>;
  else
    return nullptr;
}
struct Fft2tEntry {
  int n, ra, rb;
  K2tRho rho;    // TMA-staged density kernel (two-pass lengths only)
  K2tRho rhoh;   // the two with quarter pruning (RA % 4 == 0, populated planes in the outer quarters of the axis), else null
  K2tX xh;
  K2tX x;
  K2pZinv zinv;  // bulk-staged z stages (two-pass lengths only; null for the three-pass table)
  K2pZfwd zfwd;
};
#define QE_FFT2T_ENTRY(RA, RB) {(RA) * (RB), RA, RB, k2t_x_rho<RA, RB>, rho_half_kernel<RA, RB>(), x_half_kernel<RA, RB>(), k2t_x_vmul<RA, RB>, k2t_scatter_zinv<RA, RB>, k2t_zfwd_gather<RA, RB>}
static const Fft2tEntry kFft2tTable[] = {
    QE_FFT2T_ENTRY(6, 3),   QE_FFT2T_ENTRY(5, 4),   QE_FFT2T_ENTRY(6, 6),   QE_FFT2T_ENTRY(8, 6),   QE_FFT2T_ENTRY(8, 8),
    QE_FFT2T_ENTRY(9, 8),   QE_FFT2T_ENTRY(10, 8),  QE_FFT2T_ENTRY(12, 8),  QE_FFT2T_ENTRY(10, 10), QE_FFT2T_ENTRY(12, 9),
    QE_FFT2T_ENTRY(12, 10), QE_FFT2T_ENTRY(16, 8),  QE_FFT2T_ENTRY(12, 12), QE_FFT2T_ENTRY(16, 10), QE_FFT2T_ENTRY(15, 12),
    QE_FFT2T_ENTRY(16, 12), QE_FFT2T_ENTRY(16, 15), QE_FFT2T_ENTRY(16, 16),
};
#undef QE_FFT2T_ENTRY
// three-pass lengths: ra = R1, rb = R2*R3 as in kFft3pTable
#define QE_FFT3T_ENTRY(R1, R2, R3) {(R1) * (R2) * (R3), R1, (R2) * (R3), nullptr, nullptr, nullptr, k3t_x_vmul<R1, R2, R3>, nullptr, nullptr}
static const Fft2tEntry kFft3tTable[] = {
    QE_FFT3T_ENTRY(5, 5, 5),  QE_FFT3T_ENTRY(6, 5, 5),  QE_FFT3T_ENTRY(8, 5, 5),  QE_FFT3T_ENTRY(6, 6, 6), QE_FFT3T_ENTRY(10, 5, 5),
    QE_FFT3T_ENTRY(8, 6, 6),  QE_FFT3T_ENTRY(10, 6, 5), QE_FFT3T_ENTRY(8, 8, 5),  QE_FFT3T_ENTRY(10, 6, 6), QE_FFT3T_ENTRY(8, 8, 6),
};
#undef QE_FFT3T_ENTRY
// the (RA, RB) pair must be the one the two-pass table uses for this length (same thread layout and tables)
inline const Fft2tEntry* fft2t_find(int n, int ra, int rb, bool three_pass) {
  if (three_pass) {
    for (const Fft2tEntry& e : kFft3tTable)
      if (e.n == n && e.ra == ra && e.rb == rb) return &e;
    return nullptr;
  }
  for (const Fft2tEntry& e : kFft2tTable)
    if (e.n == n && e.ra == ra && e.rb == rb) return &e;
  return nullptr;
}

}  // namespace qehpsi
