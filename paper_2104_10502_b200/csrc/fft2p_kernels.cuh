// fft2p_kernels.cuh -- fast path of the local term (steps a1-a5) for FFT lengths that factor
// as N = RA * RB with register-resident radices (RA >= RB, RB may be 1).  Same five pruned pencil passes as
// fft_kernels.cuh (the generic path), but every 1-D transform is exactly two butterfly passes:
//     global -> registers -> radix-RA DFT -> shared tile -> twiddle + radix-RB DFT in registers -> global
// i.e. one shared-memory round trip and one barrier per transform, no zero-fill pass (unpopulated inputs are
// predicated loads), and the x stage keeps the data in registers across  iFFT -> * V(r)/N -> FFT  (the inverse
// ends with radix RB on inputs j + q*RA, which is exactly what a forward transform that starts with radix RB
// consumes).  The paper states only that the FFTs go through 1-D and 2-D transforms and that
// plane waves are mapped to FFT grids (PAPER.md:L176 (vi)).
#pragma once
#include "fft_kernels.cuh"

namespace qehpsi {

// extra tables of the fast path (all device pointers)
struct Fft2pGeom {
  const int* stick_lo;    // [S] lowest signed Miller index n3 of the stick's sphere points
  const int* stick_hi;    // [S] highest
  const int* col_of;      // [P][N2] stick index of column (plane p, i2), or -1
  const int* plane_of;    // [N1] populated-plane index of i1, or -1
  // the populated i1 planes of a convex sphere are the wrapped interval [0..x_hi] u [N1-x_lo..N1-1] (x_hi = -1 / x_lo = 0:
  // that part is empty) in this order, so plane_of[i1] = i1, resp. i1 - (N1 - P); x_hi = -2 when the pattern does not hold
  int x_hi, x_lo;
  // same rule per populated plane p for its sticks along i2: i2 in [0..y_hi[p]] u [N2-y_lo[p]..N2-1] are the plane's sticks
  // plane_stick[p] + i2, resp. plane_stick[p] + i2 - (N2 - count); y_hi == nullptr when the pattern does not hold (table lookup)
  const int* y_hi;
  const int* y_lo;
  const double2* zrow;  // ldz zeros: what an unpopulated (plane, i2) column reads, so that the loads need no branch
};

// shared tile [N][FFT_C] with the column XOR swizzle of fft_core.cuh (fft_phys)

// first pass of a two-pass transform: v[q] = x[j + q*RB], q < RA, already in registers -> radix-RA DFT -> tile.
// Stockham with Ns = 1: no twiddles, outputs at j*RA + q.
template <int RA, int DIR>
__device__ __forceinline__ void pass_a_store(double2 (&v)[RA], double2* __restrict__ tile, int j, int c) {
  Dft<RA, DIR>::run(v);
#pragma unroll
  for (int q = 0; q < RA; ++q) tile[fft_phys(j * RA + q, c)] = v[q];
}

// second pass: task j < RA reads tile[j + q*RA], q < RB, multiplies by exp(DIR 2 pi i q j / N) and runs the
// radix-RB DFT; result v[q] is X[j + q*RA].
template <int RA, int RB, int DIR>
__device__ __forceinline__ void pass_b_load(const double2* __restrict__ tile, const double2* __restrict__ tw, int j, int c,
                                            double2 (&v)[RB]) {
#pragma unroll
  for (int q = 0; q < RB; ++q) v[q] = tile[fft_phys(j + q * RA, c)];
#pragma unroll
  for (int q = 1; q < RB; ++q) {
    const double2 w = __ldg(&tw[q * j]);
    v[q] = DIR > 0 ? cmul(v[q], w) : cmulc(v[q], w);
  }
  Dft<RB, DIR>::run(v);
}

// position inside psi of the sphere point (stick with run start `start`, signed range [lo, hi]) at wrapped i3,
// or -1.  Canonical order inside a stick = ascending wrapped index: n3 = 0..hi first, then lo..-1.
__device__ __forceinline__ int stick_pos(int start, int lo, int hi, int i3, int n3grid) {
  const int n3 = i3 >= (n3grid + 1) / 2 ? i3 - n3grid : i3;
  if (n3 < lo || n3 > hi) return -1;
  const int lo_pos = max(lo, 0);
  if (n3 >= 0) return start + (n3 - lo_pos);
  const int npos = max(hi - lo_pos + 1, 0);
  return start + npos + (n3 - lo);
}

// a1 ------------------------------------------------------------------------------------------------------
// psi(G) -> z sticks (predicated loads straight from psi), inverse FFT along i3 -> W1[b][s][ldz]
template <int RA, int RB>
__global__ void __launch_bounds__(RA* FFT_C) k2p_scatter_zinv(FftGeom g, Fft2pGeom t, const double2* __restrict__ psi,
                                                              long long ldpsi, double2* __restrict__ w1) {
  constexpr int N = RA * RB;
  __shared__ __align__(16) double2 tile[RB > 1 ? N * FFT_C : 1];
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const int b = blockIdx.y;
  const int s = blockIdx.x * FFT_C + c;
  const bool sok = s < g.S;
  const double2 zero = make_double2(0.0, 0.0);
  if (j < RB) {
    double2 v[RA];
    if (sok) {
      const int start = g.stick_start[s], lo = t.stick_lo[s], hi = t.stick_hi[s];
      const double2* pb = psi + (size_t)b * ldpsi;
#pragma unroll
      for (int q = 0; q < RA; ++q) {
        const int pos = stick_pos(start, lo, hi, j + q * RB, N);
        v[q] = pos >= 0 ? pb[pos] : zero;
      }
    } else {
#pragma unroll
      for (int q = 0; q < RA; ++q) v[q] = zero;
    }
    if constexpr (RB > 1) {
      pass_a_store<RA, +1>(v, tile, j, c);
    } else {
      Dft<RA, +1>::run(v);
      if (sok) {
        double2* out = w1 + ((size_t)b * g.S + s) * g.ldz;
#pragma unroll
        for (int q = 0; q < RA; ++q) out[q] = v[q];
      }
    }
  }
  if constexpr (RB > 1) {
    __syncthreads();
    double2 u[RB];
    pass_b_load<RA, RB, +1>(tile, g.ax3.tw, j, c, u);
    if (sok) {
      double2* out = w1 + ((size_t)b * g.S + s) * g.ldz + j;
#pragma unroll
      for (int q = 0; q < RB; ++q) out[q * RA] = u[q];
    }
  }
}

// a5 ------------------------------------------------------------------------------------------------------
// forward FFT along i3 on the sticks, gather the sphere, add g2kin*psi -> hpsi
template <int RA, int RB>
__global__ void __launch_bounds__(RA* FFT_C) k2p_zfwd_gather(FftGeom g, Fft2pGeom t, const double2* __restrict__ w1,
                                                             const double2* __restrict__ psi, long long ldpsi,
                                                             double2* __restrict__ hpsi, long long ldh) {
  constexpr int N = RA * RB;
  __shared__ __align__(16) double2 tile[RB > 1 ? N * FFT_C : 1];
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const int b = blockIdx.y;
  const int s = blockIdx.x * FFT_C + c;
  const bool sok = s < g.S;
  const double2 zero = make_double2(0.0, 0.0);
  int start = 0, lo = 1, hi = 0;
  if (sok) {
    start = g.stick_start[s];
    lo = t.stick_lo[s];
    hi = t.stick_hi[s];
  }
  const double2* pb = psi + (size_t)b * ldpsi;
  double2* hb = hpsi + (size_t)b * ldh;
  auto emit = [&](int i3, double2 x) {
    const int pos = stick_pos(start, lo, hi, i3, N);
    if (pos >= 0) {
      const double2 cpsi = pb[pos];
      const double k2 = __ldg(&g.g2kin[pos]);
      hb[pos] = make_double2(x.x + k2 * cpsi.x, x.y + k2 * cpsi.y);
    }
  };
  if (j < RB) {
    double2 v[RA];
    const double2* in = w1 + ((size_t)b * g.S + (sok ? s : 0)) * g.ldz;
#pragma unroll
    for (int q = 0; q < RA; ++q) v[q] = sok ? in[j + q * RB] : zero;
    if constexpr (RB > 1) {
      pass_a_store<RA, -1>(v, tile, j, c);
    } else {
      Dft<RA, -1>::run(v);
#pragma unroll
      for (int q = 0; q < RA; ++q) emit(q, v[q]);
    }
  }
  if constexpr (RB > 1) {
    __syncthreads();
    double2 u[RB];
    pass_b_load<RA, RB, -1>(tile, g.ax3.tw, j, c, u);
#pragma unroll
    for (int q = 0; q < RB; ++q) emit(j + q * RA, u[q]);
  }
}

// a2 ------------------------------------------------------------------------------------------------------
// per populated plane p and i3 tile: inverse FFT along i2 over the plane's sticks -> W2[b][p][N2][ldz]
template <int RA, int RB>
__global__ void __launch_bounds__(RA* FFT_C) k2p_yinv(FftGeom g, Fft2pGeom t, const double2* __restrict__ w1,
                                                      double2* __restrict__ w2) {
  constexpr int N = RA * RB;
  __shared__ __align__(16) double2 tile[RB > 1 ? N * FFT_C : 1];
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const int b = blockIdx.y;
  const int p = blockIdx.x / g.ntz;
  const int z = (blockIdx.x - p * g.ntz) * FFT_C + c;  // < ldz always (ldz is a multiple of FFT_C)
  const double2 zero = make_double2(0.0, 0.0);
  const double2* in = w1 + (size_t)b * g.S * g.ldz + z;
  double2* out = w2 + ((size_t)b * g.P + p) * N * g.ldz + z;
  const int* col = t.col_of + (size_t)p * N;
  if (j < RB) {
    double2 v[RA];
    if (t.y_hi != nullptr) {
      // stick of column i2 by the wrapped-interval rule (three scalars per plane) instead of a dependent table lookup per
      // column; unpopulated columns read the zero row: sixteen independent, unconditional loads
      const int s0 = __ldg(&g.plane_stick[p]), yhi = __ldg(&t.y_hi[p]), ylo0 = N - __ldg(&t.y_lo[p]);
      const int ysh = N - (__ldg(&g.plane_stick[p + 1]) - s0);
      const double2* zr = t.zrow + z;
#pragma unroll
      for (int q = 0; q < RA; ++q) {
        const int i2 = j + q * RB;
        const int s = s0 + (i2 <= yhi ? i2 : i2 - ysh);
        const double2* src = (i2 <= yhi || i2 >= ylo0) ? in + (size_t)s * g.ldz : zr;
        v[q] = *src;
      }
    } else {
#pragma unroll
      for (int q = 0; q < RA; ++q) {
        const int s = __ldg(&col[j + q * RB]);
        v[q] = s >= 0 ? in[(size_t)s * g.ldz] : zero;
      }
    }
    if constexpr (RB > 1) {
      pass_a_store<RA, +1>(v, tile, j, c);
    } else {
      Dft<RA, +1>::run(v);
#pragma unroll
      for (int q = 0; q < RA; ++q) out[(size_t)q * g.ldz] = v[q];
    }
  }
  if constexpr (RB > 1) {
    __syncthreads();
    double2 u[RB];
    pass_b_load<RA, RB, +1>(tile, g.ax2.tw, j, c, u);
#pragma unroll
    for (int q = 0; q < RB; ++q) out[(size_t)(j + q * RA) * g.ldz] = u[q];
  }
}

// a4 ------------------------------------------------------------------------------------------------------
// forward FFT along i2, keep only the stick columns -> W1
template <int RA, int RB>
__global__ void __launch_bounds__(RA* FFT_C) k2p_yfwd(FftGeom g, Fft2pGeom t, const double2* __restrict__ w2,
                                                      double2* __restrict__ w1) {
  constexpr int N = RA * RB;
  __shared__ __align__(16) double2 tile[RB > 1 ? N * FFT_C : 1];
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const int b = blockIdx.y;
  const int p = blockIdx.x / g.ntz;
  const int z = (blockIdx.x - p * g.ntz) * FFT_C + c;
  const double2* in = w2 + ((size_t)b * g.P + p) * N * g.ldz + z;
  double2* out = w1 + (size_t)b * g.S * g.ldz + z;
  const int* col = t.col_of + (size_t)p * N;
  if (j < RB) {
    double2 v[RA];
#pragma unroll
    for (int q = 0; q < RA; ++q) v[q] = in[(size_t)(j + q * RB) * g.ldz];
    if constexpr (RB > 1) {
      pass_a_store<RA, -1>(v, tile, j, c);
    } else {
      Dft<RA, -1>::run(v);
#pragma unroll
      for (int q = 0; q < RA; ++q) {
        const int s = __ldg(&col[q]);
        if (s >= 0) out[(size_t)s * g.ldz] = v[q];
      }
    }
  }
  if constexpr (RB > 1) {
    __syncthreads();
    double2 u[RB];
    pass_b_load<RA, RB, -1>(tile, g.ax2.tw, j, c, u);
#pragma unroll
    for (int q = 0; q < RB; ++q) {
      const int s = __ldg(&col[j + q * RA]);
      if (s >= 0) out[(size_t)s * g.ldz] = u[q];
    }
  }
}

// a3 ------------------------------------------------------------------------------------------------------
// per (i2, i3 tile): inverse FFT along i1 over the P populated planes, * V(r)/N, forward FFT along i1, keep the
// populated planes.  The CTA keeps its V values in registers and loops over bands b = blockIdx.y, +gridDim.y, ...
// Dynamic shared memory: two [N][FFT_C] tiles (none when RB == 1).
template <int RA, int RB>
__global__ void __launch_bounds__(RA* FFT_C) k2p_x_vmul(FftGeom g, Fft2pGeom t, double2* __restrict__ w2, int nb) {
  constexpr int N = RA * RB;
  constexpr int NV = RB > 1 ? RB : RA;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* tile1 = reinterpret_cast<double2*>(smem_raw);
  double2* tile2 = tile1 + N * FFT_C;
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const int i2 = blockIdx.x / g.ntz;
  const int z = (blockIdx.x - i2 * g.ntz) * FFT_C + c;
  const double2 zero = make_double2(0.0, 0.0);
  const size_t pstride = (size_t)g.n2 * g.ldz;
  // V(r)/N at the points this thread holds after the inverse transform: i1 = j + q*RA (RB > 1) or q (RB == 1)
  double vv[NV];
#pragma unroll
  for (int q = 0; q < NV; ++q) {
    const int i1 = RB > 1 ? j + q * RA : q;
    vv[q] = __ldg(&g.vs[((size_t)i1 * g.n2 + i2) * g.ldz + z]);
  }
  // populated-plane index of the inputs / final outputs of this thread: i1 = j + q*RB
  int pl[RA];
  if (j < RB) {
#pragma unroll
    for (int q = 0; q < RA; ++q) pl[q] = __ldg(&t.plane_of[j + q * RB]);
  }
  for (int b = blockIdx.y; b < nb; b += gridDim.y) {
    double2* io = w2 + ((size_t)b * g.P * g.n2 + i2) * g.ldz + z;
    if constexpr (RB > 1) {
      if (j < RB) {
        double2 v[RA];
#pragma unroll
        for (int q = 0; q < RA; ++q) v[q] = pl[q] >= 0 ? io[pl[q] * pstride] : zero;
        pass_a_store<RA, +1>(v, tile1, j, c);
      }
      __syncthreads();
      {
        double2 u[RB];
        pass_b_load<RA, RB, +1>(tile1, g.ax1.tw, j, c, u);
#pragma unroll
        for (int q = 0; q < RB; ++q) u[q] = make_double2(u[q].x * vv[q], u[q].y * vv[q]);
        // forward transform, first pass = radix RB on the inputs j + q*RA this thread already holds
        Dft<RB, -1>::run(u);
#pragma unroll
        for (int q = 0; q < RB; ++q) tile2[fft_phys(j * RB + q, c)] = u[q];
      }
      __syncthreads();
      if (j < RB) {
        double2 v[RA];
        pass_b_load<RB, RA, -1>(tile2, g.ax1.tw, j, c, v);
#pragma unroll
        for (int q = 0; q < RA; ++q)
          if (pl[q] >= 0) io[pl[q] * pstride] = v[q];
      }
    } else {
      if (j < 1) {
        double2 v[RA];
#pragma unroll
        for (int q = 0; q < RA; ++q) v[q] = pl[q] >= 0 ? io[pl[q] * pstride] : zero;
        Dft<RA, +1>::run(v);
#pragma unroll
        for (int q = 0; q < RA; ++q) v[q] = make_double2(v[q].x * vv[q], v[q].y * vv[q]);
        Dft<RA, -1>::run(v);
#pragma unroll
        for (int q = 0; q < RA; ++q)
          if (pl[q] >= 0) io[pl[q] * pstride] = v[q];
      }
    }
  }
}

// NEXT-4 (charge density) ----------------------------------------------------------------------
// inverse FFT along i1 exactly as the first half of a3, then rho[i1][i2][i3] += scale * sum_b occ[b] |psi_b(r)|^2.
// One CTA owns its (i2, i3 tile) pencils for all bands of the launch (gridDim.y must be 1): no atomics, fixed order.
template <int RA, int RB>
__global__ void __launch_bounds__(RA* FFT_C) k2p_x_rho(FftGeom g, Fft2pGeom t, const double2* __restrict__ w2, int nb,
                                                       const double* __restrict__ occ, double scale,
                                                       double* __restrict__ rho) {
  constexpr int N = RA * RB;
  constexpr int NV = RB > 1 ? RB : RA;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* tile1 = reinterpret_cast<double2*>(smem_raw);
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const int i2 = blockIdx.x / g.ntz;
  const int z = (blockIdx.x - i2 * g.ntz) * FFT_C + c;
  const double2 zero = make_double2(0.0, 0.0);
  const size_t pstride = (size_t)g.n2 * g.ldz;
  int pl[RA];
  if (j < RB) {
#pragma unroll
    for (int q = 0; q < RA; ++q) pl[q] = __ldg(&t.plane_of[j + q * RB]);
  }
  double acc[NV];
#pragma unroll
  for (int q = 0; q < NV; ++q) acc[q] = 0.0;
  for (int b = 0; b < nb; ++b) {
    const double f = __ldg(&occ[b]);
    const double2* in = w2 + ((size_t)b * g.P * g.n2 + i2) * g.ldz + z;
    if constexpr (RB > 1) {
      if (j < RB) {
        double2 v[RA];
#pragma unroll
        for (int q = 0; q < RA; ++q) v[q] = pl[q] >= 0 ? in[pl[q] * pstride] : zero;
        pass_a_store<RA, +1>(v, tile1, j, c);
      }
      __syncthreads();
      double2 u[RB];
      pass_b_load<RA, RB, +1>(tile1, g.ax1.tw, j, c, u);
#pragma unroll
      for (int q = 0; q < RB; ++q) acc[q] += f * (u[q].x * u[q].x + u[q].y * u[q].y);
      __syncthreads();  // the next band's first pass overwrites tile1
    } else {
      if (j < 1) {
        double2 v[RA];
#pragma unroll
        for (int q = 0; q < RA; ++q) v[q] = pl[q] >= 0 ? in[pl[q] * pstride] : zero;
        Dft<RA, +1>::run(v);
#pragma unroll
        for (int q = 0; q < RA; ++q) acc[q] += f * (v[q].x * v[q].x + v[q].y * v[q].y);
      }
    }
  }
  if (z < g.n3 && (RB > 1 || j < 1)) {
#pragma unroll
    for (int q = 0; q < NV; ++q) {
      const int i1 = RB > 1 ? j + q * RA : q;
      double* r = rho + ((size_t)i1 * g.n2 + i2) * g.n3 + z;
      *r += scale * acc[q];
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// dispatch: one entry per supported length N = RA * RB
// ---------------------------------------------------------------------------------------------------------
using K2pZinv = void (*)(FftGeom, Fft2pGeom, const double2*, long long, double2*);
using K2pZfwd = void (*)(FftGeom, Fft2pGeom, const double2*, const double2*, long long, double2*, long long);
using K2pY = void (*)(FftGeom, Fft2pGeom, const double2*, double2*);
using K2pX = void (*)(FftGeom, Fft2pGeom, double2*, int);
using K2pRho = void (*)(FftGeom, Fft2pGeom, const double2*, int, const double*, double, double*);

struct Fft2pEntry {
  int n, ra, rb;
  int nthreads;    // CTA size of all five kernels
  size_t smem_zy;  // dynamic shared memory of the z and y kernels (0: static tiles)
  size_t smem_x;   // dynamic shared memory of the x kernel
  K2pZinv zinv;
  K2pZfwd zfwd;
  K2pY yinv, yfwd;
  K2pX x;
  K2pRho rho;      // NEXT-4: x-inverse + density accumulation (dynamic shared memory: smem_x / 2)
};

#define QE_FFT2P_ENTRY(RA, RB)                                                                                  \
  {                                                                                                             \
    (RA) * (RB), RA, RB, (RA) * FFT_C, 0, (RB) > 1 ? 2 * (size_t)(RA) * (RB) * FFT_C * sizeof(double2) : 0,     \
        k2p_scatter_zinv<RA, RB>, k2p_zfwd_gather<RA, RB>, k2p_yinv<RA, RB>, k2p_yfwd<RA, RB>, k2p_x_vmul<RA, RB>, \
        k2p_x_rho<RA, RB>                                                                                        \
  }

static const Fft2pEntry kFft2pTable[] = {
    QE_FFT2P_ENTRY(8, 1),   QE_FFT2P_ENTRY(9, 1),   QE_FFT2P_ENTRY(10, 1),  QE_FFT2P_ENTRY(12, 1),  QE_FFT2P_ENTRY(15, 1),
    QE_FFT2P_ENTRY(16, 1),  QE_FFT2P_ENTRY(6, 3),   QE_FFT2P_ENTRY(5, 4),   QE_FFT2P_ENTRY(6, 6),   QE_FFT2P_ENTRY(8, 6),
    QE_FFT2P_ENTRY(8, 8),   QE_FFT2P_ENTRY(9, 8),   QE_FFT2P_ENTRY(10, 8),  QE_FFT2P_ENTRY(12, 8),  QE_FFT2P_ENTRY(10, 10),
    QE_FFT2P_ENTRY(12, 9),  QE_FFT2P_ENTRY(12, 10), QE_FFT2P_ENTRY(16, 8),  QE_FFT2P_ENTRY(12, 12), QE_FFT2P_ENTRY(16, 10),
    QE_FFT2P_ENTRY(15, 12), QE_FFT2P_ENTRY(16, 12), QE_FFT2P_ENTRY(16, 15), QE_FFT2P_ENTRY(16, 16),
};
#undef QE_FFT2P_ENTRY

inline const Fft2pEntry* fft2p_find_in(const Fft2pEntry* tab, size_t cnt, int n) {
  for (size_t i = 0; i < cnt; ++i)
    if (tab[i].n == n) return &tab[i];
  return nullptr;
}

}  // namespace qehpsi
