// fft3p_kernels.cuh -- three-pass variant of the fast local-term path (steps a1-a5) for FFT
// lengths N = R1 * R2 * R3 whose two-factor split would need a register radix above 16 (125 = 5*5*5 is the case the
// workloads contain: the 25-point register DFT of the two-pass plan costs 254 registers and one CTA per SM).
// Every 1-D transform is three Stockham passes with two shared-memory round trips:
//     global -> regs -> radix R1 -> tile A -> twiddle + radix R2 -> tile B -> twiddle + radix R3 -> global
// with at most max(R1,R2,R3) complex values per thread.  The x stage runs the inverse as (R1,R2,R3) and the forward
// transform as (R3,R2,R1): the inverse ends holding X[j + q*R1*R2], q < R3, in registers, which is exactly what a
// forward transform that starts with radix R3 consumes, so iFFT -> *V(r)/N -> FFT costs four round trips, not six.
// Same tables, tile swizzle and global layouts as fft2p_kernels.cuh; all kernels use dynamic shared memory
// (two [N][FFT_C] tiles).  PAPER.md:L215 (FFTs as batched 1-D/2-D transforms), L176 (vi) (plane waves <-> grid).
#pragma once
#include "fft2p_kernels.cuh"

namespace qehpsi {

template <int R1, int R2, int R3>
struct P3 {
  static constexpr int N = R1 * R2 * R3;
  static constexpr int T1 = N / R1, T2 = N / R2, T3 = N / R3;  // tasks (per pencil) of the three passes
  static constexpr int TMAX = (T1 > T2 ? (T1 > T3 ? T1 : T3) : (T2 > T3 ? T2 : T3));
  static constexpr int NT = TMAX * FFT_C;
  static constexpr size_t SMEM = 2 * (size_t)N * FFT_C * sizeof(double2);
};

// middle Stockham pass, radix R, Ns = product of the radices already applied: tile in -> tile out
template <int R, int DIR>
__device__ __forceinline__ void pass_mid(const double2* __restrict__ tin, double2* __restrict__ tout,
                                         const double2* __restrict__ tw, int N, int Ns, int j, int c) {
  const int M = N / R;
  const int k = j % Ns;
  const int e = k * (M / Ns);
  double2 v[R];
#pragma unroll
  for (int q = 0; q < R; ++q) v[q] = tin[fft_phys(j + q * M, c)];
#pragma unroll
  for (int q = 1; q < R; ++q) {
    const double2 w = __ldg(&tw[q * e]);
    v[q] = DIR > 0 ? cmul(v[q], w) : cmulc(v[q], w);
  }
  Dft<R, DIR>::run(v);
  const int j0 = (j - k) * R + k;
#pragma unroll
  for (int q = 0; q < R; ++q) tout[fft_phys(j0 + q * Ns, c)] = v[q];
}

// a1 ------------------------------------------------------------------------------------------------------
template <int R1, int R2, int R3>
__global__ void __launch_bounds__(P3<R1, R2, R3>::NT) k3p_scatter_zinv(FftGeom g, Fft2pGeom t, const double2* __restrict__ psi,
                                                                      long long ldpsi, double2* __restrict__ w1) {
  using P = P3<R1, R2, R3>;
  constexpr int N = P::N;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* tA = reinterpret_cast<double2*>(smem_raw);
  double2* tB = tA + N * FFT_C;
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const int b = blockIdx.y;
  const int s = blockIdx.x * FFT_C + c;
  const bool sok = s < g.S;
  const double2 zero = make_double2(0.0, 0.0);
  if (j < P::T1) {
    double2 v[R1];
    if (sok) {
      const int start = g.stick_start[s], lo = t.stick_lo[s], hi = t.stick_hi[s];
      const double2* pb = psi + (size_t)b * ldpsi;
#pragma unroll
      for (int q = 0; q < R1; ++q) {
        const int pos = stick_pos(start, lo, hi, j + q * P::T1, N);
        v[q] = pos >= 0 ? pb[pos] : zero;
      }
    } else {
#pragma unroll
      for (int q = 0; q < R1; ++q) v[q] = zero;
    }
    pass_a_store<R1, +1>(v, tA, j, c);
  }
  __syncthreads();
  if (j < P::T2) pass_mid<R2, +1>(tA, tB, g.ax3.tw, N, R1, j, c);
  __syncthreads();
  if (j < P::T3) {
    double2 u[R3];
    pass_b_load<P::T3, R3, +1>(tB, g.ax3.tw, j, c, u);
    if (sok) {
      double2* out = w1 + ((size_t)b * g.S + s) * g.ldz + j;
#pragma unroll
      for (int q = 0; q < R3; ++q) out[q * P::T3] = u[q];
    }
  }
}

// a5 ------------------------------------------------------------------------------------------------------
template <int R1, int R2, int R3>
__global__ void __launch_bounds__(P3<R1, R2, R3>::NT) k3p_zfwd_gather(FftGeom g, Fft2pGeom t, const double2* __restrict__ w1,
                                                                     const double2* __restrict__ psi, long long ldpsi,
                                                                     double2* __restrict__ hpsi, long long ldh) {
  using P = P3<R1, R2, R3>;
  constexpr int N = P::N;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* tA = reinterpret_cast<double2*>(smem_raw);
  double2* tB = tA + N * FFT_C;
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const int b = blockIdx.y;
  const int s = blockIdx.x * FFT_C + c;
  const bool sok = s < g.S;
  const double2 zero = make_double2(0.0, 0.0);
  if (j < P::T1) {
    double2 v[R1];
    const double2* in = w1 + ((size_t)b * g.S + (sok ? s : 0)) * g.ldz;
#pragma unroll
    for (int q = 0; q < R1; ++q) v[q] = sok ? in[j + q * P::T1] : zero;
    pass_a_store<R1, -1>(v, tA, j, c);
  }
  __syncthreads();
  if (j < P::T2) pass_mid<R2, -1>(tA, tB, g.ax3.tw, N, R1, j, c);
  __syncthreads();
  if (j < P::T3) {
    double2 u[R3];
    pass_b_load<P::T3, R3, -1>(tB, g.ax3.tw, j, c, u);
    if (sok) {
      const int start = g.stick_start[s], lo = t.stick_lo[s], hi = t.stick_hi[s];
      const double2* pb = psi + (size_t)b * ldpsi;
      double2* hb = hpsi + (size_t)b * ldh;
#pragma unroll
      for (int q = 0; q < R3; ++q) {
        const int pos = stick_pos(start, lo, hi, j + q * P::T3, N);
        if (pos >= 0) {
          const double2 cpsi = pb[pos];
          const double k2 = __ldg(&g.g2kin[pos]);
          hb[pos] = make_double2(u[q].x + k2 * cpsi.x, u[q].y + k2 * cpsi.y);
        }
      }
    }
  }
}

// a2 ------------------------------------------------------------------------------------------------------
template <int R1, int R2, int R3>
__global__ void __launch_bounds__(P3<R1, R2, R3>::NT) k3p_yinv(FftGeom g, Fft2pGeom t, const double2* __restrict__ w1,
                                                              double2* __restrict__ w2) {
  using P = P3<R1, R2, R3>;
  constexpr int N = P::N;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* tA = reinterpret_cast<double2*>(smem_raw);
  double2* tB = tA + N * FFT_C;
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const int b = blockIdx.y;
  const int p = blockIdx.x / g.ntz;
  const int z = (blockIdx.x - p * g.ntz) * FFT_C + c;
  const double2 zero = make_double2(0.0, 0.0);
  const double2* in = w1 + (size_t)b * g.S * g.ldz + z;
  double2* out = w2 + ((size_t)b * g.P + p) * N * g.ldz + z;
  const int* col = t.col_of + (size_t)p * N;
  if (j < P::T1) {
    double2 v[R1];
#pragma unroll
    for (int q = 0; q < R1; ++q) {
      const int s = __ldg(&col[j + q * P::T1]);
      v[q] = s >= 0 ? in[(size_t)s * g.ldz] : zero;
    }
    pass_a_store<R1, +1>(v, tA, j, c);
  }
  __syncthreads();
  if (j < P::T2) pass_mid<R2, +1>(tA, tB, g.ax2.tw, N, R1, j, c);
  __syncthreads();
  if (j < P::T3) {
    double2 u[R3];
    pass_b_load<P::T3, R3, +1>(tB, g.ax2.tw, j, c, u);
#pragma unroll
    for (int q = 0; q < R3; ++q) out[(size_t)(j + q * P::T3) * g.ldz] = u[q];
  }
}

// a4 ------------------------------------------------------------------------------------------------------
template <int R1, int R2, int R3>
__global__ void __launch_bounds__(P3<R1, R2, R3>::NT) k3p_yfwd(FftGeom g, Fft2pGeom t, const double2* __restrict__ w2,
                                                              double2* __restrict__ w1) {
  using P = P3<R1, R2, R3>;
  constexpr int N = P::N;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* tA = reinterpret_cast<double2*>(smem_raw);
  double2* tB = tA + N * FFT_C;
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const int b = blockIdx.y;
  const int p = blockIdx.x / g.ntz;
  const int z = (blockIdx.x - p * g.ntz) * FFT_C + c;
  const double2* in = w2 + ((size_t)b * g.P + p) * N * g.ldz + z;
  double2* out = w1 + (size_t)b * g.S * g.ldz + z;
  const int* col = t.col_of + (size_t)p * N;
  if (j < P::T1) {
    double2 v[R1];
#pragma unroll
    for (int q = 0; q < R1; ++q) v[q] = in[(size_t)(j + q * P::T1) * g.ldz];
    pass_a_store<R1, -1>(v, tA, j, c);
  }
  __syncthreads();
  if (j < P::T2) pass_mid<R2, -1>(tA, tB, g.ax2.tw, N, R1, j, c);
  __syncthreads();
  if (j < P::T3) {
    double2 u[R3];
    pass_b_load<P::T3, R3, -1>(tB, g.ax2.tw, j, c, u);
#pragma unroll
    for (int q = 0; q < R3; ++q) {
      const int s = __ldg(&col[j + q * P::T3]);
      if (s >= 0) out[(size_t)s * g.ldz] = u[q];
    }
  }
}

// a3 ------------------------------------------------------------------------------------------------------
// inverse (R1,R2,R3) over the P populated planes, * V(r)/N in registers, forward (R3,R2,R1), keep populated planes
template <int R1, int R2, int R3>
__global__ void __launch_bounds__(P3<R1, R2, R3>::NT) k3p_x_vmul(FftGeom g, Fft2pGeom t, double2* __restrict__ w2, int nb) {
  using P = P3<R1, R2, R3>;
  constexpr int N = P::N;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* tA = reinterpret_cast<double2*>(smem_raw);
  double2* tB = tA + N * FFT_C;
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const int i2 = blockIdx.x / g.ntz;
  const int z = (blockIdx.x - i2 * g.ntz) * FFT_C + c;
  const double2 zero = make_double2(0.0, 0.0);
  const size_t pstride = (size_t)g.n2 * g.ldz;
  // V(r)/N at the points held after the inverse transform: i1 = j + q*T3, q < R3 (threads j < T3)
  double vv[R3];
  if (j < P::T3) {
#pragma unroll
    for (int q = 0; q < R3; ++q) vv[q] = __ldg(&g.vs[((size_t)(j + q * P::T3) * g.n2 + i2) * g.ldz + z]);
  }
  // populated-plane index of the inputs / final outputs: i1 = j + q*T1, q < R1 (threads j < T1)
  int pl[R1];
  if (j < P::T1) {
#pragma unroll
    for (int q = 0; q < R1; ++q) pl[q] = __ldg(&t.plane_of[j + q * P::T1]);
  }
  for (int b = blockIdx.y; b < nb; b += gridDim.y) {
    double2* io = w2 + ((size_t)b * g.P * g.n2 + i2) * g.ldz + z;
    if (j < P::T1) {
      double2 v[R1];
#pragma unroll
      for (int q = 0; q < R1; ++q) v[q] = pl[q] >= 0 ? io[pl[q] * pstride] : zero;
      pass_a_store<R1, +1>(v, tA, j, c);
    }
    __syncthreads();
    if (j < P::T2) pass_mid<R2, +1>(tA, tB, g.ax1.tw, N, R1, j, c);
    __syncthreads();
    if (j < P::T3) {
      double2 u[R3];
      pass_b_load<P::T3, R3, +1>(tB, g.ax1.tw, j, c, u);
#pragma unroll
      for (int q = 0; q < R3; ++q) u[q] = make_double2(u[q].x * vv[q], u[q].y * vv[q]);
      pass_a_store<R3, -1>(u, tA, j, c);  // forward pass 1 (radix R3, Ns = 1) on x[j + q*T3]
    }
    __syncthreads();
    if (j < P::T2) pass_mid<R2, -1>(tA, tB, g.ax1.tw, N, R3, j, c);
    __syncthreads();
    if (j < P::T1) {
      double2 v[R1];
      pass_b_load<P::T1, R1, -1>(tB, g.ax1.tw, j, c, v);
#pragma unroll
      for (int q = 0; q < R1; ++q)
        if (pl[q] >= 0) io[pl[q] * pstride] = v[q];
    }
    // the next band's first pass writes tile A, last read by the forward middle pass two barriers ago: safe
  }
}

// NEXT-4 (charge density): inverse (R1,R2,R3) along i1, rho += scale * sum_b occ[b] |psi_b(r)|^2 (see k2p_x_rho)
template <int R1, int R2, int R3>
__global__ void __launch_bounds__(P3<R1, R2, R3>::NT) k3p_x_rho(FftGeom g, Fft2pGeom t, const double2* __restrict__ w2, int nb,
                                                               const double* __restrict__ occ, double scale,
                                                               double* __restrict__ rho) {
  using P = P3<R1, R2, R3>;
  constexpr int N = P::N;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* tA = reinterpret_cast<double2*>(smem_raw);
  double2* tB = tA + N * FFT_C;
  const int tid = threadIdx.x, c = tid & (FFT_C - 1), j = tid / FFT_C;
  const int i2 = blockIdx.x / g.ntz;
  const int z = (blockIdx.x - i2 * g.ntz) * FFT_C + c;
  const double2 zero = make_double2(0.0, 0.0);
  const size_t pstride = (size_t)g.n2 * g.ldz;
  int pl[R1];
  if (j < P::T1) {
#pragma unroll
    for (int q = 0; q < R1; ++q) pl[q] = __ldg(&t.plane_of[j + q * P::T1]);
  }
  double acc[R3];
#pragma unroll
  for (int q = 0; q < R3; ++q) acc[q] = 0.0;
  for (int b = 0; b < nb; ++b) {
    const double f = __ldg(&occ[b]);
    const double2* in = w2 + ((size_t)b * g.P * g.n2 + i2) * g.ldz + z;
    if (j < P::T1) {
      double2 v[R1];
#pragma unroll
      for (int q = 0; q < R1; ++q) v[q] = pl[q] >= 0 ? in[pl[q] * pstride] : zero;
      pass_a_store<R1, +1>(v, tA, j, c);
    }
    __syncthreads();
    if (j < P::T2) pass_mid<R2, +1>(tA, tB, g.ax1.tw, N, R1, j, c);
    __syncthreads();
    if (j < P::T3) {
      double2 u[R3];
      pass_b_load<P::T3, R3, +1>(tB, g.ax1.tw, j, c, u);
#pragma unroll
      for (int q = 0; q < R3; ++q) acc[q] += f * (u[q].x * u[q].x + u[q].y * u[q].y);
    }
    // next band: tile A is rewritten before the first barrier (last read before the second barrier above: safe);
    // tile B is rewritten after the next band's first barrier, i.e. after every thread has left this read
  }
  if (z < g.n3 && j < P::T3) {
#pragma unroll
    for (int q = 0; q < R3; ++q) {
      double* r = rho + ((size_t)(j + q * P::T3) * g.n2 + i2) * g.n3 + z;
      *r += scale * acc[q];
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// dispatch: lengths served by the three-pass plan (ra = R1, rb = R2*R3 in the shared entry type)
// ---------------------------------------------------------------------------------------------------------
#define QE_FFT3P_ENTRY(R1, R2, R3)                                                                                 \
  {                                                                                                                \
    (R1) * (R2) * (R3), R1, (R2) * (R3), P3<R1, R2, R3>::NT, P3<R1, R2, R3>::SMEM, P3<R1, R2, R3>::SMEM,            \
        k3p_scatter_zinv<R1, R2, R3>, k3p_zfwd_gather<R1, R2, R3>, k3p_yinv<R1, R2, R3>, k3p_yfwd<R1, R2, R3>,      \
        k3p_x_vmul<R1, R2, R3>, k3p_x_rho<R1, R2, R3>                                                              \
  }

static const Fft2pEntry kFft3pTable[] = {
    QE_FFT3P_ENTRY(5, 5, 5),  // 125
    QE_FFT3P_ENTRY(6, 5, 5),  // 150
    QE_FFT3P_ENTRY(8, 5, 5),  // 200
    QE_FFT3P_ENTRY(6, 6, 6),  // 216
    QE_FFT3P_ENTRY(10, 5, 5), // 250
    QE_FFT3P_ENTRY(8, 6, 6),  // 288
    QE_FFT3P_ENTRY(10, 6, 5), // 300
    QE_FFT3P_ENTRY(8, 8, 5),  // 320
    QE_FFT3P_ENTRY(10, 6, 6), // 360
    QE_FFT3P_ENTRY(8, 8, 6),  // 384
};
#undef QE_FFT3P_ENTRY

// two-pass plan first (one shared-memory round trip; measured 1.1-1.9x faster than three passes at 96, 144 and 192 on
// B200, where the extra round trips make shared memory the limiter), three-pass plan for the lengths it does not serve
inline const Fft2pEntry* fft2p_find(int n, bool prefer3 = false) {
  const Fft2pEntry* e2 = fft2p_find_in(kFft2pTable, sizeof(kFft2pTable) / sizeof(kFft2pTable[0]), n);
  const Fft2pEntry* e3 = fft2p_find_in(kFft3pTable, sizeof(kFft3pTable) / sizeof(kFft3pTable[0]), n);
  if (prefer3) return e3 ? e3 : e2;
  return e2 ? e2 : e3;
}

}  // namespace qehpsi
