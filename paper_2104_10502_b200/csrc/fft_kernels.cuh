// fft_kernels.cuh -- the five pruned pencil passes of the local term (steps a1-a5 of DESIGN.md section 2).
//   a1 k_scatter_zinv : psi(G) -> zero-padded z sticks, inverse (exp +) FFT along i3          -> W1[b][s][ldz]
//   a2 k_yinv         : per populated plane, inverse FFT along i2 over the plane's sticks    -> W2[b][p][N2][ldz]
//   a3 k_x_vmul       : inverse FFT along i1 over the P populated planes, * V(r)/N, forward FFT along i1,
//                       keep the P populated planes (the full N1 x N2 x N3 grid is never written)
//   a4 k_yfwd         : forward FFT along i2, keep only stick rows                             -> W1
//   a5 k_zfwd_gather  : forward FFT along i3, gather the sphere, add g2kin*psi                 -> hpsi
// The paper states only that the FFTs go through 1-D and 2-D transforms and that plane waves
// are mapped to FFT grids (PAPER.md:L176 (vi)); sticks/planes pruning is the standard dual-space technique.
#pragma once
#include "fft_core.cuh"

namespace qehpsi {

struct FftGeom {
  int n1, n2, n3, ldz;  // grid; ldz = N3 rounded up to a multiple of 8 (128-byte rows)
  int npw, S, P, ntz;   // ntz = ceil(n3 / FFT_C) i3 tiles
  const int* stick_start;  // [S+1] first sphere index of each stick (canonical order makes sticks contiguous runs)
  const int* stick_i2;     // [S]
  const int* plane_stick;  // [P+1] stick range of each populated plane
  const int* plane_i1;     // [P]
  const int* pw_pos;       // [npw] tile offset phys(i3, s % FFT_C) of each sphere point inside its z tile
  const double* g2kin;     // [npw] |k+G|^2
  const double* vs;        // [N1][N2][ldz] V(r)/N
  FftAxis ax1, ax2, ax3;
};

constexpr int FFT_NT = 128;  // threads per CTA in every pass

__device__ __forceinline__ void tile_zero(double2* buf, int count, int tid) {
  const double2 z = make_double2(0.0, 0.0);
  for (int i = tid; i < count; i += FFT_NT) buf[i] = z;
}

// a1 ------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(FFT_NT) k_scatter_zinv(FftGeom g, const double2* __restrict__ psi, long long ldpsi,
                                                         double2* __restrict__ w1) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* bufA = reinterpret_cast<double2*>(smem_raw);
  double2* bufB = bufA + g.n3 * FFT_C;
  const int tid = threadIdx.x;
  const int b = blockIdx.y;
  const int s0 = blockIdx.x * FFT_C;
  const int s1 = min(s0 + FFT_C, g.S);
  tile_zero(bufA, g.n3 * FFT_C, tid);
  __syncthreads();
  const int ig0 = g.stick_start[s0], ig1 = g.stick_start[s1];
  const double2* pb = psi + (size_t)b * ldpsi;
  for (int ig = ig0 + tid; ig < ig1; ig += FFT_NT) bufA[__ldg(&g.pw_pos[ig])] = pb[ig];
  __syncthreads();
  double2* r = fft_tile<+1>(bufA, bufB, g.ax3, tid, FFT_NT);
  const int total = (s1 - s0) * g.n3;
  double2* out = w1 + ((size_t)b * g.S + s0) * g.ldz;
  for (int idx = tid; idx < total; idx += FFT_NT) {
    const int c = idx / g.n3, n = idx - c * g.n3;
    out[(size_t)c * g.ldz + n] = r[fft_phys(n, c)];
  }
}

// a2 ------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(FFT_NT) k_yinv(FftGeom g, const double2* __restrict__ w1, double2* __restrict__ w2) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* bufA = reinterpret_cast<double2*>(smem_raw);
  double2* bufB = bufA + g.n2 * FFT_C;
  const int tid = threadIdx.x;
  const int b = blockIdx.y;
  const int p = blockIdx.x / g.ntz;
  const int z0 = (blockIdx.x - p * g.ntz) * FFT_C;
  tile_zero(bufA, g.n2 * FFT_C, tid);
  __syncthreads();
  const int sp0 = g.plane_stick[p], ns = g.plane_stick[p + 1] - sp0;
  const double2* in = w1 + ((size_t)b * g.S + sp0) * g.ldz + z0;
  for (int idx = tid; idx < ns * FFT_C; idx += FFT_NT) {
    const int c = idx & (FFT_C - 1), si = idx / FFT_C;
    if (z0 + c < g.n3) bufA[fft_phys(__ldg(&g.stick_i2[sp0 + si]), c)] = in[(size_t)si * g.ldz + c];
  }
  __syncthreads();
  double2* r = fft_tile<+1>(bufA, bufB, g.ax2, tid, FFT_NT);
  double2* out = w2 + ((size_t)b * g.P + p) * g.n2 * g.ldz + z0;
  for (int idx = tid; idx < g.n2 * FFT_C; idx += FFT_NT) {
    const int c = idx & (FFT_C - 1), n = idx / FFT_C;
    if (z0 + c < g.n3) out[(size_t)n * g.ldz + c] = r[fft_phys(n, c)];
  }
}

// a3 ------------------------------------------------------------------------------------------------------
// One CTA owns the (i2, i3-tile) pencil group, keeps its V(r)/N tile in shared memory and loops over bands
// b = blockIdx.y, blockIdx.y + gridDim.y, ... so that V is read once per CTA, not once per band.
__global__ void __launch_bounds__(FFT_NT) k_x_vmul(FftGeom g, double2* __restrict__ w2, int nb) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* bufA = reinterpret_cast<double2*>(smem_raw);
  double2* bufB = bufA + g.n1 * FFT_C;
  double* vt = reinterpret_cast<double*>(bufB + g.n1 * FFT_C);
  const int tid = threadIdx.x;
  const int i2 = blockIdx.x / g.ntz;
  const int z0 = (blockIdx.x - i2 * g.ntz) * FFT_C;
  const int tile = g.n1 * FFT_C;
  for (int idx = tid; idx < tile; idx += FFT_NT) {
    const int c = idx & (FFT_C - 1), n = idx / FFT_C;
    vt[fft_phys(n, c)] = (z0 + c < g.n3) ? __ldg(&g.vs[((size_t)n * g.n2 + i2) * g.ldz + z0 + c]) : 0.0;
  }
  for (int b = blockIdx.y; b < nb; b += gridDim.y) {
    tile_zero(bufA, tile, tid);
    __syncthreads();
    double2* io = w2 + ((size_t)b * g.P * g.n2 + i2) * g.ldz + z0;
    const size_t pstride = (size_t)g.n2 * g.ldz;
    for (int idx = tid; idx < g.P * FFT_C; idx += FFT_NT) {
      const int c = idx & (FFT_C - 1), pi = idx / FFT_C;
      if (z0 + c < g.n3) bufA[fft_phys(__ldg(&g.plane_i1[pi]), c)] = io[pi * pstride + c];
    }
    __syncthreads();
    double2* r = fft_tile<+1>(bufA, bufB, g.ax1, tid, FFT_NT);
    double2* o = (r == bufA) ? bufB : bufA;
    for (int idx = tid; idx < tile; idx += FFT_NT) {
      const double v = vt[idx];
      double2 x = r[idx];
      r[idx] = make_double2(x.x * v, x.y * v);
    }
    __syncthreads();
    double2* r2 = fft_tile<-1>(r, o, g.ax1, tid, FFT_NT);
    for (int idx = tid; idx < g.P * FFT_C; idx += FFT_NT) {
      const int c = idx & (FFT_C - 1), pi = idx / FFT_C;
      if (z0 + c < g.n3) io[pi * pstride + c] = r2[fft_phys(__ldg(&g.plane_i1[pi]), c)];
    }
    __syncthreads();
  }
}

// NEXT-4 (charge density), generic plan: inverse FFT along i1, rho += scale * sum_b occ[b] |psi_b(r)|^2.
// Dynamic shared memory: two [N1][FFT_C] tiles.  gridDim.y must be 1 (one CTA owns its pencils: no atomics).
__global__ void __launch_bounds__(FFT_NT) k_x_rho(FftGeom g, const double2* __restrict__ w2, int nb,
                                                  const double* __restrict__ occ, double scale, double* __restrict__ rho) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* bufA = reinterpret_cast<double2*>(smem_raw);
  double2* bufB = bufA + g.n1 * FFT_C;
  const int tid = threadIdx.x;
  const int i2 = blockIdx.x / g.ntz;
  const int z0 = (blockIdx.x - i2 * g.ntz) * FFT_C;
  const int tile = g.n1 * FFT_C;
  const size_t pstride = (size_t)g.n2 * g.ldz;
  for (int b = 0; b < nb; ++b) {
    const double f = scale * __ldg(&occ[b]);
    tile_zero(bufA, tile, tid);
    __syncthreads();
    const double2* in = w2 + ((size_t)b * g.P * g.n2 + i2) * g.ldz + z0;
    for (int idx = tid; idx < g.P * FFT_C; idx += FFT_NT) {
      const int c = idx & (FFT_C - 1), pi = idx / FFT_C;
      if (z0 + c < g.n3) bufA[fft_phys(__ldg(&g.plane_i1[pi]), c)] = in[pi * pstride + c];
    }
    __syncthreads();
    const double2* r = fft_tile<+1>(bufA, bufB, g.ax1, tid, FFT_NT);
    for (int idx = tid; idx < tile; idx += FFT_NT) {  // the same thread owns the same grid points for every band
      const int c = idx & (FFT_C - 1), n = idx / FFT_C;
      if (z0 + c < g.n3) {
        const double2 x = r[fft_phys(n, c)];
        double* o = rho + ((size_t)n * g.n2 + i2) * g.n3 + z0 + c;
        *o += f * (x.x * x.x + x.y * x.y);
      }
    }
    __syncthreads();
  }
}

// a4 ------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(FFT_NT) k_yfwd(FftGeom g, const double2* __restrict__ w2, double2* __restrict__ w1) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* bufA = reinterpret_cast<double2*>(smem_raw);
  double2* bufB = bufA + g.n2 * FFT_C;
  const int tid = threadIdx.x;
  const int b = blockIdx.y;
  const int p = blockIdx.x / g.ntz;
  const int z0 = (blockIdx.x - p * g.ntz) * FFT_C;
  const double2* in = w2 + ((size_t)b * g.P + p) * g.n2 * g.ldz + z0;
  const double2 zero = make_double2(0.0, 0.0);
  for (int idx = tid; idx < g.n2 * FFT_C; idx += FFT_NT) {
    const int c = idx & (FFT_C - 1), n = idx / FFT_C;
    bufA[fft_phys(n, c)] = (z0 + c < g.n3) ? in[(size_t)n * g.ldz + c] : zero;
  }
  __syncthreads();
  double2* r = fft_tile<-1>(bufA, bufB, g.ax2, tid, FFT_NT);
  const int sp0 = g.plane_stick[p], ns = g.plane_stick[p + 1] - sp0;
  double2* out = w1 + ((size_t)b * g.S + sp0) * g.ldz + z0;
  for (int idx = tid; idx < ns * FFT_C; idx += FFT_NT) {
    const int c = idx & (FFT_C - 1), si = idx / FFT_C;
    if (z0 + c < g.n3) out[(size_t)si * g.ldz + c] = r[fft_phys(__ldg(&g.stick_i2[sp0 + si]), c)];
  }
}

// a5 ------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(FFT_NT) k_zfwd_gather(FftGeom g, const double2* __restrict__ w1,
                                                        const double2* __restrict__ psi, long long ldpsi,
                                                        double2* __restrict__ hpsi, long long ldh) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* bufA = reinterpret_cast<double2*>(smem_raw);
  double2* bufB = bufA + g.n3 * FFT_C;
  const int tid = threadIdx.x;
  const int b = blockIdx.y;
  const int s0 = blockIdx.x * FFT_C;
  const int s1 = min(s0 + FFT_C, g.S);
  const int total = FFT_C * g.n3;
  const int valid = (s1 - s0) * g.n3;
  const double2* in = w1 + ((size_t)b * g.S + s0) * g.ldz;
  const double2 zero = make_double2(0.0, 0.0);
  for (int idx = tid; idx < total; idx += FFT_NT) {
    const int c = idx / g.n3, n = idx - c * g.n3;
    bufA[fft_phys(n, c)] = (idx < valid) ? in[(size_t)c * g.ldz + n] : zero;
  }
  __syncthreads();
  double2* r = fft_tile<-1>(bufA, bufB, g.ax3, tid, FFT_NT);
  const int ig0 = g.stick_start[s0], ig1 = g.stick_start[s1];
  const double2* pb = psi + (size_t)b * ldpsi;
  double2* hb = hpsi + (size_t)b * ldh;
  for (int ig = ig0 + tid; ig < ig1; ig += FFT_NT) {
    const double2 v = r[__ldg(&g.pw_pos[ig])];
    const double2 c = pb[ig];
    const double k2 = __ldg(&g.g2kin[ig]);
    hb[ig] = make_double2(v.x + k2 * c.x, v.y + k2 * c.y);
  }
}

}  // namespace qehpsi
