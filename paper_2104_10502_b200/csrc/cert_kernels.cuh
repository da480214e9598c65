// cert_kernels.cuh -- a-posteriori check of the int8 digit path of the projector contractions (create flag
// QE_HPSI_PROJ_CERTIFY; include/qe_hpsi.h).  The agreement the paper reports between its CPU and GPU
// runs is an FP64 statement; the int8 path is block fixed point, so each chunk is tested after the fact:
//
//   v_b = V_NL psi_b as computed by the int8 path (kept apart in a scratch array),  s_t = random sign vectors (t < NPROBE),
//   y_t = V_NL s_t computed once at create on the FP64 tensor path (V_NL is Hermitian: D real symmetric),
//   d_tb = sum_G s_t(G) v_b(G) - sum_G conj(y_t(G)) psi_b(G)          (= <s_t | v_b - V_NL psi_b>, zero for an exact v_b)
//   est_b^2 = mean_t |d_tb|^2    estimates ||v_b - V_NL psi_b||^2      (E |<s|e>|^2 = ||e||^2 for independent random signs)
//
// Bands with est_b > tol ||v_b|| (or non-finite) are re-computed on the FP64 tensor path: chosen, compacted and launched on
// the device (the DMMA kernels take the band count from device memory), no host synchronisation.  All sums run in a fixed
// order, so the decision is reproducible run to run.
#pragma once
#include <cuda_runtime.h>

namespace qehpsi {
namespace cert {

constexpr int NPROBE = 8;
constexpr int NT = 256;
constexpr int NVAL = 2 * NPROBE + 1;  // Re/Im of d_t, then ||v||^2

// 8 independent sign bits per plane wave from a 64-bit mix hash of its index (bit t set: s_t(G) = -1)
__device__ __forceinline__ unsigned sign_bits(long long g) {
  unsigned long long x = (unsigned long long)g * 0x9E3779B97F4A7C15ull + 0xD1B54A32D192ED03ull;
  x ^= x >> 32;
  x *= 0xD6E8FEB86659FD93ull;
  x ^= x >> 32;
  x *= 0xD6E8FEB86659FD93ull;
  x ^= x >> 32;
  return (unsigned)x & 0xFFu;
}

// S[t][G] = (s_t(G), 0): the probe "bands" whose image under V_NL is y_t
__global__ void k_cert_signs(double2* __restrict__ S, long long ld, long long npw) {
  const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= npw) return;
  const unsigned bits = sign_bits(g);
#pragma unroll
  for (int t = 0; t < NPROBE; ++t) S[(size_t)t * ld + g] = make_double2((bits >> t) & 1u ? -1.0 : 1.0, 0.0);
}

// part[b][c][0..NVAL) for band b = blockIdx.y and the plane waves [c gchunk, (c+1) gchunk) of CTA c = blockIdx.x
__global__ void __launch_bounds__(NT)
k_cert_probe(const double2* __restrict__ v, long long ldv, const double2* __restrict__ psi, long long ldpsi,
             const double2* __restrict__ y, long long ldy, long long npw, int gchunk, double* __restrict__ part, int nch) {
  const int b = blockIdx.y, c = blockIdx.x;
  const long long g0 = (long long)c * gchunk, g1 = min(npw, g0 + gchunk);
  double acc[NVAL];
#pragma unroll
  for (int i = 0; i < NVAL; ++i) acc[i] = 0.0;
  const double2* vb = v + (size_t)b * ldv;
  const double2* pb = psi + (size_t)b * ldpsi;
  for (long long g = g0 + threadIdx.x; g < g1; g += NT) {
    const double2 vv = vb[g], pp = pb[g];
    const unsigned bits = sign_bits(g);
    acc[2 * NPROBE] = fma(vv.x, vv.x, fma(vv.y, vv.y, acc[2 * NPROBE]));
#pragma unroll
    for (int t = 0; t < NPROBE; ++t) {
      const double2 yy = y[(size_t)t * ldy + g];
      const double sg = (bits >> t) & 1u ? -1.0 : 1.0;
      // s v - conj(y) psi
      acc[2 * t] += sg * vv.x - (yy.x * pp.x + yy.y * pp.y);
      acc[2 * t + 1] += sg * vv.y - (yy.x * pp.y - yy.y * pp.x);
    }
  }
  // fixed-order block reduction: butterflies inside a warp, then warp 0 adds the 8 warp sums in order
  __shared__ double red[NT / 32][NVAL];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int i = 0; i < NVAL; ++i) {
    double x = acc[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    if (lane == 0) red[warp][i] = x;
  }
  __syncthreads();
  if (threadIdx.x < NVAL) {
    double x = 0.0;
#pragma unroll
    for (int w = 0; w < NT / 32; ++w) x += red[w][threadIdx.x];
    part[((size_t)b * nch + c) * NVAL + threadIdx.x] = x;
  }
}

// one CTA: per band sum the chunk partials in ascending order, rel_b = est_b / ||v_b||, redo_b = !(rel_b <= tol); then the
// ordered list of the bands to re-compute (slot <-> band) and its length
__global__ void __launch_bounds__(NT)
k_cert_decide(const double* __restrict__ part, int nch, int nb, double tol, double* __restrict__ rel, int* __restrict__ redo,
              int* __restrict__ slot, int* __restrict__ list, int* __restrict__ count) {
  for (int b = threadIdx.x; b < nb; b += NT) {
    double s[NVAL];
#pragma unroll
    for (int i = 0; i < NVAL; ++i) s[i] = 0.0;
    for (int c = 0; c < nch; ++c)
#pragma unroll
      for (int i = 0; i < NVAL; ++i) s[i] += part[((size_t)b * nch + c) * NVAL + i];
    double e2 = 0.0;
#pragma unroll
    for (int i = 0; i < 2 * NPROBE; ++i) e2 = fma(s[i], s[i], e2);
    e2 *= 1.0 / NPROBE;
    const double n2 = s[2 * NPROBE];
    double r;
    if (n2 > 0.0)
      r = sqrt(e2 / n2);
    else
      r = (e2 == 0.0 && n2 == 0.0) ? 0.0 : 1.0 / 0.0;  // zero output for zero input is exact; anything else fails the check
    rel[b] = r;
    redo[b] = (r <= tol) ? 0 : 1;  // NaN compares false: re-computed
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    int n = 0;
    for (int b = 0; b < nb; ++b) {
      if (redo[b]) {
        slot[b] = n;
        list[n++] = b;
      } else
        slot[b] = -1;
    }
    *count = n;
  }
}

// psif[slot] = psi[list[slot]], vf[slot] = 0 for slot < count
__global__ void k_cert_gather(const double2* __restrict__ psi, long long ldpsi, long long npw, const int* __restrict__ list,
                              const int* __restrict__ count, double2* __restrict__ psif, double2* __restrict__ vf, long long ld) {
  const int sl = blockIdx.y;
  if (sl >= *count) return;
  const int b = list[sl];
  for (long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x; g < npw; g += (long long)gridDim.x * blockDim.x) {
    psif[(size_t)sl * ld + g] = psi[(size_t)b * ldpsi + g];
    vf[(size_t)sl * ld + g] = make_double2(0.0, 0.0);
  }
}

// hpsi[b] += redo[b] ? vf[slot[b]] : v8[b]
__global__ void k_cert_commit(const double2* __restrict__ v8, const double2* __restrict__ vf, long long ld,
                              const int* __restrict__ redo, const int* __restrict__ slot, long long npw,
                              double2* __restrict__ hpsi, long long ldh) {
  const int b = blockIdx.y;
  const double2* src = redo[b] ? vf + (size_t)slot[b] * ld : v8 + (size_t)b * ld;
  double2* dst = hpsi + (size_t)b * ldh;
  for (long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x; g < npw; g += (long long)gridDim.x * blockDim.x) {
    double2 t = dst[g];
    const double2 a = src[g];
    t.x += a.x;
    t.y += a.y;
    dst[g] = t;
  }
}

}  // namespace cert

// ---- NEXT-3 (Davidson step): residual with its squared norm, and per-band scaling -----------------
// r[b][G] = hx[b][G] - e[b] sx[b][G]; rnorm2[b] = sum_G |r|^2.  One CTA per band, fixed summation order.
__global__ void __launch_bounds__(1024)
k_residual(const double2* __restrict__ hx, long long ldh, const double2* __restrict__ sx, long long lds,
           const double* __restrict__ e, double2* __restrict__ r, long long ldr, long long npw, double* __restrict__ rnorm2) {
  const int b = blockIdx.x;
  const double eb = e[b];
  double acc = 0.0;
  for (long long g = threadIdx.x; g < npw; g += 1024) {
    const double2 h = hx[(size_t)b * ldh + g], s = sx[(size_t)b * lds + g];
    const double2 v = make_double2(h.x - eb * s.x, h.y - eb * s.y);
    r[(size_t)b * ldr + g] = v;
    acc = fma(v.x, v.x, fma(v.y, v.y, acc));
  }
  __shared__ double red[32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0 && rnorm2) {
    double t = 0.0;
    for (int w = 0; w < 32; ++w) t += red[w];
    rnorm2[b] = t;
  }
}
__global__ void k_scale_rows(double2* __restrict__ x, long long ldx, long long npw, const double* __restrict__ fac) {
  const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= npw) return;
  const double f = fac[blockIdx.y];
  double2 v = x[(size_t)blockIdx.y * ldx + g];
  x[(size_t)blockIdx.y * ldx + g] = make_double2(v.x * f, v.y * f);
}

}  // namespace qehpsi
