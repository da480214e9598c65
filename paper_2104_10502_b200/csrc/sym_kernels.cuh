// sym_kernels.cuh -- Gamma-symmetric projector mode of the FP64 nonlocal term ("Gamma-point specific
// algorithms"; the three H terms PAPER.md:L224-226).
//
// At k = 0 a projector that is real in real space obeys beta_p(-G) = conj(beta_p(G)) (class 0), or beta_p(-G) = -conj(beta_p(G))
// (class 1: odd l without the (-i)^l factor; then i*beta_p is Hermitian).  The library CHECKS this bit for bit at create
// (k_sym_classify); if every projector falls in one of the two classes and D couples equal classes only, a generic complex
// psi = u + i v (u, v Hermitian: u(G) = (psi(G) + conj psi(-G)) / 2, v(G) = (psi(G) - conj psi(-G)) / 2i) is contracted as TWO
// real-wavefunction problems over the half sphere:
//     <beta_p|u> = 2 sum_half (b_r u_r + b_i u_i)  (real)      with b = beta_p (class 0) or i beta_p (class 1)
//     V psi (G) = X(G) + i Y(G),  V psi (-G) = conj X(G) + i conj Y(G),   X = sum_p b_p Re e_p,  Y = sum_p b_p Im e_p
// i.e. 2 real DMMAs per complex K element and band instead of the 3 of the 3M complex product: 2/3 of the tensor work and half
// of the beta traffic, in the same FP64 arithmetic.  The half sphere is read from the leading M entries (n1 >= 0) of the
// caller's own beta rows (canonical order puts them first), so no copy of beta is made.
#pragma once
#include <cuda_runtime.h>

namespace qehpsi {
namespace sym {

// cls[p] = 0: beta_p(-G) == conj(beta_p(G)) for every pair, bit for bit; 1: == -conj; 2: neither.  One CTA per projector.
// minus[g] for g < M: position of -G (>= 0), -1 = not in the half sphere (partner row handled from the other side), -2 = G = 0.
__global__ void __launch_bounds__(256)
k_sym_classify(const double2* __restrict__ beta, long long ldb, int M, const int* __restrict__ minus, unsigned char* __restrict__ cls) {
  const double2* row = beta + (size_t)blockIdx.x * ldb;
  bool herm = true, anti = true;
  for (int g = threadIdx.x; g < M; g += 256) {
    const int m = minus[g];
    if (m == -1) continue;
    const double2 a = row[g];
    if (m == -2) {  // G = 0: conj(a) = +-a
      herm &= (a.y == 0.0);
      anti &= (a.x == 0.0);
      continue;
    }
    const double2 c = row[m];
    herm &= (c.x == a.x) && (c.y == -a.y);
    anti &= (c.x == -a.x) && (c.y == a.y);
  }
  __shared__ int sh, sa;
  if (threadIdx.x == 0) sh = 1, sa = 1;
  __syncthreads();
  if (!herm) sh = 0;
  if (!anti) sa = 0;
  __syncthreads();
  if (threadIdx.x == 0) cls[blockIdx.x] = sh ? 0 : (sa ? 1 : 2);
}

// U[2b][g] = u'_b(g), U[2b+1][g] = v'_b(g) for g < M with the weights of the half-sphere sum folded in:
//   u' = psi(G) + conj psi(-G),  v' = (psi(G) - conj psi(-G)) / i   (= 2u, 2v);  G = 0: (Re psi, 0), (Im psi, 0);  skipped rows: 0
__global__ void k_sym_merge(const double2* __restrict__ psi, long long ldpsi, int M, const int* __restrict__ minus,
                            double2* __restrict__ U, long long ldu) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  const int b = blockIdx.y;
  if (g >= M) return;
  const int m = minus[g];
  double2 u = make_double2(0.0, 0.0), v = u;
  if (m != -1) {
    const double2 a = psi[(size_t)b * ldpsi + g];
    if (m == -2) {
      u = make_double2(a.x, 0.0);
      v = make_double2(a.y, 0.0);
    } else {
      const double2 c = psi[(size_t)b * ldpsi + m];
      u = make_double2(a.x + c.x, a.y - c.y);
      v = make_double2(a.y + c.y, c.x - a.x);
    }
  }
  U[(size_t)(2 * b) * ldu + g] = u;
  U[(size_t)(2 * b + 1) * ldu + g] = v;
}

// a7 front end: becp[p][b] from the split-K partials of the real form (columns 2b = <b_p|u>, 2b+1 = <b_p|v>, value in .x),
// slices summed in ascending order.  class 0: becp = A_u + i A_v;  class 1 (b = i beta): <beta|u> = i A_u  ->  becp = -A_v + i A_u
__global__ void k_sym_reduce(const double2* __restrict__ partial, int nsplit, int nproj, int ldc2, int nb,
                             const unsigned char* __restrict__ cls, double2* __restrict__ becp, int ldc) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  const int p = blockIdx.y;
  if (b >= nb) return;
  double au = 0.0, av = 0.0;
  for (int ks = 0; ks < nsplit; ++ks) {
    const double2* row = partial + ((size_t)ks * nproj + p) * ldc2;
    au += row[2 * b].x;
    av += row[2 * b + 1].x;
  }
  becp[(size_t)p * ldc + b] = cls[p] ? make_double2(-av, au) : make_double2(au, av);
}

// B operand of the symmetric a8: e_p = dbecp_p (class 0) or dbecp_p / i (class 1);  E[2b][p] = (Re e, s Re e), E[2b+1][p] =
// (Im e, s Im e) with s = +1 (class 0) / -1 (class 1): the second slot carries the sign of the i*beta row (k_vnl_add, SYM)
__global__ void k_sym_coef(const double2* __restrict__ dbecp, int nproj, int ldc, int nb, const unsigned char* __restrict__ cls,
                           double2* __restrict__ E, int ldp) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  const int p = blockIdx.y;
  if (b >= nb) return;
  const double2 d = dbecp[(size_t)p * ldc + b];
  const double2 e = cls[p] ? make_double2(d.y, -d.x) : d;
  const double sg = cls[p] ? -1.0 : 1.0;
  E[(size_t)(2 * b) * ldp + p] = make_double2(e.x, sg * e.x);
  E[(size_t)(2 * b + 1) * ldp + p] = make_double2(e.y, sg * e.y);
}

}  // namespace sym
}  // namespace qehpsi
