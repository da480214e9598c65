// qe_hpsi.cu -- C ABI of libqe_hpsi.so (include/qe_hpsi.h): handle, plan, G-sphere maps (a0) and the launch
// sequence of the hot path (a1-a8).  No torch types, no cuFFT / cuBLAS: every step runs in this library's kernels.
// PAPER.md:L105 (the operation), L224-226 (the three terms), L176 (vi) (sphere + FFT mapping); formulas and
// readings: DESIGN.md sections 2-3.
#include "../../include/qe_hpsi_test.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "fft_kernels.cuh"
#include "fft3p_kernels.cuh"
#include "fft2t_kernels.cuh"
#include "zgemm_kernels.cuh"
#include "zgemm_tma_kernels.cuh"
#include "ozaki_kernels.cuh"
#include "cert_kernels.cuh"
#include "sym_kernels.cuh"

using namespace qehpsi;

namespace {

constexpr double TWO_PI = 6.283185307179586;
constexpr int NUM_SMS_FALLBACK = 148;

// ZGEMM tile configurations (see zgemm_kernels.cuh): BM, BN, warps along M, warps along N, BK, pipeline stages.
// Variant 0 is the product default; the others exist for tuning runs (env QE_HPSI_ZG_VARIANT).
using ZgV0 = ZgCfg<64, 64, 2, 4, 16, 4>;
using ZgS = ZgCfg<64, 128, 2, 4, 16, 4>;  // real forms of the Gamma-symmetric mode: 2 nb columns, 4 x 4 blocks per warp

struct DevBuf {
  void* p = nullptr;
  size_t bytes = 0;
};

}  // namespace

struct qe_hpsi_handle {
  int device = 0;
  int num_sms = NUM_SMS_FALLBACK;
  int last_cuda = 0;
  // geometry
  int nr[3] = {0, 0, 0};
  int ldz = 0;
  int npw = 0, S = 0, P = 0;
  // maps (device)
  int* miller = nullptr;   // [npw][3]
  int* fftidx = nullptr;   // [npw]
  double* g2kin = nullptr; // [npw]
  int *stick_start = nullptr, *stick_i2 = nullptr, *plane_stick = nullptr, *plane_i1 = nullptr, *pw_pos = nullptr;
  double* vs = nullptr;    // V(r)/N  [N1][N2][ldz]
  double2* tw[3] = {nullptr, nullptr, nullptr};
  FftGeom geom{};
  size_t smem_z = 0, smem_y = 0, smem_x = 0;
  int fft_nb = 1;  // bands per FFT sub-chunk
  int x_split = 1;
  double2 *w1 = nullptr, *w2 = nullptr;
  // fast two-pass FFT path (fft2p_kernels.cuh): used when every grid dimension has a table entry
  const Fft2pEntry* f2p[3] = {nullptr, nullptr, nullptr};  // per axis j = 0..2 (N1, N2, N3)
  Fft2pGeom g2p{};
  int *stick_lo = nullptr, *stick_hi = nullptr, *col_of = nullptr, *plane_of = nullptr;
  int *plane_yhi = nullptr, *plane_ylo = nullptr;  // wrapped-interval rule of the sticks of a plane along i2
  double2* zrow = nullptr;                          // ldz zeros
  size_t smem_x2p = 0;
  // TMA-staged x stage (fft2t_kernels.cuh): tensor map over W2, used when the length has a two-pass plan with RB > 1
  K2tX x_tma = nullptr;
  int x_half = 0;  // x stage with quarter pruning (k2t_x_vmul<RA, RB, true>)
  K2tRho rho_tma = nullptr;  // TMA-staged density kernel (needs the unswizzled tensor map of x_tma)
  size_t smem_rho = 0;
  int x_one_tile = 0;  // two-pass x stage with one shared tile (tuning knob QE_HPSI_X_ONE_TILE)
  K2pZinv z_tma_inv = nullptr;  // bulk-staged a1 / a5 (fft2t_kernels.cuh)
  K2pZfwd z_tma_fwd = nullptr;
  size_t smem_zt = 0;
  CUtensorMap tmap_w2{};
  size_t smem_xt = 0;
  // nonlocal
  int nproj = 0;
  const double2* beta = nullptr;  // borrowed or owned
  double2* beta_own = nullptr;
  long long ldbeta = 0;
  int *proj_blk0 = nullptr, *proj_nh = nullptr;
  long long* proj_doff = nullptr;
  double* dpk = nullptr;
  int max_batch = 0;
  int ldc = 0, ldp = 0;
  int nsplit = 1, kchunk = 0;
  double2 *partial = nullptr, *becp = nullptr, *dbecp = nullptr, *dbT = nullptr;
  // projector contractions on tcgen05 int8 slices (ozaki_kernels.cuh): oz_s = slices per FP64 operand, 0 = FP64 DMMA path
  int oz_s = 0, oz_stages = 0, oz_nsplit = 1, oz_kchunk = 0, oz_kchunk2 = 0;  // K blocks per CTA of a6 / per launch of a8
  size_t oz_smem = 0;
  long long oz_k1 = 0, oz_k2 = 0;  // padded real K of a6 (2 npw) and a8 (2 nproj), bytes per int8 row
  int8_t *oz_a1 = nullptr, *oz_a2 = nullptr, *oz_b = nullptr;  // [S][nproj][k1], [S][npw][k2], [S][2 max_batch][max(k1,k2)]
  int *oz_ep = nullptr, *oz_eg = nullptr, *oz_eb = nullptr;     // exponents: per projector, per plane wave, per band
  double2* oz_partial = nullptr;
  CUtensorMap oz_tm_a1{}, oz_tm_a2{}, oz_tm_b1{}, oz_tm_b2{};
  // integer 3M form of a6 (complex handles): planar digit planes (Re, Im, (Re -/+ Im)/2), three real GEMMs over the complex index
  bool oz_3m = false;
  long long oz_k1c = 0;
  CUtensorMap oz_tm_a3[3] = {}, oz_tm_b3[3] = {};
  bool oz_3m8 = false;  // a8 in the 3M form too (k_oz_vnl3): needs the padded nproj within one exact-int32 K range
  long long oz_k2c = 0;
  CUtensorMap oz_tm_a4[3] = {}, oz_tm_b4[3] = {};
  // NEXT-2: overlap operator S (q blocks packed like D; qbecp/qbT mirror dbecp/dbT)
  long long d_total = 0;
  double* qpk = nullptr;
  double2 *qbecp = nullptr, *qbT = nullptr;
  // NEXT-3: split-K workspace of qe_hpsi_overlap (allocated at create: its size depends on npw only)
  double2* ovl_partial = nullptr;
  int ovl_ns = 1, ovl_kchunk = 0;
  // Gamma-symmetric projector mode of the FP64 path (sym_kernels.cuh): detected at create
  bool sym = false;
  int sym_m = 0;                      // leading sphere entries with n1 >= 0 (they hold the half sphere)
  int* sym_minus = nullptr;           // [sym_m] position of -G, -1 skip, -2 G = 0
  unsigned char* sym_cls = nullptr;   // [nproj] 0: beta(-G) = conj beta(G), 1: = -conj
  unsigned* sym_cmask = nullptr;      // [ceil(nproj / 16)] bit j: class of projector 16 t + j (K tiles of the symmetric a8)
  int sym_wide = 1;                   // 128-column tiles (ZgS) instead of ZgV0 (tuning knob QE_HPSI_SYM_WIDE)
  bool sym_tma = false;               // operand tiles of the symmetric FP64 kernels by TMA (zgemm_tma_kernels.cuh; knob QE_HPSI_SYM_TMA)
  CUtensorMap tm_a6_beta, tm_a6_u, tm_a8_beta, tm_a8_e;
  bool zg_tma = false;                // the same for the general complex / Gamma-only kernels (knob QE_HPSI_ZG_TMA); beta maps over
  CUtensorMap tm_g6_beta, tm_g8_beta; // the whole sphere made at create, the maps of psi / coefficient rows per call
  double2 *sym_u = nullptr, *sym_e = nullptr, *sym_partial = nullptr;  // [2 max_batch][sym_ldu], [2 max_batch][ldp], [nsplit][nproj][ldc2]
  long long sym_ldu = 0;
  int sym_nsplit = 1, sym_ldc2 = 0, sym_kchunk = 0;
  int* sym_live = nullptr;            // row tiles (64 rows) of the half-sphere prefix that have at least one row to store, ascending
  int sym_nlive = 0;
  CUtensorMap tm_a8_e64, tm_a6_u64;   // E / U with 64-row boxes: the last partial wave of the symmetric a8, and calls of at most
                                      // 32 bands (64 real columns), run on 64 x 64 tiles
  bool sym_tail = false;
  int sym_dead0 = 0, sym_dead1 = 0;   // K tiles [dead0, dead1) of 16 rows of the half-sphere prefix hold rows of the other half only (U = 0 there)
  std::vector<unsigned char> sym_cls_host;  // copy of sym_cls for qe_hpsi_set_s
  bool sym_q_ok = false;                    // the q blocks of qe_hpsi_set_s couple equal classes only
  std::vector<int> blk_off;                 // atom block table (for the same check)
  // QE_HPSI_PROJ_CERTIFY: a-posteriori check of the int8 nonlocal part + FP64 re-computation
  bool certify = false;
  double cert_tol = 1e-11;
  long long cert_ld = 0;                      // row stride of the scratch arrays below
  double2* cert_y = nullptr;                  // [QE_HPSI_NPROBE][cert_ld]  y_t = V_NL s_t (FP64 tensor path, at create)
  double2 *cert_v8 = nullptr, *cert_psif = nullptr, *cert_vf = nullptr;  // [max_batch][cert_ld]: int8 v, compacted psi, FP64 v
  double* cert_part = nullptr;                // [max_batch][cert_nch][2 NPROBE + 1] partial sums of the check
  int cert_nch = 0;
  double* cert_rel = nullptr;                 // [max_batch] est_b / ||v_b||
  int *cert_redo = nullptr, *cert_slot = nullptr, *cert_list = nullptr, *cert_count = nullptr;
  double2 *partial_f = nullptr, *becp_f = nullptr, *dbecp_f = nullptr, *dbT_f = nullptr;  // a6-a7 buffers of the re-computation
  bool rho_attr_done = false;
  // NEXT-1: this handle is the half-sphere nonlocal part of a Gamma-only handle (real becp, two real DMMAs per block)
  bool gamma = false;
  int nb_last = 0;
  size_t workspace_bytes = 0;
  // apply_host staging
  double2* hbuf_psi[2] = {nullptr, nullptr};
  double2* hbuf_h[2] = {nullptr, nullptr};
  long long ldint = 0;
  cudaStream_t st_in = nullptr, st_comp = nullptr, st_out = nullptr;
  // optional overlap of the FFT chain with the projector ZGEMM (QE_HPSI_OVERLAP)
  int overlap = 0;
  cudaStream_t st_fft = nullptr;
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  cudaEvent_t ev_in[2] = {nullptr, nullptr}, ev_comp[2] = {nullptr, nullptr}, ev_out[2] = {nullptr, nullptr};
  // optional stage timing (qe_hpsi_profile): CUDA events recorded around stages on the caller's stream
  int prof_mode = 0;
  std::vector<cudaEvent_t> prof_pool;
  size_t prof_used = 0;
  struct ProfSpan {
    size_t e0, e1;
    int slot;
  };
  std::vector<ProfSpan> prof_spans;
  double prof_ms[16] = {0};
  long long prof_cnt[16] = {0};
  // guard bands: every device buffer the handle owns ends in a pattern-filled tail that qe_hpsi_test_check_guards verifies
  struct Guard {
    const unsigned char* p;
    size_t n;
  };
  std::vector<Guard> guards;
};

namespace {

#define CU_TRY(h, expr)                                   \
  do {                                                    \
    cudaError_t e__ = (expr);                             \
    if (e__ != cudaSuccess) {                             \
      if (h) (h)->last_cuda = (int)e__;                   \
      g_last_cuda = (int)e__;                             \
      return QE_HPSI_ECUDA;                               \
    }                                                     \
  } while (0)

std::atomic<int> g_last_cuda{0};  // last CUDA error of calls that have no handle (diagnostic only)

// Device allocation of a buffer the handle owns, with a guard band: the bytes from `bytes` up to the next multiple of 256
// plus 256 more are filled with 0xA5 and registered; qe_hpsi_test_check_guards (include/qe_hpsi_test.h) verifies them, so
// any kernel that writes past the end of a workspace is caught by the ordinary GPU tests (compute-sanitizer is not
// available on the test pool).  Costs <= 511 bytes and one small memset per buffer, at create time only.
constexpr size_t GUARD_BYTES = 256;
template <typename T>
cudaError_t guarded_malloc(qe_hpsi_handle* h, T** p, size_t bytes) {
  const size_t padded = (bytes + 255) / 256 * 256 + GUARD_BYTES;
  cudaError_t e = cudaMalloc(p, padded);
  if (e != cudaSuccess) return e;
  unsigned char* tail = reinterpret_cast<unsigned char*>(*p) + bytes;
  e = cudaMemset(tail, 0xA5, padded - bytes);
  if (e != cudaSuccess) return e;
  try {
    h->guards.push_back({tail, padded - bytes});
  } catch (...) {  // out of host memory: this buffer is simply not watched
  }
  return cudaSuccess;
}

// ---- stage timing helpers ---------------------------------------------------------------------------------
enum { SLOT_BECP = 0, SLOT_DMUL = 1, SLOT_FFT = 2, SLOT_VNL = 3, SLOT_A1 = 4, SLOT_A2 = 5, SLOT_A3 = 6, SLOT_A4 = 7, SLOT_A5 = 8,
       SLOT_OZ_SLICE = 9, SLOT_CERT = 10 };

void prof_drain(qe_hpsi_handle* h) {
  if (h->prof_spans.empty()) {
    h->prof_used = 0;
    return;
  }
  cudaEventSynchronize(h->prof_pool[h->prof_spans.back().e1]);
  for (const auto& sp : h->prof_spans) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, h->prof_pool[sp.e0], h->prof_pool[sp.e1]) == cudaSuccess) {
      h->prof_ms[sp.slot] += ms;
      h->prof_cnt[sp.slot] += 1;
    }
  }
  h->prof_spans.clear();
  h->prof_used = 0;
}
// returns the index of a freshly recorded event, or (size_t)-1 when timing is off
size_t prof_mark(qe_hpsi_handle* h, cudaStream_t st) {
  if (!h->prof_mode) return (size_t)-1;
  if (h->prof_used == h->prof_pool.size()) {
    if (h->prof_pool.size() >= 16384) {
      prof_drain(h);
    } else {
      cudaEvent_t e;
      if (cudaEventCreate(&e) != cudaSuccess) return (size_t)-1;
      try {
        h->prof_pool.push_back(e);
      } catch (...) {  // out of host memory: this span is simply not timed
        cudaEventDestroy(e);
        return (size_t)-1;
      }
    }
  }
  const size_t i = h->prof_used++;
  cudaEventRecord(h->prof_pool[i], st);
  return i;
}
void prof_span(qe_hpsi_handle* h, size_t e0, size_t e1, int slot) {
  if (e0 == (size_t)-1 || e1 == (size_t)-1 || e1 < e0) return;
  try {
    h->prof_spans.push_back({e0, e1, slot});
  } catch (...) {
  }
}

// ---------------------------------------------------------------------------------------------------------
// host geometry: reciprocal lattice and fractional k with a FIXED operation order so
// that the sphere test is reproducible bit for bit (compiled with -ffp-contract=off on the host side)
// ---------------------------------------------------------------------------------------------------------
struct SphereGeom {
  double b[3][3];
  double kap[3];
  double ecut;
  int n1, n2, n3;
};

void host_recip(const double at[9], double b[3][3], double* vol) {
  const double* a[3] = {at, at + 3, at + 6};
  double c[3][3];
  auto cross = [](const double* u, const double* v, double* o) {
    o[0] = u[1] * v[2] - u[2] * v[1];
    o[1] = u[2] * v[0] - u[0] * v[2];
    o[2] = u[0] * v[1] - u[1] * v[0];
  };
  cross(a[1], a[2], c[0]);
  cross(a[2], a[0], c[1]);
  cross(a[0], a[1], c[2]);
  volatile double t0 = a[0][0] * c[0][0], t1 = a[0][1] * c[0][1], t2 = a[0][2] * c[0][2];
  volatile double s = t0 + t1;
  *vol = s + t2;
  for (int j = 0; j < 3; ++j)
    for (int k = 0; k < 3; ++k) {
      volatile double num = TWO_PI * c[j][k];
      b[j][k] = num / *vol;
    }
}
void host_kfrac(const double at[9], const double xk[3], double kap[3]) {
  for (int j = 0; j < 3; ++j) {
    volatile double t0 = at[3 * j] * xk[0], t1 = at[3 * j + 1] * xk[1], t2 = at[3 * j + 2] * xk[2];
    volatile double s = t0 + t1;
    volatile double s2 = s + t2;
    kap[j] = s2 / TWO_PI;
  }
}

bool factor_235(int n) {
  if (n < 1) return false;
  for (int p : {2, 3, 5})
    while (n % p == 0) n /= p;
  return n == 1;
}

// fewest passes, then smallest largest radix; radices sorted descending
void plan_radices(int n, bool generic, std::vector<int>* best) {
  static const int fast_set[] = {16, 12, 10, 9, 8, 6, 5, 4, 3, 2};
  static const int gen_set[] = {5, 4, 3, 2};
  const int* set = generic ? gen_set : fast_set;
  const int nset = generic ? 4 : 10;
  std::vector<int> cur;
  best->clear();
  bool have = false;
  struct Rec {
    const int* set;
    int nset;
    std::vector<int>* cur;
    std::vector<int>* best;
    bool* have;
    void go(int rem, int maxr) {
      if (rem == 1) {
        bool better = !*have || cur->size() < best->size();
        if (!better && cur->size() == best->size()) {
          int mc = 0, mb = 0;
          for (int r : *cur) mc = std::max(mc, r);
          for (int r : *best) mb = std::max(mb, r);
          better = mc < mb;
        }
        if (better) {
          *best = *cur;
          *have = true;
        }
        return;
      }
      if (*have && cur->size() + 1 > best->size()) return;
      for (int i = 0; i < nset; ++i) {
        int r = set[i];
        if (r > maxr || rem % r) continue;
        cur->push_back(r);
        go(rem / r, r);
        cur->pop_back();
      }
    }
  } rec{set, nset, &cur, best, &have};
  if (n == 1) return;
  rec.go(n, 16);
}

// exp(+2 pi i k / n) in long double with exact quadrant reduction
void host_twiddles(int n, std::vector<double2>* out) {
  out->resize(n);
  const long double pi = 3.14159265358979323846264338327950288L;
  for (int k = 0; k < n; ++k) {
    int q = (8 * k + n) / (2 * n);
    int num = 4 * k - q * n;
    long double d = pi * (long double)num / (long double)(2 * n);
    long double c = num == 0 ? 1.0L : cosl(d), s = num == 0 ? 0.0L : sinl(d);
    long double re, im;
    switch (q & 3) {
      case 0: re = c; im = s; break;
      case 1: re = -s; im = c; break;
      case 2: re = -c; im = -s; break;
      default: re = s; im = -c; break;
    }
    (*out)[k] = make_double2((double)re, (double)im);
  }
}

// ---------------------------------------------------------------------------------------------------------
// a0: sphere enumeration kernels.  Each CTA of 256 threads owns 1024 consecutive linear indices (4 per thread,
// consecutive), so a block-ordered compaction keeps ascending idx = the canonical order.
// ---------------------------------------------------------------------------------------------------------
constexpr int SPH_NT = 256, SPH_PER = 4;

__device__ __forceinline__ int signed_idx(int i, int n) { return i >= (n + 1) / 2 ? i - n : i; }

__device__ __forceinline__ bool sphere_test(const SphereGeom& g, long long idx, int m[3], double* q2out) {
  const int i3 = (int)(idx % g.n3);
  const long long t = idx / g.n3;
  const int i2 = (int)(t % g.n2), i1 = (int)(t / g.n2);
  m[0] = signed_idx(i1, g.n1);
  m[1] = signed_idx(i2, g.n2);
  m[2] = signed_idx(i3, g.n3);
  const double x1 = __dadd_rn((double)m[0], g.kap[0]);
  const double x2 = __dadd_rn((double)m[1], g.kap[1]);
  const double x3 = __dadd_rn((double)m[2], g.kap[2]);
  double q[3];
#pragma unroll
  for (int c = 0; c < 3; ++c)
    q[c] = __dadd_rn(__dadd_rn(__dmul_rn(x1, g.b[0][c]), __dmul_rn(x2, g.b[1][c])), __dmul_rn(x3, g.b[2][c]));
  const double q2 = __dadd_rn(__dadd_rn(__dmul_rn(q[0], q[0]), __dmul_rn(q[1], q[1])), __dmul_rn(q[2], q[2]));
  *q2out = q2;
  return q2 <= g.ecut;
}

__global__ void __launch_bounds__(SPH_NT) k_sphere_count(SphereGeom g, long long ntot, int* __restrict__ counts) {
  const long long base = ((long long)blockIdx.x * SPH_NT + threadIdx.x) * SPH_PER;
  int cnt = 0;
#pragma unroll
  for (int e = 0; e < SPH_PER; ++e) {
    int m[3];
    double q2;
    if (base + e < ntot && sphere_test(g, base + e, m, &q2)) ++cnt;
  }
  __shared__ int wsum[SPH_NT / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) cnt += __shfl_down_sync(0xffffffffu, cnt, o);
  if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = cnt;
  __syncthreads();
  if (threadIdx.x == 0) {
    int s = 0;
    for (int w = 0; w < SPH_NT / 32; ++w) s += wsum[w];
    counts[blockIdx.x] = s;
  }
}

__global__ void __launch_bounds__(SPH_NT) k_sphere_fill(SphereGeom g, long long ntot, const int* __restrict__ offsets,
                                                        int* __restrict__ miller, int* __restrict__ fftidx,
                                                        double* __restrict__ g2kin) {
  const long long base = ((long long)blockIdx.x * SPH_NT + threadIdx.x) * SPH_PER;
  int m[SPH_PER][3];
  double q2[SPH_PER];
  bool in[SPH_PER];
  int cnt = 0;
#pragma unroll
  for (int e = 0; e < SPH_PER; ++e) {
    in[e] = base + e < ntot && sphere_test(g, base + e, m[e], &q2[e]);
    cnt += in[e] ? 1 : 0;
  }
  // exclusive scan of cnt over the block
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int incl = cnt;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int v = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += v;
  }
  __shared__ int wsum[SPH_NT / 32];
  if (lane == 31) wsum[warp] = incl;
  __syncthreads();
  int woff = 0;
  for (int w = 0; w < warp; ++w) woff += wsum[w];
  int pos = offsets[blockIdx.x] + woff + incl - cnt;
#pragma unroll
  for (int e = 0; e < SPH_PER; ++e) {
    if (in[e]) {
      miller[3 * (size_t)pos + 0] = m[e][0];
      miller[3 * (size_t)pos + 1] = m[e][1];
      miller[3 * (size_t)pos + 2] = m[e][2];
      fftidx[pos] = (int)(base + e);
      g2kin[pos] = q2[e];
      ++pos;
    }
  }
}

// V(r) -> V(r)/N in the padded [N1][N2][ldz] layout
__global__ void k_scale_pad_v(const double* __restrict__ vr, double* __restrict__ vs, int n3, int ldz, long long rows,
                              double scale) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= rows * ldz) return;
  const long long r = i / ldz;
  const int z = (int)(i - r * ldz);
  vs[i] = z < n3 ? vr[r * n3 + z] * scale : 0.0;
}

struct SphereOut {
  int npw = 0;
  int* miller = nullptr;
  int* fftidx = nullptr;
  double* g2kin = nullptr;
};

void free_sphere(SphereOut* s) {
  cudaFree(s->miller);
  cudaFree(s->fftidx);
  cudaFree(s->g2kin);
  *s = SphereOut{};
}

int validate_grid(const double at[9], const double xk[3], double ecutwfc, const int nr[3], SphereGeom* sg) {
  if (!at || !xk || !nr) return QE_HPSI_EINVAL;
  if (!(ecutwfc >= 0.0) || !std::isfinite(ecutwfc)) return QE_HPSI_EINVAL;
  double vol;
  host_recip(at, sg->b, &vol);
  if (!(std::fabs(vol) > 0.0) || !std::isfinite(vol)) return QE_HPSI_EINVAL;
  host_kfrac(at, xk, sg->kap);
  sg->ecut = ecutwfc;
  sg->n1 = nr[0];
  sg->n2 = nr[1];
  sg->n3 = nr[2];
  for (int j = 0; j < 3; ++j) {
    if (nr[j] < 1 || nr[j] > QE_HPSI_MAX_N || !factor_235(nr[j])) return QE_HPSI_EGRID;
    // |n_j + kappa_j| <= sqrt(ecut) |a_j| / 2 pi for every sphere point: the sphere must fit the box unwrapped
    const double* a = at + 3 * j;
    const double alen = std::sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
    const double ext = std::sqrt(ecutwfc) * alen / TWO_PI;
    const int nmax = (int)std::floor(ext + std::fabs(sg->kap[j]) + 1e-9);
    if (nr[j] < 2 * nmax + 1) return QE_HPSI_EGRID;
  }
  return QE_HPSI_OK;
}

int build_sphere(const SphereGeom& sg, cudaStream_t st, SphereOut* out) {
  qe_hpsi_handle* h = nullptr;
  const long long ntot = (long long)sg.n1 * sg.n2 * sg.n3;
  const int nblk = (int)((ntot + SPH_NT * SPH_PER - 1) / (SPH_NT * SPH_PER));
  std::vector<int> counts(nblk);  // (may throw: before any device allocation; the C entry points catch it)
  int* d_counts = nullptr;
  CU_TRY(h, cudaMalloc(&d_counts, sizeof(int) * (size_t)nblk));
  k_sphere_count<<<nblk, SPH_NT, 0, st>>>(sg, ntot, d_counts);
  cudaError_t e = cudaMemcpyAsync(counts.data(), d_counts, sizeof(int) * (size_t)nblk, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) {
    cudaFree(d_counts);
    g_last_cuda = (int)e;
    return QE_HPSI_ECUDA;
  }
  long long tot = 0;
  for (int i = 0; i < nblk; ++i) {
    int c = counts[i];
    counts[i] = (int)tot;
    tot += c;
  }
  out->npw = (int)tot;
  const size_t n = (size_t)std::max<long long>(tot, 1);
  e = cudaMalloc(&out->miller, sizeof(int) * 3 * n);
  if (e == cudaSuccess) e = cudaMalloc(&out->fftidx, sizeof(int) * n);
  if (e == cudaSuccess) e = cudaMalloc(&out->g2kin, sizeof(double) * n);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_counts, counts.data(), sizeof(int) * (size_t)nblk, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) {
    k_sphere_fill<<<nblk, SPH_NT, 0, st>>>(sg, ntot, d_counts, out->miller, out->fftidx, out->g2kin);
    e = cudaStreamSynchronize(st);
  }
  cudaFree(d_counts);
  if (e != cudaSuccess) {
    free_sphere(out);
    g_last_cuda = (int)e;
    return e == cudaErrorMemoryAllocation ? QE_HPSI_ENOMEM : QE_HPSI_ECUDA;
  }
  return QE_HPSI_OK;
}

template <typename T>
cudaError_t upload(T** dst, const std::vector<T>& v, cudaStream_t st) {
  cudaError_t e = cudaMalloc(dst, sizeof(T) * std::max<size_t>(v.size(), 1));
  if (e != cudaSuccess) return e;
  if (!v.empty()) e = cudaMemcpyAsync(*dst, v.data(), sizeof(T) * v.size(), cudaMemcpyHostToDevice, st);
  return e;
}

// cudaFuncSetAttribute is per device: keep the "done" state per device id, under a mutex (handles may be created from
// several host threads and on several devices of one process)
constexpr int MAX_DEVICES = 64;
bool g_attr_done[MAX_DEVICES] = {};
std::mutex g_attr_mutex;
long long g_int8_kmax = 0;  // qe_hpsi_test_set_int8_kmax
long long g_sym_min = 1LL << 20;  // qe_hpsi_test_set_sym_min: entries of beta from which the Gamma-symmetric mode is used
cudaError_t set_kernel_attrs() {
  int dev = 0, optin = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lock(g_attr_mutex);
  if (dev >= 0 && dev < MAX_DEVICES && g_attr_done[dev]) return cudaSuccess;
  e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (e != cudaSuccess) return e;
#define SET_SMEM(k)                                                                     \
  e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);      \
  if (e != cudaSuccess) return e;
  SET_SMEM(k_scatter_zinv);
  SET_SMEM(k_yinv);
  SET_SMEM(k_x_vmul);
  SET_SMEM(k_x_rho);
  SET_SMEM(k_yfwd);
  SET_SMEM(k_zfwd_gather);
  // the DMMA kernels keep their mbarriers in static shared memory: ask for what the tile pipeline needs, not for the device maximum
#define SET_ZG(Cfg, ...)                                                                                                 \
  e = cudaFuncSetAttribute(k_becp<Cfg, ##__VA_ARGS__>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM_BECP); \
  if (e != cudaSuccess) return e;                                                                                        \
  e = cudaFuncSetAttribute(k_vnl_add<Cfg, ##__VA_ARGS__>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM_VNL); \
  if (e != cudaSuccess) return e;
  SET_ZG(ZgV0);
  SET_ZG(ZgV0, true);
  SET_ZG(ZgS, true);
#undef SET_ZG
#define SET_ZT(Cfg, FORM)                                                                                                        \
  e = cudaFuncSetAttribute(k_becp_tma<Cfg, FORM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM_BECP + 1024); \
  if (e != cudaSuccess) return e;                                                                                              \
  e = cudaFuncSetAttribute(k_vnl_tma<Cfg, FORM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM_VNL);           \
  if (e != cudaSuccess) return e;
  SET_ZT(ZgV0, ZF_3M);
  SET_ZT(ZgV0, ZF_GAMMA);
  SET_ZT(ZgS, ZF_GAMMA);
  SET_ZT(ZgS, ZF_SYM);
  SET_ZT(ZgV0, ZF_SYM);
#undef SET_ZT
  e = cudaFuncSetAttribute(k_vnl_add<ZgV0, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZgV0::SMEM_VNL);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(k_vnl_add<ZgS, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZgS::SMEM_VNL);
  if (e != cudaSuccess) return e;
#undef SET_SMEM
  if (dev >= 0 && dev < MAX_DEVICES) g_attr_done[dev] = true;
  return cudaSuccess;
}

}  // namespace

// =========================================================================================================
// C ABI
// =========================================================================================================

extern "C" const char* qe_hpsi_strerror(int status) {
  switch (status) {
    case QE_HPSI_OK: return "ok";
    case QE_HPSI_EINVAL: return "invalid argument";
    case QE_HPSI_EGRID: return "unsupported FFT grid (factors other than 2,3,5, too large, or smaller than the sphere)";
    case QE_HPSI_ENOMEM: return "out of memory";
    case QE_HPSI_ECUDA: return "CUDA error (see qe_hpsi_last_error)";
    case QE_HPSI_ESTATE: return "invalid handle";
    default: return "unknown status";
  }
}

extern "C" int qe_hpsi_last_error(qe_hpsi_t h) { return h ? h->last_cuda : g_last_cuda.load(); }
extern "C" int64_t qe_hpsi_test_check_guards(qe_hpsi_t h) {
  if (!h) return QE_HPSI_ESTATE;
  if (cudaDeviceSynchronize() != cudaSuccess) return QE_HPSI_ECUDA;
  int64_t bad = 0;
  unsigned char buf[512];
  for (const auto& g : h->guards) {
    if (g.n > sizeof(buf) || cudaMemcpy(buf, g.p, g.n, cudaMemcpyDeviceToHost) != cudaSuccess) return QE_HPSI_ECUDA;
    for (size_t i = 0; i < g.n; ++i)
      if (buf[i] != 0xA5) {
        ++bad;
        break;
      }
  }
  return bad;
}
extern "C" int qe_hpsi_test_set_sym_min(int64_t entries) {
  g_sym_min = entries < 0 ? (1LL << 20) : entries;
  return QE_HPSI_OK;
}
extern "C" int qe_hpsi_test_set_int8_kmax(int64_t kmax) {
  if (kmax < 0) return QE_HPSI_EINVAL;
  g_int8_kmax = kmax;
  return QE_HPSI_OK;
}

extern "C" int qe_hpsi_gsphere(const double at[9], const double xk[3], double ecutwfc, const int nr[3], int64_t* npw,
                               int32_t* miller_host) {
  if (!npw) return QE_HPSI_EINVAL;
  SphereGeom sg;
  int rc = validate_grid(at, xk, ecutwfc, nr, &sg);
  if (rc) return rc;
  SphereOut so;
  try {
    rc = build_sphere(sg, nullptr, &so);
  } catch (const std::bad_alloc&) {
    rc = QE_HPSI_ENOMEM;
  }
  if (rc) return rc;
  *npw = so.npw;
  if (miller_host && so.npw > 0) {
    cudaError_t e = cudaMemcpy(miller_host, so.miller, sizeof(int) * 3 * (size_t)so.npw, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) {
      free_sphere(&so);
      g_last_cuda = (int)e;
      return QE_HPSI_ECUDA;
    }
  }
  free_sphere(&so);
  return QE_HPSI_OK;
}

extern "C" int qe_hpsi_destroy(qe_hpsi_t h) {
  if (!h) return QE_HPSI_OK;
  cudaFree(h->miller);
  cudaFree(h->fftidx);
  cudaFree(h->g2kin);
  cudaFree(h->stick_start);
  cudaFree(h->stick_i2);
  cudaFree(h->plane_stick);
  cudaFree(h->plane_i1);
  cudaFree(h->pw_pos);
  cudaFree(h->stick_lo);
  cudaFree(h->stick_hi);
  cudaFree(h->col_of);
  cudaFree(h->plane_of);
  cudaFree(h->plane_yhi);
  cudaFree(h->plane_ylo);
  cudaFree(h->zrow);
  cudaFree(h->vs);
  for (int j = 0; j < 3; ++j) cudaFree(h->tw[j]);
  cudaFree(h->w1);
  cudaFree(h->w2);
  cudaFree(h->beta_own);
  cudaFree(h->proj_blk0);
  cudaFree(h->proj_nh);
  cudaFree(h->proj_doff);
  cudaFree(h->dpk);
  cudaFree(h->partial);
  cudaFree(h->becp);
  cudaFree(h->dbecp);
  cudaFree(h->dbT);
  cudaFree(h->qpk);
  cudaFree(h->qbecp);
  cudaFree(h->qbT);
  cudaFree(h->ovl_partial);
  cudaFree(h->oz_a1);
  cudaFree(h->oz_a2);
  cudaFree(h->oz_b);
  cudaFree(h->oz_ep);
  cudaFree(h->oz_eg);
  cudaFree(h->oz_eb);
  cudaFree(h->oz_partial);
  cudaFree(h->sym_minus);
  cudaFree(h->sym_live);
  cudaFree(h->sym_cls);
  cudaFree(h->sym_cmask);
  cudaFree(h->sym_u);
  cudaFree(h->sym_e);
  cudaFree(h->sym_partial);
  cudaFree(h->cert_y);
  cudaFree(h->cert_v8);
  cudaFree(h->cert_psif);
  cudaFree(h->cert_vf);
  cudaFree(h->cert_part);
  cudaFree(h->cert_rel);
  cudaFree(h->cert_redo);
  cudaFree(h->cert_slot);
  cudaFree(h->cert_list);
  cudaFree(h->cert_count);
  cudaFree(h->partial_f);
  cudaFree(h->becp_f);
  cudaFree(h->dbecp_f);
  cudaFree(h->dbT_f);
  for (int i = 0; i < 2; ++i) {
    cudaFree(h->hbuf_psi[i]);
    cudaFree(h->hbuf_h[i]);
    if (h->ev_in[i]) cudaEventDestroy(h->ev_in[i]);
    if (h->ev_comp[i]) cudaEventDestroy(h->ev_comp[i]);
    if (h->ev_out[i]) cudaEventDestroy(h->ev_out[i]);
  }
  for (cudaEvent_t e : h->prof_pool) cudaEventDestroy(e);
  if (h->st_in) cudaStreamDestroy(h->st_in);
  if (h->st_comp) cudaStreamDestroy(h->st_comp);
  if (h->st_fft) cudaStreamDestroy(h->st_fft);
  if (h->ev_fork) cudaEventDestroy(h->ev_fork);
  if (h->ev_join) cudaEventDestroy(h->ev_join);
  if (h->st_out) cudaStreamDestroy(h->st_out);
  delete h;
  return QE_HPSI_OK;
}

namespace {

int env_int(const char* name, int dflt) {
  const char* s = std::getenv(name);
  if (!s || !*s) return dflt;
  return std::atoi(s);
}

// choose the split-K count of a6 so that (M tiles x N tiles x nsplit) fills whole waves of CTAs
// split-K plan of an a6-type contraction: ntile output tiles, K entries; fills whole waves of the SMs where K allows
void pick_split(int ntile, int klen, int num_sms, int bk, int* kchunk_out, int* nsplit_out) {
  // slices of at least 512 plane waves, unless that cannot even fill two waves (few projectors, small sphere): then 128
  int ksmax = std::max(1, klen / 512);
  if ((long long)ntile * ksmax < 2LL * num_sms) ksmax = std::max(1, klen / 128);
  int best = 1;
  double best_score = -1.0;
  for (int ks = 1; ks <= std::min(ksmax, 1024); ++ks) {
    const long long ctas = (long long)ntile * ks;
    const long long waves = (ctas + num_sms - 1) / num_sms;
    double eff = (double)ctas / (double)(waves * num_sms);
    if (waves < 2) eff *= 0.5 + 0.25 * (double)ctas / num_sms;  // prefer at least two waves when K allows
    const double score = eff - 1e-4 * ks;  // ties -> fewer splits (less partial traffic)
    if (score > best_score) {
      best_score = score;
      best = ks;
    }
    if (waves >= 16 && eff > 0.97) break;
  }
  int kchunk = (klen + best - 1) / best;
  kchunk = (kchunk + bk - 1) / bk * bk;
  if (kchunk < bk) kchunk = bk;
  *kchunk_out = kchunk;
  *nsplit_out = std::max(1, (klen + kchunk - 1) / kchunk);
}
void choose_split(qe_hpsi_handle* h) {
  // the Gamma-only handle contracts more than 64 bands on 64 x 128 tiles
  const int bn = (h->gamma && h->max_batch > ZgV0::BN) ? ZgS::BN : ZgV0::BN;
  const int ntile = ((h->nproj + ZgV0::BM - 1) / ZgV0::BM) * ((h->max_batch + bn - 1) / bn);
  pick_split(ntile, h->npw, h->num_sms, ZgV0::BK, &h->kchunk, &h->nsplit);
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda); looked up once, thread-safe
// (handles may be created, and maps of psi encoded, from several host threads)
using TmaEncodeFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                 CUtensorMapFloatOOBfill);
TmaEncodeFn tma_encoder() {
  static const TmaEncodeFn enc = [] {
    TmaEncodeFn f = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", (void**)&f, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess)
      f = nullptr;
    return f;
  }();
  return enc;
}

// FP64 matrix [rows][row_stride_bytes / 8] as a 2-D tensor map with boxes of box0 doubles x box1 rows, no swizzle, zero fill
bool make_map_f64(CUtensorMap* tm, const void* base, long long dim0, long long rows, long long row_stride_bytes, int box0, int box1,
                  bool swizzle128 = false) {
  const TmaEncodeFn enc = tma_encoder();
  if (!enc || dim0 <= 0 || rows <= 0 || (reinterpret_cast<uintptr_t>(base) & 15) || (row_stride_bytes & 15)) return false;
  cuuint64_t dims[2] = {(cuuint64_t)dim0, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)row_stride_bytes};
  cuuint32_t box[2] = {(cuuint32_t)box0, (cuuint32_t)box1};
  cuuint32_t estr[2] = {1, 1};
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
             swizzle128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// buffers of one a6-a7 pass on the FP64 tensor path: split-K partials, becp, dbecp, dbecp transposed
struct NlBufs {
  double2 *partial, *becp, *dbecp, *dbT;
};

// TMA-fed a6 / a8 of the general complex and Gamma-only forms (zgemm_tma_kernels.cuh): beta maps from create, the map of the
// K-contiguous B operand (psi [nb][ldpsi] or coefficient rows [nb][ldp]) encoded here, on the host, per call.  false = not
// launched (maps unavailable): the caller launches the cp.async kernel
template <class Cfg, int FORM>
bool becp_tma_launch(qe_hpsi_t h, const double2* psi, long long ldpsi, int nb, cudaStream_t st, double2* partial, const int* nb_dev) {
  CUtensorMap tb;
  if (!h->zg_tma || !make_map_f64(&tb, psi, 2LL * h->npw, nb, ldpsi * 16, 16, Cfg::BN, true)) return false;
  const int mt = (h->nproj + Cfg::BM - 1) / Cfg::BM, nt = (nb + Cfg::BN - 1) / Cfg::BN;
  k_becp_tma<Cfg, FORM><<<dim3(mt * nt, h->nsplit), Cfg::NT, Cfg::SMEM_BECP + 1024, st>>>(h->tm_g6_beta, tb, h->nproj, nb, h->npw, h->kchunk,
                                                                                          partial, h->ldc, nullptr, nb_dev, 0, 0);
  return true;
}
template <class Cfg, int FORM>
bool vnl_tma_launch(qe_hpsi_t h, const double2* bT, double2* hpsi, long long ldh, int nb, cudaStream_t st, const int* nb_dev,
                    int mt0 = 0, int mt1 = -1) {  // row tiles [mt0, mt1) of Cfg::BM rows; mt1 < 0: to the end
  CUtensorMap tb;
  if (!h->zg_tma || !make_map_f64(&tb, bT, 2LL * h->nproj, nb, (long long)h->ldp * 16, 8, Cfg::BN)) return false;
  const int mt = (h->npw + Cfg::BM - 1) / Cfg::BM, nt = (nb + Cfg::BN - 1) / Cfg::BN;
  if (mt1 < 0) mt1 = mt;
  if (mt1 > mt0)
    k_vnl_tma<Cfg, FORM><<<(unsigned)((mt1 - mt0) * nt), Cfg::NT, Cfg::SMEM_VNL, st>>>(h->tm_g8_beta, tb, h->nproj, h->npw, nb, hpsi, ldh,
                                                                                       nb_dev, nullptr, nullptr, 0, nullptr, mt0);
  return true;
}

template <class Cfg>
void becp_launch(qe_hpsi_t h, const double2* psi, long long ldpsi, int nb, cudaStream_t st, double2* partial, const int* nb_dev) {
  if (becp_tma_launch<Cfg, ZF_3M>(h, psi, ldpsi, nb, st, partial, nb_dev)) return;
  const int mt = (h->nproj + Cfg::BM - 1) / Cfg::BM, nt = (nb + Cfg::BN - 1) / Cfg::BN;
  k_becp<Cfg><<<dim3(mt * nt, h->nsplit), Cfg::NT, Cfg::SMEM_BECP, st>>>(h->beta, h->ldbeta, h->nproj, psi, ldpsi, nb,
                                                                         h->npw, h->kchunk, partial, h->ldc, nb_dev);
}
template <class Cfg>
void vnl_launch(qe_hpsi_t h, const double2* bT, double2* hpsi, long long ldh, int nb, cudaStream_t st, const int* nb_dev) {
  if (vnl_tma_launch<Cfg, ZF_3M>(h, bT, hpsi, ldh, nb, st, nb_dev)) return;
  const int mt = (h->npw + Cfg::BM - 1) / Cfg::BM, nt = (nb + Cfg::BN - 1) / Cfg::BN;
  if (mt == 0) return;
  k_vnl_add<Cfg><<<(unsigned)(mt * nt), Cfg::NT, Cfg::SMEM_VNL, st>>>(h->beta, h->ldbeta, h->nproj, h->npw, bT, h->ldp,
                                                                    nb, hpsi, ldh, nb_dev);
}

// a6 on the FP64 tensor path (complex handles): split-K partials of conj(beta) psi.  nb_dev != nullptr: the band count is
// min(nb, *nb_dev), read on the device (re-computation pass of QE_HPSI_PROJ_CERTIFY)
void becp_fp64(qe_hpsi_t h, const double2* psi, long long ldpsi, int nb, cudaStream_t st, double2* partial, const int* nb_dev) {
  becp_launch<ZgV0>(h, psi, ldpsi, nb, st, partial, nb_dev);
}
void vnl_fp64(qe_hpsi_t h, const double2* bT, double2* hpsi, long long ldh, int nb, cudaStream_t st, const int* nb_dev) {
  vnl_launch<ZgV0>(h, bT, hpsi, ldh, nb, st, nb_dev);
}
// a6-a8 entirely on the FP64 tensor path of a complex handle: out[b] += V_NL psi[b] (used by the certified path's
// re-computation and, at create, for its probe images)
void nonlocal_fp64(qe_hpsi_t h, const double2* psi, long long ldpsi, double2* out, long long ldo, int nb, cudaStream_t st,
                   const NlBufs& B, const int* nb_dev) {
  becp_fp64(h, psi, ldpsi, nb, st, B.partial, nb_dev);
  const dim3 rg((nb + 127) / 128, h->nproj);
  k_becp_reduce<<<rg, 128, 0, st>>>(B.partial, h->nsplit, h->nproj, h->ldc, nb, B.becp, nb_dev);
  k_dmul<<<rg, 128, 0, st>>>(B.becp, h->nproj, h->ldc, nb, h->proj_blk0, h->proj_nh, h->proj_doff, h->dpk, B.dbecp, B.dbT, h->ldp, nb_dev);
  vnl_fp64(h, B.dbT, out, ldo, nb, st, nb_dev);
}

// ---- projector contractions on tcgen05 int8 slices (ozaki_kernels.cuh) --------------------------
long long round_up(long long x, long long m) { return (x + m - 1) / m * m; }

// int8 planes [S][rows][kpad] as a 3-D tensor map (K bytes, rows, slice), SWIZZLE_64B boxes of box_rows x 64 bytes
bool oz_make_map(CUtensorMap* tm, void* base, long long kpad, long long rows, int S, long long slice_stride, int box_rows) {
  const TmaEncodeFn enc = tma_encoder();
  if (!enc) return false;
  cuuint64_t dims[3] = {(cuuint64_t)kpad, (cuuint64_t)rows, (cuuint64_t)S};
  cuuint64_t strides[2] = {(cuuint64_t)kpad, (cuuint64_t)slice_stride};
  cuuint32_t box[3] = {(cuuint32_t)oz::KB, (cuuint32_t)box_rows, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int S>
cudaError_t oz_prepare_t(qe_hpsi_handle* h, cudaStream_t st) {
  cudaError_t e = cudaSuccess;
  const void* kern[5] = {(const void*)oz::k_oz_gemm<S, 0>, (const void*)oz::k_oz_gemm<S, 1>, (const void*)oz::k_oz_gemm<S, 2>,
                         (const void*)oz::k_oz_gemm<S, 3>, (const void*)oz::k_oz_gemm<S, 4>};
  for (const void* k : kern)
    if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->oz_smem)) != cudaSuccess) return e;
  const long long k1 = h->oz_k1, k2 = h->oz_k2;
  // Gamma-symmetric mode: the planes cover the leading sym_m sphere entries only, and rows of class 1 are sliced as i*beta
  const long long ksph = h->sym ? h->sym_m : h->npw;
  const unsigned char* cls = h->sym ? h->sym_cls : nullptr;
  // a6 operand: rows p scaled by 2^-ep[p]; a8 operand: rows g scaled by 2^-eg[g] (transposed beta)
  oz::k_oz_rowexp<<<h->nproj, 256, 0, st>>>(h->beta, h->ldbeta, ksph, h->oz_ep);
  if (h->oz_3m)
    oz::k_oz_slice3<S><<<dim3((unsigned)((h->oz_k1c / 16 + 127) / 128), h->nproj), 128, 0, st>>>(
        h->beta, h->ldbeta, h->npw, h->oz_ep, h->oz_a1, h->oz_k1c, (long long)h->nproj * h->oz_k1c, 3LL * h->nproj * h->oz_k1c, -1.0);
  else
    oz::k_oz_slice<S><<<dim3((unsigned)((k1 / 16 + 127) / 128), h->nproj), 128, 0, st>>>(h->beta, h->ldbeta, ksph, h->oz_ep, h->oz_a1,
                                                                                      k1, (long long)h->nproj * k1, 0, cls);
  oz::k_oz_colexp<<<(unsigned)((ksph + 127) / 128), 128, 0, st>>>(h->beta, h->ldbeta, h->nproj, ksph, h->oz_eg);
  if (h->oz_3m8) {
    if ((e = cudaFuncSetAttribute(oz::k_oz_vnl3<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->oz_smem)) != cudaSuccess) return e;
    oz::k_oz_slice_t3<S><<<dim3((unsigned)((h->npw + 127) / 128), (unsigned)(h->oz_k2c / 16)), 128, 0, st>>>(
        h->beta, h->ldbeta, h->nproj, h->npw, h->oz_eg, h->oz_a2, h->oz_k2c, (long long)h->npw * h->oz_k2c, 3LL * h->npw * h->oz_k2c);
  } else if (h->gamma || h->sym)  // real form: rows 2g + c, K = p
    oz::k_oz_slice_tp<S><<<dim3((unsigned)((ksph + 127) / 128), (unsigned)(k2 / 16)), 128, 0, st>>>(
        h->beta, h->ldbeta, h->nproj, ksph, h->oz_eg, h->oz_a2, k2, 2LL * ksph * k2, cls);
  else
    oz::k_oz_slice_t<S><<<dim3((unsigned)((h->npw + 127) / 128), (unsigned)(k2 / 16)), 128, 0, st>>>(
        h->beta, h->ldbeta, h->nproj, h->npw, h->oz_eg, h->oz_a2, k2, (long long)h->npw * k2);
  return cudaGetLastError();
}

// a6 on int8 slices: exponents + digits of psi (oz_becp_slice_t), then the level GEMM into oz_partial[split][nproj][ldc]
template <int S>
void oz_becp_slice_t(qe_hpsi_handle* h, const double2* psi, long long ldpsi, int nb, cudaStream_t st) {
  const long long k1 = h->oz_k1;
  if (h->sym) {  // psi = u + i v: 2 nb real-wavefunction rows over the leading sym_m entries (sym_kernels.cuh), one B row each
    sym::k_sym_merge<<<dim3((h->sym_m + 255) / 256, nb), 256, 0, st>>>(psi, ldpsi, h->sym_m, h->sym_minus, h->sym_u, h->sym_ldu);
    oz::k_oz_rowexp<<<2 * nb, 256, 0, st>>>(h->sym_u, h->sym_ldu, h->sym_m, h->oz_eb);
    oz::k_oz_slice<S><<<dim3((unsigned)((k1 / 16 + 127) / 128), 2 * nb), 128, 0, st>>>(h->sym_u, h->sym_ldu, h->sym_m, h->oz_eb, h->oz_b, k1,
                                                                                     2LL * h->max_batch * k1, 0);
    return;
  }
  oz::k_oz_rowexp<<<nb, 256, 0, st>>>(psi, ldpsi, h->npw, h->oz_eb);
  if (h->oz_3m) {  // planes Re, Im, (Re + Im) / 2 of every band
    oz::k_oz_slice3<S><<<dim3((unsigned)((h->oz_k1c / 16 + 127) / 128), nb), 128, 0, st>>>(
        psi, ldpsi, h->npw, h->oz_eb, h->oz_b, h->oz_k1c, (long long)h->max_batch * h->oz_k1c, 3LL * h->max_batch * h->oz_k1c, 1.0);
    return;
  }
  // Gamma-only: becp is real, one B row (psi_r, psi_i) per band; otherwise the (Re, Im) row pair
  oz::k_oz_slice<S><<<dim3((unsigned)((k1 / 16 + 127) / 128), nb), 128, 0, st>>>(psi, ldpsi, h->npw, h->oz_eb, h->oz_b, k1,
                                                                             2LL * h->max_batch * k1, h->gamma ? 0 : 1);
}
template <int S>
void oz_becp_gemm_t(qe_hpsi_handle* h, int nb, cudaStream_t st) {
  if (h->oz_3m) {
    const dim3 g3((nb + oz::BN - 1) / oz::BN, (h->nproj + oz::BM - 1) / oz::BM, h->oz_nsplit);
    const size_t slab = (size_t)h->nproj * h->ldc;
    for (int pl = 0; pl < 3; ++pl)
      oz::k_oz_gemm<S, 2><<<g3, oz::NT, h->oz_smem, st>>>(h->oz_tm_a3[pl], h->oz_tm_b3[pl], h->oz_stages, (int)(h->oz_k1c / oz::KB),
                                                         h->oz_kchunk, h->oz_ep, h->oz_eb, h->nproj, nb,
                                                         h->oz_partial + (size_t)pl * h->oz_nsplit * slab, h->ldc, (long long)slab, 0);
    return;
  }
  if (h->sym) {  // real form, 2 nb columns (u_b, v_b)
    const dim3 gs((2 * nb + oz::BN - 1) / oz::BN, (h->nproj + oz::BM - 1) / oz::BM, h->oz_nsplit);
    oz::k_oz_gemm<S, 2><<<gs, oz::NT, h->oz_smem, st>>>(h->oz_tm_a1, h->oz_tm_b1, h->oz_stages, (int)(h->oz_k1 / oz::KB), h->oz_kchunk,
                                                       h->oz_ep, h->oz_eb, h->nproj, 2 * nb, h->oz_partial, h->sym_ldc2,
                                                       (long long)h->nproj * h->sym_ldc2, 0);
    return;
  }
  const dim3 grid(((h->gamma ? 1 : 2) * nb + oz::BN - 1) / oz::BN, (h->nproj + oz::BM - 1) / oz::BM, h->oz_nsplit);
  auto kern = h->gamma ? oz::k_oz_gemm<S, 2> : oz::k_oz_gemm<S, 0>;
  kern<<<grid, oz::NT, h->oz_smem, st>>>(h->oz_tm_a1, h->oz_tm_b1, h->oz_stages, (int)(h->oz_k1 / oz::KB), h->oz_kchunk, h->oz_ep,
                                        h->oz_eb, h->nproj, nb, h->oz_partial, h->ldc, (long long)h->nproj * h->ldc, 0, nullptr);
}
// a8 on int8 slices: hpsi[b][g] += sum_p beta[p][g] bT[b][p]
template <int S>
void oz_vnl_slice_t(qe_hpsi_handle* h, const double2* bT, int nb, cudaStream_t st) {
  const long long k2 = h->oz_k2;
  if (h->sym) {  // rows (Re e, Im e) of every band from k_sym_coef (bT is ignored: the coefficients are in sym_e)
    oz::k_oz_rowexp<<<2 * nb, 256, 0, st>>>(h->sym_e, h->ldp, h->nproj, h->oz_eb);
    oz::k_oz_slice_re<S><<<dim3((unsigned)((k2 / 16 + 127) / 128), 2 * nb), 128, 0, st>>>(h->sym_e, h->ldp, h->nproj, h->oz_eb, h->oz_b, k2,
                                                                                        2LL * h->max_batch * k2);
    return;
  }
  oz::k_oz_rowexp<<<nb, 256, 0, st>>>(bT, h->ldp, h->nproj, h->oz_eb);
  if (h->oz_3m8)  // planes Re, Im, (Re + Im) / 2 of dbecp^T, K = p
    oz::k_oz_slice3<S><<<dim3((unsigned)((h->oz_k2c / 16 + 127) / 128), nb), 128, 0, st>>>(
        bT, h->ldp, h->nproj, h->oz_eb, h->oz_b, h->oz_k2c, (long long)h->max_batch * h->oz_k2c, 3LL * h->max_batch * h->oz_k2c, 1.0);
  else if (h->gamma)  // dbecp is real: K = p
    oz::k_oz_slice_re<S><<<dim3((unsigned)((k2 / 16 + 127) / 128), nb), 128, 0, st>>>(bT, h->ldp, h->nproj, h->oz_eb, h->oz_b, k2,
                                                                                  2LL * h->max_batch * k2);
  else
    oz::k_oz_slice<S><<<dim3((unsigned)((k2 / 16 + 127) / 128), nb), 128, 0, st>>>(bT, h->ldp, h->nproj, h->oz_eb, h->oz_b, k2,
                                                                               2LL * h->max_batch * k2, 2);
}
template <int S>
void oz_vnl_gemm_t(qe_hpsi_handle* h, double2* hpsi, long long ldh, int nb, cudaStream_t st) {
  const int nkb = (int)(h->oz_k2 / oz::KB);
  // the K ranges (int32 level sums must stay exact) accumulate into the same hpsi entries: one launch after the other
  if (h->oz_3m8) {
    oz::k_oz_vnl3<S><<<dim3((nb + oz::BN - 1) / oz::BN, (unsigned)((h->npw + oz::BM - 1) / oz::BM), 1), oz::NT, h->oz_smem, st>>>(
        h->oz_tm_a4[0], h->oz_tm_a4[1], h->oz_tm_a4[2], h->oz_tm_b4[0], h->oz_tm_b4[1], h->oz_tm_b4[2], h->oz_stages,
        (int)(h->oz_k2c / oz::KB), h->oz_eg, h->oz_eb, h->npw, nb, hpsi, ldh);
    return;
  }
  if (h->sym) {  // rows 2g + c over the leading sym_m entries, columns (X, Y) of every band; epilogue writes G and -G
    const long long mr = 2LL * h->sym_m;
    const dim3 gs((2 * nb + oz::BN - 1) / oz::BN, (unsigned)((mr + oz::BM - 1) / oz::BM), 1);
    for (int ks = 0; ks * h->oz_kchunk2 < nkb; ++ks)
      oz::k_oz_gemm<S, 4><<<gs, oz::NT, h->oz_smem, st>>>(h->oz_tm_a2, h->oz_tm_b2, h->oz_stages, nkb, h->oz_kchunk2, h->oz_eg, h->oz_eb, mr,
                                                         2 * nb, hpsi, ldh, 0, ks, h->sym_minus);
    return;
  }
  const long long mrows = (h->gamma ? 2LL : 1LL) * h->npw;  // Gamma-only: rows 2g + c of the planar transposed digits
  const dim3 grid(((h->gamma ? 1 : 2) * nb + oz::BN - 1) / oz::BN, (unsigned)((mrows + oz::BM - 1) / oz::BM), 1);
  auto kern = h->gamma ? oz::k_oz_gemm<S, 3> : oz::k_oz_gemm<S, 1>;
  for (int ks = 0; ks * h->oz_kchunk2 < nkb; ++ks)
    kern<<<grid, oz::NT, h->oz_smem, st>>>(h->oz_tm_a2, h->oz_tm_b2, h->oz_stages, nkb, h->oz_kchunk2, h->oz_eg, h->oz_eb, mrows, nb, hpsi,
                                          ldh, 0, ks, nullptr);
}
#define OZ_DISPATCH(S_, CALL)            \
  switch (S_) {                          \
    case 4: CALL(4); break;              \
    case 5: CALL(5); break;              \
    case 7: CALL(7); break;              \
    default: CALL(6); break;             \
  }

// plan + operand digit planes of the int8 path (flag QE_HPSI_PROJ_INT8; digits and 3M forms from the flag fields).  Any
// failure is returned: a handle never changes its accuracy class on its own.
cudaError_t setup_ozaki(qe_hpsi_handle* h, int max_batch, unsigned flags, cudaStream_t st) {
  if (h->nproj <= 0 || h->npw <= 0) return cudaSuccess;
  int S = (int)((flags >> 8) & 15u);
  if (S == 0) S = 7;
  cudaError_t e = cudaSuccess;
  // Gamma-symmetric mode (h->sym, sym_kernels.cuh): real forms over the leading sym_m sphere entries, like a Gamma-only handle
  const bool realf = h->gamma || h->sym;
  const long long ksph = h->sym ? h->sym_m : h->npw;  // sphere entries the digit planes cover
  const long long k1 = round_up(2LL * ksph, 128), k2 = round_up((realf ? 1LL : 2LL) * h->nproj, 128);
  // K range per CTA: int32 level sums must not overflow (qe_hpsi_test_set_int8_kmax lowers it: the multi-range paths on small cases)
  const long long kmax_t = g_int8_kmax;
  const long long kmax = kmax_t >= oz::KB ? std::min<long long>(oz::max_k_per_cta(S), kmax_t / oz::KB * oz::KB) : oz::max_k_per_cta(S);
  h->oz_k1 = k1;
  h->oz_k2 = k2;
  // 3M form of a6 (three real GEMMs instead of a real-form complex one: -25 % MMAs, three launches): pays from ~2^26 entries of beta
  const unsigned m3 = (flags >> 12) & 3u;  // 0 by size, 1 off, 2 a6 only, 3 a6 and a8 whatever the size
  h->oz_3m = !realf && (m3 == 0 ? (long long)h->nproj * h->npw >= (1LL << 26) : m3 >= 2);
  h->oz_k1c = round_up(h->npw, 128);
  h->oz_k2c = round_up(h->nproj, 128);
  // a8 in the 3M form: one exact-int32 K range, and enough K blocks per plane to amortise the three epilogues (measured: pays at
  // nproj = 1728, not at 1024)
  h->oz_3m8 = h->oz_3m && h->oz_k2c <= kmax && m3 != 2 && (h->oz_k2c >= 1536 || m3 == 3);
  const long long ka6 = h->oz_3m ? h->oz_k1c : k1;  // contraction length of one a6 GEMM (reals)
  const int stage = S * (oz::A_BYTES + oz::B_BYTES);
  h->oz_stages = std::min(oz::MAX_STAGES, (222 * 1024) / stage);
  h->oz_smem = (size_t)h->oz_stages * stage + 1024;  // + 1 KB: the kernel aligns its ring to 1024 bytes itself
  // split-K of a6: K ranges short enough for exact int32 sums, and enough CTAs for two waves
  const int nkb = (int)(ka6 / oz::KB);
  const long long tiles = (long long)(((h->oz_3m || h->gamma ? 1 : 2) * max_batch + oz::BN - 1) / oz::BN) * ((h->nproj + oz::BM - 1) / oz::BM);
  long long ns = (ka6 + kmax - 1) / kmax;
  ns = std::max(ns, (2LL * h->num_sms + tiles - 1) / tiles);
  ns = std::min<long long>(ns, std::max(1, nkb / 8));
  ns = std::max<long long>(ns, (ka6 + kmax - 1) / kmax);
  {  // a few more splits if that fills the last wave: cost = rounds of CTAs x K blocks per CTA (one CTA per SM)
    long long best = ns, best_cost = -1;
    for (long long c = ns; c <= ns + 40 && c <= std::max<long long>(ns, nkb / 8); ++c) {
      const long long cost = ((tiles * c + h->num_sms - 1) / h->num_sms) * ((nkb + c - 1) / c + 4);  // + 4: prologue / epilogue
      if (best_cost < 0 || cost < best_cost) best = c, best_cost = cost;
    }
    ns = best;
  }
  h->oz_kchunk = (int)((nkb + ns - 1) / ns);
  h->oz_nsplit = (nkb + h->oz_kchunk - 1) / h->oz_kchunk;
  h->oz_kchunk2 = (int)std::min<long long>(k2, kmax) / oz::KB;  // a8: sequential launches over K ranges of this many blocks
  const long long a2rows = (realf ? 2LL : 1LL) * ksph;
  const size_t a1 = h->oz_3m ? (size_t)S * 3 * h->nproj * h->oz_k1c : (size_t)S * h->nproj * k1, a2 = h->oz_3m8 ? (size_t)S * 3 * h->npw * h->oz_k2c : (size_t)S * a2rows * k2, bb = (size_t)S * 2 * max_batch * std::max(k1, k2);
  const size_t pc = (size_t)h->nproj * h->ldc * sizeof(double2) * h->oz_nsplit * (h->oz_3m ? 3 : (h->sym ? 2 : 1));
  if ((e = guarded_malloc(h, &h->oz_a1, a1)) != cudaSuccess || (e = guarded_malloc(h, &h->oz_a2, a2)) != cudaSuccess ||
      (e = guarded_malloc(h, &h->oz_b, bb)) != cudaSuccess || (e = guarded_malloc(h, &h->oz_partial, pc)) != cudaSuccess ||
      (e = guarded_malloc(h, &h->oz_ep, sizeof(int) * (size_t)h->nproj)) != cudaSuccess ||
      (e = guarded_malloc(h, &h->oz_eg, sizeof(int) * (size_t)h->npw)) != cudaSuccess ||
      (e = guarded_malloc(h, &h->oz_eb, sizeof(int) * 2 * (size_t)max_batch)) != cudaSuccess) {
    // the digit planes do not fit (or another CUDA error): qe_hpsi_create fails with QE_HPSI_ENOMEM / QE_HPSI_ECUDA; the buffers
    // allocated so far are released by qe_hpsi_destroy
    return e;
  }
  if ((e = cudaMemsetAsync(h->oz_b, 0, bb, st)) != cudaSuccess) return e;
  if (!oz_make_map(&h->oz_tm_a1, h->oz_a1, k1, h->nproj, S, (long long)h->nproj * k1, oz::BM) ||
      !oz_make_map(&h->oz_tm_a2, h->oz_a2, k2, a2rows, S, a2rows * k2, oz::BM) ||
      !oz_make_map(&h->oz_tm_b1, h->oz_b, k1, 2LL * max_batch, S, 2LL * max_batch * k1, oz::BN) ||
      !oz_make_map(&h->oz_tm_b2, h->oz_b, k2, 2LL * max_batch, S, 2LL * max_batch * k2, oz::BN))
    return cudaErrorNotSupported;
  if (h->oz_3m)
    for (int pl = 0; pl < 3; ++pl)
      if (!oz_make_map(&h->oz_tm_a3[pl], h->oz_a1 + (size_t)pl * h->nproj * h->oz_k1c, h->oz_k1c, h->nproj, S, 3LL * h->nproj * h->oz_k1c,
                       oz::BM) ||
          !oz_make_map(&h->oz_tm_b3[pl], h->oz_b + (size_t)pl * max_batch * h->oz_k1c, h->oz_k1c, max_batch, S,
                       3LL * max_batch * h->oz_k1c, oz::BN))
        return cudaErrorNotSupported;
  if (h->oz_3m8)
    for (int pl = 0; pl < 3; ++pl)
      if (!oz_make_map(&h->oz_tm_a4[pl], h->oz_a2 + (size_t)pl * h->npw * h->oz_k2c, h->oz_k2c, h->npw, S, 3LL * h->npw * h->oz_k2c,
                       oz::BM) ||
          !oz_make_map(&h->oz_tm_b4[pl], h->oz_b + (size_t)pl * max_batch * h->oz_k2c, h->oz_k2c, max_batch, S,
                       3LL * max_batch * h->oz_k2c, oz::BN))
        return cudaErrorNotSupported;
#define OZ_CALL(S_) e = oz_prepare_t<S_>(h, st)
  OZ_DISPATCH(S, OZ_CALL)
#undef OZ_CALL
  if (e != cudaSuccess) return e;
  h->oz_s = S;
  h->workspace_bytes += a1 + a2 + bb + pc;
  return cudaSuccess;
}

// nonlocal state of a handle whose npw is already set (K dimension of a6 / M dimension of a8): beta (copied or
// borrowed), D tables, split-K plan and workspaces.  Shared by qe_hpsi_create and qe_hpsi_gamma_create.
cudaError_t setup_nonlocal(qe_hpsi_handle* h, int nproj, const void* beta_dev, int64_t ldbeta, int nblocks,
                           const int32_t* blk_off_host, const double* d_host, long long d_total, int max_batch,
                           unsigned flags, cudaStream_t st) {
#define CR_TRY(expr)                     \
  do {                                   \
    cudaError_t e__ = (expr);            \
    if (e__ != cudaSuccess) return e__;  \
  } while (0)

    if (flags & QE_HPSI_BORROW_BETA) {
      h->beta = static_cast<const double2*>(beta_dev);
      h->ldbeta = ldbeta;
    } else {
      h->ldbeta = ((long long)h->npw + 7) / 8 * 8;
      CR_TRY(guarded_malloc(h, &h->beta_own, sizeof(double2) * (size_t)nproj * h->ldbeta));
      CR_TRY(cudaMemsetAsync(h->beta_own, 0, sizeof(double2) * (size_t)nproj * h->ldbeta, st));
      CR_TRY(cudaMemcpy2DAsync(h->beta_own, sizeof(double2) * h->ldbeta, beta_dev, sizeof(double2) * (size_t)ldbeta,
                               sizeof(double2) * (size_t)h->npw, (size_t)nproj, cudaMemcpyDeviceToDevice, st));
      h->beta = h->beta_own;
    }
    std::vector<int> blk0((size_t)nproj), nhv((size_t)nproj);
    std::vector<long long> doff((size_t)nproj);
    long long off = 0;
    for (int a = 0; a < nblocks; ++a) {
      const int q0 = blk_off_host[a], nh = blk_off_host[a + 1] - q0;
      for (int i = 0; i < nh; ++i) {
        blk0[q0 + i] = q0;
        nhv[q0 + i] = nh;
        doff[q0 + i] = off + (long long)i * nh;
      }
      off += (long long)nh * nh;
    }
    h->d_total = d_total;
    std::vector<double> dv(d_host, d_host + d_total);
    CR_TRY(upload(&h->proj_blk0, blk0, st));
    CR_TRY(upload(&h->proj_nh, nhv, st));
    CR_TRY(upload(&h->proj_doff, doff, st));
    CR_TRY(upload(&h->dpk, dv, st));
    h->ldc = (max_batch + 1) / 2 * 2;
    h->ldp = (nproj + 7) / 8 * 8;
    choose_split(h);
    const int forced = env_int("QE_HPSI_NSPLIT", 0);
    if (forced > 0) {
      constexpr int ZG_BK = ZgV0::BK;
      int kchunk = (h->npw + forced - 1) / forced;
      kchunk = std::max(ZG_BK, (kchunk + ZG_BK - 1) / ZG_BK * ZG_BK);
      h->kchunk = kchunk;
      h->nsplit = std::max(1, (h->npw + kchunk - 1) / kchunk);
    }
    const size_t pc = (size_t)nproj * h->ldc * sizeof(double2);
    CR_TRY(guarded_malloc(h, &h->partial, pc * h->nsplit));
    CR_TRY(guarded_malloc(h, &h->becp, pc));
    CR_TRY(guarded_malloc(h, &h->dbecp, pc));
    CR_TRY(guarded_malloc(h, &h->dbT, (size_t)max_batch * h->ldp * sizeof(double2)));
    CR_TRY(cudaMemsetAsync(h->dbT, 0, (size_t)max_batch * h->ldp * sizeof(double2), st));
    h->workspace_bytes += pc * (h->nsplit + 2) + (size_t)max_batch * h->ldp * sizeof(double2);
    // TMA-fed FP64 kernels: beta never moves, its two maps (K-contiguous tiles of a6, M-contiguous tiles of a8) are made once
    if (h->npw > 0 && env_int("QE_HPSI_ZG_TMA", 1))
      h->zg_tma = make_map_f64(&h->tm_g6_beta, h->beta, 2LL * h->npw, nproj, (long long)h->ldbeta * 16, 16, ZgV0::BM, true) &&
                  make_map_f64(&h->tm_g8_beta, h->beta, 2LL * h->npw, nproj, (long long)h->ldbeta * 16, 2 * ZgV0::LDA_M, ZgV0::BK);
    static_assert(ZgV0::BM == ZgS::BM && ZgV0::BK == ZgS::BK, "one set of beta maps serves both tile shapes");
  #undef CR_TRY
  return cudaSuccess;
}

// QE_HPSI_PROJ_CERTIFY: scratch arrays, the second set of a6-a7 buffers, and the probe images y_t = V_NL s_t computed on the
// FP64 tensor path.  Runs after setup_nonlocal; synchronises the stream.
cudaError_t setup_certify(qe_hpsi_handle* h, cudaStream_t st) {
#define CR_TRY(expr)                     \
  do {                                   \
    cudaError_t e__ = (expr);            \
    if (e__ != cudaSuccess) return e__;  \
  } while (0)
  const long long ld = round_up(h->npw, 8);
  h->cert_ld = ld;
  const size_t row = sizeof(double2) * (size_t)ld, mb = (size_t)h->max_batch;
  h->cert_nch = (int)std::max<long long>(1, std::min<long long>(64, (h->npw + 32767) / 32768));
  CR_TRY(guarded_malloc(h, &h->cert_y, row * cert::NPROBE));
  CR_TRY(guarded_malloc(h, &h->cert_v8, row * mb));
  CR_TRY(guarded_malloc(h, &h->cert_psif, row * mb));
  CR_TRY(guarded_malloc(h, &h->cert_vf, row * mb));
  CR_TRY(guarded_malloc(h, &h->cert_part, sizeof(double) * mb * h->cert_nch * cert::NVAL));
  CR_TRY(guarded_malloc(h, &h->cert_rel, sizeof(double) * mb));
  CR_TRY(guarded_malloc(h, &h->cert_redo, sizeof(int) * mb));
  CR_TRY(guarded_malloc(h, &h->cert_slot, sizeof(int) * mb));
  CR_TRY(guarded_malloc(h, &h->cert_list, sizeof(int) * mb));
  CR_TRY(guarded_malloc(h, &h->cert_count, sizeof(int)));
  const size_t pc = (size_t)h->nproj * h->ldc * sizeof(double2);
  CR_TRY(guarded_malloc(h, &h->partial_f, pc * h->nsplit));
  CR_TRY(guarded_malloc(h, &h->becp_f, pc));
  CR_TRY(guarded_malloc(h, &h->dbecp_f, pc));
  CR_TRY(guarded_malloc(h, &h->dbT_f, mb * h->ldp * sizeof(double2)));
  CR_TRY(cudaMemsetAsync(h->dbT_f, 0, mb * h->ldp * sizeof(double2), st));
  CR_TRY(cudaMemsetAsync(h->cert_y, 0, row * cert::NPROBE, st));
  CR_TRY(cudaMemsetAsync(h->cert_rel, 0, sizeof(double) * mb, st));
  CR_TRY(cudaMemsetAsync(h->cert_redo, 0, sizeof(int) * mb, st));
  CR_TRY(cudaMemsetAsync(h->cert_count, 0, sizeof(int), st));
  h->workspace_bytes += row * (cert::NPROBE + 3 * mb) + pc * (h->nsplit + 2) + mb * h->ldp * sizeof(double2);
  double2* sgn = nullptr;
  CR_TRY(cudaMalloc(&sgn, row * cert::NPROBE));
  cudaError_t e = cudaMemsetAsync(sgn, 0, row * cert::NPROBE, st);
  if (e == cudaSuccess) {
    cert::k_cert_signs<<<(unsigned)((h->npw + 255) / 256), 256, 0, st>>>(sgn, ld, h->npw);
    const NlBufs B{h->partial_f, h->becp_f, h->dbecp_f, h->dbT_f};
    for (int t0 = 0; t0 < cert::NPROBE; t0 += h->max_batch)
      nonlocal_fp64(h, sgn + (size_t)t0 * ld, ld, h->cert_y + (size_t)t0 * ld, ld, std::min(h->max_batch, cert::NPROBE - t0), st, B,
                    nullptr);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  }
  cudaFree(sgn);
  CR_TRY(e);
  h->certify = true;
#undef CR_TRY
  return cudaSuccess;
}


// Gamma-symmetric projector mode (sym_kernels.cuh): at k = 0, FP64 path.  Builds the -G map of the leading sphere entries,
// classifies every projector ON THE DEVICE by exact comparison, checks that D couples equal classes only, and allocates the
// real-form operands.  Leaves h->sym = false (general complex contraction) whenever any check fails; only CUDA errors are errors.
cudaError_t setup_symmetric(qe_hpsi_handle* h, const std::vector<int>& idx, const int nr[3], int nblocks,
                            const int32_t* blk_off_host, const double* d_host, bool int8_path, cudaStream_t st) {
#define CR_TRY(expr)                     \
  do {                                   \
    cudaError_t e__ = (expr);            \
    if (e__ != cudaSuccess) return e__;  \
  } while (0)
  const int n1 = nr[0], n2 = nr[1], n3 = nr[2];
  auto sgn = [](int i, int n) { return i >= (n + 1) / 2 ? i - n : i; };
  int M = 0;
  while (M < h->npw && (idx[M] / (n2 * n3)) < (n1 + 1) / 2) ++M;  // canonical order: n1 >= 0 comes first
  std::vector<int> minus((size_t)std::max(M, 1));
  for (int g = 0; g < M; ++g) {
    const int i3 = idx[g] % n3, i2 = (idx[g] / n3) % n2, i1 = idx[g] / (n2 * n3);
    const int m[3] = {sgn(i1, n1), sgn(i2, n2), sgn(i3, n3)};
    const bool keep = m[0] > 0 || (m[0] == 0 && (m[1] > 0 || (m[1] == 0 && m[2] >= 0)));
    if (!keep) {
      minus[g] = -1;
      continue;
    }
    if (m[0] == 0 && m[1] == 0 && m[2] == 0) {
      minus[g] = -2;
      continue;
    }
    const long long lin = ((long long)((n1 - m[0]) % n1) * n2 + (n2 - m[1]) % n2) * n3 + (n3 - m[2]) % n3;
    auto it = std::lower_bound(idx.begin(), idx.end(), (int)lin);
    if (it == idx.end() || *it != (int)lin) return cudaSuccess;  // sphere not closed under G -> -G: general path
    minus[g] = (int)(it - idx.begin());
  }
  CR_TRY(upload(&h->sym_minus, minus, st));
  {  // longest run of whole 16-row K tiles with minus = -1 only (the n1 = 0, n2 < 0 half plane): a6 skips it, U is zero there
    int best0 = 0, best1 = 0, run0 = -1;
    const int nt16 = M / ZgS::BK;
    for (int t = 0; t <= nt16; ++t) {
      bool dead = t < nt16;
      for (int r = 0; dead && r < ZgS::BK; ++r) dead = minus[(size_t)t * ZgS::BK + r] == -1;
      if (dead && run0 < 0) run0 = t;
      if (!dead && run0 >= 0) {
        if (t - run0 > best1 - best0) best0 = run0, best1 = t;
        run0 = -1;
      }
    }
    h->sym_dead0 = best0;
    h->sym_dead1 = best1;
  }
  {  // row tiles of the symmetric a8 that store something
    std::vector<int> live;
    for (int t = 0; t * ZgS::BM < M; ++t) {
      bool any = false;
      for (int r = t * ZgS::BM; !any && r < std::min(M, (t + 1) * ZgS::BM); ++r) any = minus[(size_t)r] != -1;
      if (any) live.push_back(t);
    }
    h->sym_nlive = (int)live.size();
    CR_TRY(upload(&h->sym_live, live, st));
    CR_TRY(cudaStreamSynchronize(st));  // live leaves scope
  }
  CR_TRY(guarded_malloc(h, &h->sym_cls, (size_t)h->nproj));
  sym::k_sym_classify<<<h->nproj, 256, 0, st>>>(h->beta, h->ldbeta, M, h->sym_minus, h->sym_cls);
  std::vector<unsigned char> cls((size_t)h->nproj);
  CR_TRY(cudaMemcpyAsync(cls.data(), h->sym_cls, (size_t)h->nproj, cudaMemcpyDeviceToHost, st));
  CR_TRY(cudaStreamSynchronize(st));
  for (unsigned char c : cls)
    if (c > 1) return cudaSuccess;  // a projector without the symmetry: general path
  long long off = 0;
  for (int a = 0; a < nblocks; ++a) {
    const int q0 = blk_off_host[a], nh = blk_off_host[a + 1] - q0;
    for (int i = 0; i < nh; ++i)
      for (int j = 0; j < nh; ++j)
        if (d_host[off + (long long)i * nh + j] != 0.0 && cls[q0 + i] != cls[q0 + j]) return cudaSuccess;  // D mixes the classes
    off += (long long)nh * nh;
  }
  {
    std::vector<unsigned> cm((size_t)(h->nproj + 15) / 16, 0u);
    for (int p_ = 0; p_ < h->nproj; ++p_)
      if (cls[(size_t)p_]) cm[(size_t)p_ / 16] |= 1u << (p_ % 16);
    CR_TRY(upload(&h->sym_cmask, cm, st));
    CR_TRY(cudaStreamSynchronize(st));  // cm leaves scope
  }
  h->sym_cls_host = cls;
  h->blk_off.assign(blk_off_host, blk_off_host + nblocks + 1);
  h->sym_wide = env_int("QE_HPSI_SYM_WIDE", 1);
  h->sym_m = M;
  h->sym_ldu = round_up(M, 8);
  h->sym_ldc2 = 2 * h->ldc;
  {  // own split-K plan: 2 max_batch real columns on the tiles the symmetric kernels use, K = the half sphere
    const int bn = h->sym_wide ? ZgS::BN : ZgV0::BN;
    const int ntile = ((h->nproj + ZgS::BM - 1) / ZgS::BM) * ((2 * h->max_batch + bn - 1) / bn);
    pick_split(ntile, M, h->num_sms, ZgS::BK, &h->sym_kchunk, &h->sym_nsplit);
    const int forced = env_int("QE_HPSI_SYM_NSPLIT", 0);
    if (forced > 0) {
      int kc = (M + forced - 1) / forced;
      kc = std::max((int)ZgS::BK, (kc + ZgS::BK - 1) / ZgS::BK * ZgS::BK);
      h->sym_kchunk = kc;
      h->sym_nsplit = std::max(1, (M + kc - 1) / kc);
    }
  }
  const size_t ub = sizeof(double2) * 2 * (size_t)h->max_batch * h->sym_ldu, eb = sizeof(double2) * 2 * (size_t)h->max_batch * h->ldp;
  const size_t pb = int8_path ? 16 : sizeof(double2) * (size_t)h->sym_nsplit * h->nproj * h->sym_ldc2;  // (the int8 path has its own)
  CR_TRY(guarded_malloc(h, &h->sym_u, ub));
  CR_TRY(guarded_malloc(h, &h->sym_e, eb));
  CR_TRY(guarded_malloc(h, &h->sym_partial, pb));
  CR_TRY(cudaMemsetAsync(h->sym_u, 0, ub, st));
  CR_TRY(cudaMemsetAsync(h->sym_e, 0, eb, st));
  h->workspace_bytes += ub + eb + pb;
  h->sym = true;
  // TMA-fed kernels of the FP64 path (64 x 128 tiles): beta and the two workspaces never move, so the maps are made once
  if (!int8_path && h->sym_wide && env_int("QE_HPSI_SYM_TMA", 1)) {
    const long long rb = (long long)h->ldbeta * 16;
    h->sym_tma = make_map_f64(&h->tm_a6_beta, h->beta, 2LL * M, h->nproj, rb, 16, ZgS::BM, true) &&
                 make_map_f64(&h->tm_a6_u, h->sym_u, 2LL * M, 2LL * h->max_batch, h->sym_ldu * 16, 16, ZgS::BN, true) &&
                 make_map_f64(&h->tm_a8_beta, h->beta, 2LL * M, h->nproj, rb, 2 * ZgS::LDA_M, ZgS::BK) &&
                 make_map_f64(&h->tm_a8_e, h->sym_e, 2LL * h->nproj, 2LL * h->max_batch, (long long)h->ldp * 16, 8, ZgS::BN);
    h->sym_tail = h->sym_tma && env_int("QE_HPSI_SYM_TAIL", 1) &&
                  make_map_f64(&h->tm_a8_e64, h->sym_e, 2LL * h->nproj, 2LL * h->max_batch, (long long)h->ldp * 16, 8, ZgV0::BN) &&
                  make_map_f64(&h->tm_a6_u64, h->sym_u, 2LL * M, 2LL * h->max_batch, h->sym_ldu * 16, 16, ZgV0::BN, true);
  }
#undef CR_TRY
  return cudaSuccess;
}

// create flags: known bits only, one accuracy class, int8 sub-fields only with QE_HPSI_PROJ_INT8, 4..7 digits
int validate_flags(unsigned flags, bool gamma) {
  const unsigned known = QE_HPSI_BORROW_BETA | QE_HPSI_GENERIC_FFT | QE_HPSI_FP64_DMMA | QE_HPSI_PROJ_INT8 | QE_HPSI_PROJ_CERTIFY |
                         QE_HPSI_NO_GAMMA_SYM | (15u << 8) | (3u << 12);
  if (flags & ~known) return QE_HPSI_EINVAL;
  if ((flags & QE_HPSI_FP64_DMMA) && (flags & QE_HPSI_PROJ_INT8)) return QE_HPSI_EINVAL;
  if (!(flags & QE_HPSI_PROJ_INT8) && (flags & (QE_HPSI_PROJ_CERTIFY | (15u << 8) | (3u << 12)))) return QE_HPSI_EINVAL;
  const unsigned dig = (flags >> 8) & 15u;
  if (dig != 0 && (dig < 4 || dig > 7)) return QE_HPSI_EINVAL;
  if (gamma && (flags & QE_HPSI_PROJ_CERTIFY)) return QE_HPSI_EINVAL;
  return QE_HPSI_OK;
}

int create_impl(qe_hpsi_t* out, qe_hpsi_handle** live, const double at[9], double ecutwfc, const double xk[3], const int nr[3],
                const double* vr_dev, int nproj, const void* beta_dev, int64_t ldbeta, int nblocks,
                const int32_t* blk_off_host, const double* d_host, int max_batch, unsigned flags, void* cuda_stream);

}  // namespace

// The C entry point never lets a C++ exception (std::bad_alloc of the host-side tables) cross the boundary
extern "C" int qe_hpsi_create(qe_hpsi_t* out, const double at[9], double ecutwfc, const double xk[3], const int nr[3],
                              const double* vr_dev, int nproj, const void* beta_dev, int64_t ldbeta, int nblocks,
                              const int32_t* blk_off_host, const double* d_host, int max_batch, unsigned flags,
                              void* cuda_stream) {
  if (!out) return QE_HPSI_EINVAL;
  *out = nullptr;
  qe_hpsi_handle* live = nullptr;
  int rc;
  try {
    rc = create_impl(out, &live, at, ecutwfc, xk, nr, vr_dev, nproj, beta_dev, ldbeta, nblocks, blk_off_host, d_host, max_batch,
                     flags, cuda_stream);
  } catch (const std::bad_alloc&) {
    rc = QE_HPSI_ENOMEM;
  } catch (...) {
    rc = QE_HPSI_ESTATE;
  }
  if (rc != QE_HPSI_OK) {
    if (live) qe_hpsi_destroy(live);
    *out = nullptr;
  }
  return rc;
}

namespace {

int create_impl(qe_hpsi_t* out, qe_hpsi_handle** live, const double at[9], double ecutwfc, const double xk[3], const int nr[3],
                const double* vr_dev, int nproj, const void* beta_dev, int64_t ldbeta, int nblocks,
                const int32_t* blk_off_host, const double* d_host, int max_batch, unsigned flags, void* cuda_stream) {
  if (!vr_dev || nproj < 0 || max_batch < 1) return QE_HPSI_EINVAL;
  int rc = validate_flags(flags, false);
  if (rc) return rc;
  SphereGeom sg;
  rc = validate_grid(at, xk, ecutwfc, nr, &sg);
  if (rc) return rc;
  long long d_total = 0;
  if (nproj > 0) {
    if (!beta_dev || !blk_off_host || !d_host || nblocks < 1) return QE_HPSI_EINVAL;
    if (blk_off_host[0] != 0 || blk_off_host[nblocks] != nproj) return QE_HPSI_EINVAL;
    for (int a = 0; a < nblocks; ++a) {
      const long long nh = (long long)blk_off_host[a + 1] - blk_off_host[a];
      if (nh <= 0) return QE_HPSI_EINVAL;
      d_total += nh * nh;
    }
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  qe_hpsi_handle* h = new (std::nothrow) qe_hpsi_handle();
  if (!h) return QE_HPSI_ENOMEM;
  *live = h;  // on any failure below the caller (qe_hpsi_create) destroys it
#define CR_TRY(expr)                                                             \
  do {                                                                           \
    cudaError_t e__ = (expr);                                                    \
    if (e__ != cudaSuccess) {                                                    \
      g_last_cuda = (int)e__;                                                    \
      (void)cudaGetLastError();                                                  \
      return e__ == cudaErrorMemoryAllocation ? QE_HPSI_ENOMEM : QE_HPSI_ECUDA;  \
    }                                                                            \
  } while (0)
  CR_TRY(cudaGetDevice(&h->device));
  CR_TRY(cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, h->device));
  CR_TRY(set_kernel_attrs());
  for (int j = 0; j < 3; ++j) h->nr[j] = nr[j];
  h->ldz = (nr[2] + 7) / 8 * 8;
  h->max_batch = max_batch;
  h->nproj = nproj;

  // ---- a0: sphere maps --------------------------------------------------------------------------------
  SphereOut so;
  rc = build_sphere(sg, st, &so);
  if (rc) return rc;
  h->npw = so.npw;
  h->miller = so.miller;
  h->fftidx = so.fftidx;
  h->g2kin = so.g2kin;
  if (nproj > 0 && ldbeta < h->npw) return QE_HPSI_EINVAL;
  std::vector<int> idx((size_t)h->npw);
  if (h->npw) CR_TRY(cudaMemcpy(idx.data(), h->fftidx, sizeof(int) * (size_t)h->npw, cudaMemcpyDeviceToHost));
  // sticks ((i1,i2) columns) and populated planes, in canonical order
  std::vector<int> stick_start, stick_i2, plane_stick, plane_i1, pw_pos((size_t)h->npw);
  {
    const int n2 = nr[1], n3 = nr[2];
    int last_col = -1, last_plane = -1;
    for (int ig = 0; ig < h->npw; ++ig) {
      const int col = idx[ig] / n3, i3 = idx[ig] - col * n3;
      if (col != last_col) {
        const int i1 = col / n2;
        if (i1 != last_plane) {
          plane_stick.push_back((int)stick_start.size());
          plane_i1.push_back(i1);
          last_plane = i1;
        }
        stick_start.push_back(ig);
        stick_i2.push_back(col - i1 * n2);
        last_col = col;
      }
      const int c = ((int)stick_start.size() - 1) % FFT_C;
      pw_pos[ig] = i3 * FFT_C + (c ^ (i3 & 7));
    }
    h->S = (int)stick_start.size();
    h->P = (int)plane_i1.size();
    stick_start.push_back(h->npw);
    plane_stick.push_back(h->S);
  }
  CR_TRY(upload(&h->stick_start, stick_start, st));
  CR_TRY(upload(&h->stick_i2, stick_i2, st));
  CR_TRY(upload(&h->plane_stick, plane_stick, st));
  CR_TRY(upload(&h->plane_i1, plane_i1, st));
  CR_TRY(upload(&h->pw_pos, pw_pos, st));
  // tables of the fast two-pass path: signed i3 range of every stick (its sphere points are one interval, the
  // sphere being convex), stick index of every (plane, i2) column, populated-plane index of every i1
  bool sticks_are_intervals = true;
  {
    const int n1 = nr[0], n2 = nr[1], n3 = nr[2];
    std::vector<int> lo((size_t)h->S), hi((size_t)h->S), col_of((size_t)h->P * n2, -1), plane_of((size_t)n1, -1);
    for (int s_ = 0; s_ < h->S; ++s_) {
      int l = n3, u = -n3;
      for (int ig = stick_start[s_]; ig < stick_start[s_ + 1]; ++ig) {
        const int i3 = idx[ig] % n3, m3 = i3 >= (n3 + 1) / 2 ? i3 - n3 : i3;
        l = std::min(l, m3);
        u = std::max(u, m3);
      }
      lo[s_] = l;
      hi[s_] = u;
      if (u - l + 1 != stick_start[s_ + 1] - stick_start[s_]) sticks_are_intervals = false;
    }
    for (int p_ = 0; p_ < h->P; ++p_) {
      plane_of[plane_i1[p_]] = p_;
      for (int s_ = plane_stick[p_]; s_ < plane_stick[p_ + 1]; ++s_) col_of[(size_t)p_ * n2 + stick_i2[s_]] = s_;
    }
    CR_TRY(upload(&h->stick_lo, lo, st));
    CR_TRY(upload(&h->stick_hi, hi, st));
    CR_TRY(upload(&h->col_of, col_of, st));
    CR_TRY(upload(&h->plane_of, plane_of, st));
    h->g2p.stick_lo = h->stick_lo;
    h->g2p.stick_hi = h->stick_hi;
    h->g2p.col_of = h->col_of;
    h->g2p.plane_of = h->plane_of;
    // wrapped-interval rule of the populated planes (Fft2pGeom::x_hi / x_lo), verified against the table
    {
      int hi = -1, lo = 0;
      for (int p_ = 0; p_ < h->P; ++p_) {
        if (plane_i1[p_] < (n1 + 1) / 2) hi = std::max(hi, plane_i1[p_]);
        else ++lo;
      }
      bool ok = (hi + 1) + lo == h->P;
      for (int i1 = 0; i1 < n1 && ok; ++i1) {
        const int want = i1 <= hi ? i1 : (i1 >= n1 - lo ? i1 - (n1 - h->P) : -1);
        ok = plane_of[(size_t)i1] == want;
      }
      h->g2p.x_hi = ok ? hi : -2;
      h->g2p.x_lo = ok ? lo : 0;
    }
    // the same rule per plane along i2 (Fft2pGeom::y_hi / y_lo), verified against col_of
    {
      std::vector<int> yhi((size_t)std::max(h->P, 1), -1), ylo((size_t)std::max(h->P, 1), 0);
      bool ok = true;
      for (int p_ = 0; p_ < h->P && ok; ++p_) {
        const int s0 = plane_stick[p_], cnt = plane_stick[p_ + 1] - s0;
        int hi = -1, lo = 0;
        for (int s_ = s0; s_ < s0 + cnt; ++s_) {
          if (stick_i2[s_] < (n2 + 1) / 2) hi = std::max(hi, stick_i2[s_]);
          else ++lo;
        }
        ok = (hi + 1) + lo == cnt;
        for (int i2 = 0; i2 < n2 && ok; ++i2) {
          const int want = i2 <= hi ? s0 + i2 : (i2 >= n2 - lo ? s0 + i2 - (n2 - cnt) : -1);
          ok = col_of[(size_t)p_ * n2 + i2] == want;
        }
        yhi[(size_t)p_] = hi;
        ylo[(size_t)p_] = lo;
      }
      h->g2p.y_hi = h->g2p.y_lo = nullptr;
      if (ok) {
        CR_TRY(upload(&h->plane_yhi, yhi, st));
        CR_TRY(upload(&h->plane_ylo, ylo, st));
        CR_TRY(cudaStreamSynchronize(st));  // the host vectors leave scope
        h->g2p.y_hi = h->plane_yhi;
        h->g2p.y_lo = h->plane_ylo;
      }
      CR_TRY(guarded_malloc(h, &h->zrow, sizeof(double2) * (size_t)h->ldz));
      CR_TRY(cudaMemsetAsync(h->zrow, 0, sizeof(double2) * (size_t)h->ldz, st));
      h->g2p.zrow = h->zrow;
    }
  }

  // ---- FFT plan ---------------------------------------------------------------------------------------
  FftGeom& g = h->geom;
  g.n1 = nr[0];
  g.n2 = nr[1];
  g.n3 = nr[2];
  g.ldz = h->ldz;
  g.npw = h->npw;
  g.S = h->S;
  g.P = h->P;
  g.ntz = (nr[2] + FFT_C - 1) / FFT_C;
  g.stick_start = h->stick_start;
  g.stick_i2 = h->stick_i2;
  g.plane_stick = h->plane_stick;
  g.plane_i1 = h->plane_i1;
  g.pw_pos = h->pw_pos;
  g.g2kin = h->g2kin;
  FftAxis* axes[3] = {&g.ax1, &g.ax2, &g.ax3};
  for (int j = 0; j < 3; ++j) {
    std::vector<int> rad;
    plan_radices(nr[j], (flags & QE_HPSI_GENERIC_FFT) != 0, &rad);
    if ((int)rad.size() > FFT_MAX_PASS) return QE_HPSI_EGRID;
    axes[j]->n = nr[j];
    axes[j]->npass = (int)rad.size();
    for (size_t p = 0; p < rad.size(); ++p) axes[j]->radix[p] = rad[p];
    std::vector<double2> tw;
    host_twiddles(nr[j], &tw);
    CR_TRY(upload(&h->tw[j], tw, st));
    axes[j]->tw = h->tw[j];
  }
  h->smem_z = 2 * (size_t)nr[2] * FFT_C * sizeof(double2);
  h->smem_y = 2 * (size_t)nr[1] * FFT_C * sizeof(double2);
  h->smem_x = 2 * (size_t)nr[0] * FFT_C * sizeof(double2) + (size_t)nr[0] * FFT_C * sizeof(double);

  if (!(flags & QE_HPSI_GENERIC_FFT) && sticks_are_intervals && env_int("QE_HPSI_FFT2P", 1)) {
    const int p3 = env_int("QE_HPSI_FFT3P", 0);  // bit j set: prefer the three-pass plan on axis j (tuning knob)
    const Fft2pEntry* e[3] = {fft2p_find(nr[0], p3 & 1), fft2p_find(nr[1], p3 & 2), fft2p_find(nr[2], p3 & 4)};
    if (e[0] && e[1] && e[2]) {
      for (int j = 0; j < 3; ++j) h->f2p[j] = e[j];
      h->smem_x2p = e[0]->smem_x;
      CR_TRY(cudaFuncSetAttribute((const void*)e[0]->x, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)e[0]->smem_x));
      for (int j = 1; j < 3; ++j) {
        if (!e[j]->smem_zy) continue;
        const void* fns[2] = {j == 1 ? (const void*)e[j]->yinv : (const void*)e[j]->zinv,
                              j == 1 ? (const void*)e[j]->yfwd : (const void*)e[j]->zfwd};
        for (const void* fn : fns)
          CR_TRY(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)e[j]->smem_zy));
      }
    }
  }

  // V(r)/N in the padded layout
  {
    const long long rows = (long long)nr[0] * nr[1];
    CR_TRY(guarded_malloc(h, &h->vs, sizeof(double) * (size_t)rows * h->ldz));
    const long long tot = rows * h->ldz;
    const double scale = 1.0 / ((double)nr[0] * (double)nr[1] * (double)nr[2]);
    k_scale_pad_v<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(vr_dev, h->vs, nr[2], h->ldz, rows, scale);
    CR_TRY(cudaGetLastError());
    g.vs = h->vs;
  }

  // FFT workspace: sub-chunks of fft_nb bands (workspace budget QE_HPSI_FFT_WS_MB, default up to 12 GB)
  {
    const size_t per_band = ((size_t)h->S + (size_t)h->P * nr[1]) * h->ldz * sizeof(double2);
    // Measured on B200 (profiles/r1b): the chain gets faster with more bands per launch up to ~32 (fewer partial
    // waves, V(r) reused across the bands of a sub-chunk in a3); L2 residency of one band's workspace is worth less.
    // Capture G: one sub-chunk per call is best on every config (cfg 2: 15.7 -> 14.6 ms per 512 bands, cfg 4: 10.6 -> 10.4 ms per
    // 128), so the default budget is 12 GB, but never more than a quarter of what is free on the device right now.
    size_t mem_free = 0, mem_total = 0;
    if (cudaMemGetInfo(&mem_free, &mem_total) != cudaSuccess) mem_free = (size_t)10 << 30;
    const size_t dflt_mb = std::max<size_t>(256, std::min<size_t>(12288, (mem_free / 4) >> 20));
    const size_t budget = (size_t)env_int("QE_HPSI_FFT_WS_MB", (int)dflt_mb) << 20;
    long long nbf = per_band ? (long long)(budget / per_band) : max_batch;
    nbf = std::max<long long>(1, std::min<long long>(nbf, max_batch));
    const int forced = env_int("QE_HPSI_FFT_NB", 0);
    if (forced > 0) nbf = std::min(forced, max_batch);
    h->fft_nb = (int)nbf;
    CR_TRY(guarded_malloc(h, &h->w1, std::max<size_t>(16, (size_t)h->fft_nb * h->S * h->ldz * sizeof(double2))));
    CR_TRY(guarded_malloc(h, &h->w2, std::max<size_t>(16, (size_t)h->fft_nb * h->P * nr[1] * h->ldz * sizeof(double2))));
    // pad columns i3 in [N3, ldz) are carried through the y and x passes of the fast path: keep them finite
    CR_TRY(cudaMemsetAsync(h->w1, 0, std::max<size_t>(16, (size_t)h->fft_nb * h->S * h->ldz * sizeof(double2)), st));
    CR_TRY(cudaMemsetAsync(h->w2, 0, std::max<size_t>(16, (size_t)h->fft_nb * h->P * nr[1] * h->ldz * sizeof(double2)), st));
    h->workspace_bytes += (size_t)h->fft_nb * per_band;
    // x pass: one CTA per (i2, i3 tile) loops over the bands of the sub-chunk; split the band loop over
    // gridDim.y only as far as needed to give every SM a few CTAs
    if (h->f2p[0] && h->f2p[0]->rb > 1 && h->P > 0 && h->P <= 256 && h->g2p.x_hi != -2 && env_int("QE_HPSI_X_TMA", 1)) {
      const Fft2tEntry* et = fft2t_find(nr[0], h->f2p[0]->ra, h->f2p[0]->rb, h->f2p[0]->smem_zy != 0);
      h->x_one_tile = h->f2p[0]->smem_zy == 0 ? env_int("QE_HPSI_X_ONE_TILE", 1) : 0;
      const size_t sm = fft2t_smem(nr[0], h->P, h->f2p[0]->smem_zy == 0, h->x_one_tile != 0);
      const TmaEncodeFn enc = tma_encoder();
      if (et && sm <= (size_t)110 * 1024 && enc) {
        const cuuint64_t row = (cuuint64_t)nr[1] * h->ldz;  // complex elements per plane
        cuuint64_t dims[3] = {row * 2, (cuuint64_t)h->P, (cuuint64_t)h->fft_nb};
        cuuint64_t strides[2] = {row * sizeof(double2), row * sizeof(double2) * (cuuint64_t)h->P};
        cuuint32_t box[3] = {2 * FFT_C, (cuuint32_t)h->P, 1};
        cuuint32_t estr[3] = {1, 1, 1};
        if (enc(&h->tmap_w2, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, h->w2, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS &&
            cudaFuncSetAttribute((const void*)et->x, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm) == cudaSuccess) {
          h->x_tma = et->x;
          // quarter pruning: every populated plane in [0, N/4) or [3N/4, N) (x_hi, x_lo of the wrapped-interval rule)
          const int n1 = nr[0];
          if (et->xh && h->f2p[0]->smem_zy == 0 && env_int("QE_HPSI_X_HALF", 1) && 4 * (h->g2p.x_hi + 1) <= n1 && 4 * h->g2p.x_lo <= n1 &&
              cudaFuncSetAttribute((const void*)et->xh, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm) == cudaSuccess) {
            h->x_tma = et->xh;
            h->x_half = 1;
          }
          h->smem_xt = sm;
          const size_t smr = fft2t_smem_rho(nr[0], h->P);
          const K2tRho kr = (h->x_half && et->rhoh) ? et->rhoh : et->rho;
          if (kr && smr <= (size_t)110 * 1024 &&
              cudaFuncSetAttribute((const void*)kr, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smr) == cudaSuccess) {
            h->rho_tma = kr;
            h->smem_rho = smr;
          }
        }
      }
      (void)cudaGetLastError();  // a failed probe falls back to k2p_x_vmul
    }
    if (h->f2p[2] && h->f2p[2]->smem_zy == 0 && h->f2p[2]->rb > 1 && env_int("QE_HPSI_Z_TMA", 1)) {
      const Fft2tEntry* et = fft2t_find(nr[2], h->f2p[2]->ra, h->f2p[2]->rb, false);
      const size_t sm = fft2t_smem_z(nr[2]);
      if (et && et->zinv && sm <= (size_t)100 * 1024 &&
          cudaFuncSetAttribute((const void*)et->zinv, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm) == cudaSuccess &&
          cudaFuncSetAttribute((const void*)et->zfwd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm) == cudaSuccess) {
        const int m = env_int("QE_HPSI_Z_TMA", 1);  // bit 0: a1, bit 1: a5 (default 1 -> both via the mask below)
        h->z_tma_inv = (m == 1 || (m & 2)) ? et->zinv : nullptr;
        h->z_tma_fwd = (m == 1 || (m & 4)) ? et->zfwd : nullptr;
        h->smem_zt = sm;
      }
      (void)cudaGetLastError();
    }
    // (fewer splits = V(r) reused over more bands), choosing the split that fills whole waves of resident CTAs
    const long long xt = (long long)nr[1] * g.ntz;
    int occ = 0;
    if (h->x_tma)
      CR_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, h->x_tma, h->f2p[0]->nthreads, h->smem_xt));
    else if (h->f2p[0])
      CR_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, h->f2p[0]->x, h->f2p[0]->nthreads, h->smem_x2p));
    else
      CR_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_x_vmul, FFT_NT, h->smem_x));
    const long long slots = (long long)std::max(occ, 1) * h->num_sms;
    int best = 1;
    double best_score = -1.0;
    for (int sp = 1; sp <= std::min(h->fft_nb, 8); ++sp) {
      const long long ctas = xt * sp, waves = (ctas + slots - 1) / slots;
      const double score = (double)ctas / (double)(waves * slots) - 0.01 * (sp - 1);
      if (score > best_score) {
        best_score = score;
        best = sp;
      }
    }
    h->x_split = env_int("QE_HPSI_X_SPLIT", best);
    h->x_split = std::max(1, std::min(h->x_split, h->fft_nb));
  }

  h->overlap = env_int("QE_HPSI_OVERLAP", 0);
  if (h->overlap) {
    CR_TRY(cudaStreamCreateWithFlags(&h->st_fft, cudaStreamNonBlocking));
    CR_TRY(cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming));
    CR_TRY(cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming));
  }

  // ---- nonlocal ---------------------------------------------------------------------------------------
  if (nproj > 0)
    CR_TRY(setup_nonlocal(h, nproj, beta_dev, ldbeta, nblocks, blk_off_host, d_host, d_total, max_batch, flags, st));
  // (below ~1e6 entries of beta the step is launch-latency bound and the two extra small kernels of the symmetric form cost more
  // than the contraction saves: same FP64 arithmetic either way, so this size rule is a scheduling choice, not an accuracy one)
  if (nproj > 0 && h->npw > 0 && !(flags & QE_HPSI_NO_GAMMA_SYM) && sg.kap[0] == 0.0 && sg.kap[1] == 0.0 && sg.kap[2] == 0.0 &&
      (long long)nproj * h->npw >= g_sym_min)
    CR_TRY(setup_symmetric(h, idx, nr, nblocks, blk_off_host, d_host, (flags & QE_HPSI_PROJ_INT8) != 0, st));
  if (nproj > 0 && (flags & QE_HPSI_PROJ_INT8)) CR_TRY(setup_ozaki(h, max_batch, flags, st));
  if ((flags & QE_HPSI_PROJ_CERTIFY) && h->oz_s) CR_TRY(setup_certify(h, st));
  // NEXT-3: split-K workspace of qe_hpsi_overlap; K slices depend on npw only, so an element's bits do not depend on how many
  // rows / columns a call has (chunks of 512 x 128)
  if (h->npw > 0) {
    const int ns0 = std::max(1, std::min(32, h->npw / 2048));
    int kchunk = (h->npw + ns0 - 1) / ns0;
    kchunk = std::max(ZgV0::BK, (kchunk + ZgV0::BK - 1) / ZgV0::BK * ZgV0::BK);
    h->ovl_kchunk = kchunk;
    h->ovl_ns = std::max(1, (h->npw + kchunk - 1) / kchunk);
    CR_TRY(guarded_malloc(h, &h->ovl_partial, sizeof(double2) * (size_t)h->ovl_ns * 512 * 128));
    h->workspace_bytes += sizeof(double2) * (size_t)h->ovl_ns * 512 * 128;
  }
  CR_TRY(cudaStreamSynchronize(st));
#undef CR_TRY
  *live = nullptr;
  *out = h;
  return QE_HPSI_OK;
}

}  // namespace

namespace {

int check_apply_args(qe_hpsi_t h, const void* psi, int64_t ldpsi, void* hpsi, int64_t ldhpsi, int nbands) {
  if (!h) return QE_HPSI_ESTATE;
  if (nbands < 0) return QE_HPSI_EINVAL;
  if (nbands == 0) return QE_HPSI_OK;
  if (!psi || !hpsi || ldpsi < h->npw || ldhpsi < h->npw) return QE_HPSI_EINVAL;
  // complex128 rows are moved in 16-byte units (cp.async, TMA, double2 loads): a pointer that is only 8-byte aligned is an error
  if ((reinterpret_cast<uintptr_t>(psi) | reinterpret_cast<uintptr_t>(hpsi)) & 15u) return QE_HPSI_EINVAL;
  const char* a0 = static_cast<const char*>(psi);
  const char* a1 = a0 + ((size_t)(nbands - 1) * ldpsi + h->npw) * sizeof(double2);
  const char* b0 = static_cast<const char*>(hpsi);
  const char* b1 = b0 + ((size_t)(nbands - 1) * ldhpsi + h->npw) * sizeof(double2);
  if (a0 < b1 && b0 < a1) return QE_HPSI_EINVAL;
  return QE_HPSI_OK;
}

// a1-a5 for nb bands (nb <= max_batch), processed in sub-chunks of fft_nb bands
int launch_local(qe_hpsi_t h, const double2* psi, long long ldpsi, double2* hpsi, long long ldh, int nb, cudaStream_t st) {
  const FftGeom& g = h->geom;
  if (h->npw == 0) return QE_HPSI_OK;
  const unsigned zt = (unsigned)((g.S + FFT_C - 1) / FFT_C);
  const unsigned yt = (unsigned)(g.P * g.ntz);
  const unsigned xt = (unsigned)(g.n2 * g.ntz);
  // equal sub-chunks (128 bands at fft_nb = 36 go as 4 x 32, not 36 + 36 + 36 + 20)
  const int nsub = (nb + h->fft_nb - 1) / h->fft_nb, per = (nb + nsub - 1) / nsub;
  for (int b0 = 0; b0 < nb; b0 += per) {
    const int n = std::min(per, nb - b0);
    const double2* p = psi + (size_t)b0 * ldpsi;
    double2* o = hpsi + (size_t)b0 * ldh;
    const bool fine = h->prof_mode == 2;
    const bool fast = h->f2p[0] != nullptr;
    const Fft2pEntry *ex = h->f2p[0], *ey = h->f2p[1], *ez = h->f2p[2];
    size_t m0 = fine ? prof_mark(h, st) : (size_t)-1;
    if (h->z_tma_inv)
      h->z_tma_inv<<<dim3(zt, n), ez->nthreads, h->smem_zt, st>>>(g, h->g2p, p, ldpsi, h->w1);
    else if (fast)
      ez->zinv<<<dim3(zt, n), ez->nthreads, ez->smem_zy, st>>>(g, h->g2p, p, ldpsi, h->w1);
    else
      k_scatter_zinv<<<dim3(zt, n), FFT_NT, h->smem_z, st>>>(g, p, ldpsi, h->w1);
    size_t m1 = fine ? prof_mark(h, st) : (size_t)-1;
    if (fast)
      ey->yinv<<<dim3(yt, n), ey->nthreads, ey->smem_zy, st>>>(g, h->g2p, h->w1, h->w2);
    else
      k_yinv<<<dim3(yt, n), FFT_NT, h->smem_y, st>>>(g, h->w1, h->w2);
    size_t m2 = fine ? prof_mark(h, st) : (size_t)-1;
    if (h->x_tma)
      h->x_tma<<<dim3(xt, std::min(n, h->x_split)), ex->nthreads, h->smem_xt, st>>>(g, h->g2p, h->tmap_w2, n, h->x_one_tile);
    else if (fast)
      ex->x<<<dim3(xt, std::min(n, h->x_split)), ex->nthreads, h->smem_x2p, st>>>(g, h->g2p, h->w2, n);
    else
      k_x_vmul<<<dim3(xt, std::min(n, h->x_split)), FFT_NT, h->smem_x, st>>>(g, h->w2, n);
    size_t m3 = fine ? prof_mark(h, st) : (size_t)-1;
    if (fast)
      ey->yfwd<<<dim3(yt, n), ey->nthreads, ey->smem_zy, st>>>(g, h->g2p, h->w2, h->w1);
    else
      k_yfwd<<<dim3(yt, n), FFT_NT, h->smem_y, st>>>(g, h->w2, h->w1);
    size_t m4 = fine ? prof_mark(h, st) : (size_t)-1;
    if (h->z_tma_fwd)
      h->z_tma_fwd<<<dim3(zt, n), ez->nthreads, h->smem_zt, st>>>(g, h->g2p, h->w1, p, ldpsi, o, ldh);
    else if (fast)
      ez->zfwd<<<dim3(zt, n), ez->nthreads, ez->smem_zy, st>>>(g, h->g2p, h->w1, p, ldpsi, o, ldh);
    else
      k_zfwd_gather<<<dim3(zt, n), FFT_NT, h->smem_z, st>>>(g, h->w1, p, ldpsi, o, ldh);
    if (fine) {
      size_t m5 = prof_mark(h, st);
      if (m5 != (size_t)-1 && m5 > m0) {  // a drain in between would have reset the indices
        prof_span(h, m0, m1, SLOT_A1);
        prof_span(h, m1, m2, SLOT_A2);
        prof_span(h, m2, m3, SLOT_A3);
        prof_span(h, m3, m4, SLOT_A4);
        prof_span(h, m4, m5, SLOT_A5);
      }
    }
  }
  CU_TRY(h, cudaGetLastError());
  return QE_HPSI_OK;
}

// a6-a7 for nb bands: becp, dbecp, dbT
int launch_becp(qe_hpsi_t h, const double2* psi, long long ldpsi, int nb, cudaStream_t st) {
  const size_t t0 = prof_mark(h, st);
  size_t ts = t0;
  if (h->oz_s) {
#define OZ_CALL(S_) oz_becp_slice_t<S_>(h, psi, ldpsi, nb, st)
    OZ_DISPATCH(h->oz_s, OZ_CALL)
#undef OZ_CALL
    ts = prof_mark(h, st);
    prof_span(h, t0, ts, SLOT_OZ_SLICE);
#define OZ_CALL(S_) oz_becp_gemm_t<S_>(h, nb, st)
    OZ_DISPATCH(h->oz_s, OZ_CALL)
#undef OZ_CALL
  } else if (h->gamma) {
    auto go = [&](auto cfg) {
      using Cfg = decltype(cfg);
      if (becp_tma_launch<Cfg, ZF_GAMMA>(h, psi, ldpsi, nb, st, h->partial, nullptr)) return;
      const int mt = (h->nproj + Cfg::BM - 1) / Cfg::BM, nt = (nb + Cfg::BN - 1) / Cfg::BN;
      k_becp<Cfg, true><<<dim3(mt * nt, h->nsplit), Cfg::NT, Cfg::SMEM_BECP, st>>>(h->beta, h->ldbeta, h->nproj, psi, ldpsi, nb,
                                                                                   h->npw, h->kchunk, h->partial, h->ldc);
    };
    if (nb > 64) go(ZgS{}); else go(ZgV0{});  // 64 x 128 tiles from 65 bands on (same sums in the same order: same bits)
  } else if (h->sym) {
    // Gamma-symmetric projector mode: psi = u + i v as 2 nb real-wavefunction columns over the leading sym_m sphere entries
    sym::k_sym_merge<<<dim3((h->sym_m + 255) / 256, nb), 256, 0, st>>>(psi, ldpsi, h->sym_m, h->sym_minus, h->sym_u, h->sym_ldu);
    auto go = [&](auto cfg) {
      using Cfg = decltype(cfg);
      const int mt = (h->nproj + Cfg::BM - 1) / Cfg::BM, nt = (2 * nb + Cfg::BN - 1) / Cfg::BN;
      k_becp<Cfg, true><<<dim3(mt * nt, h->sym_nsplit), Cfg::NT, Cfg::SMEM_BECP, st>>>(h->beta, h->ldbeta, h->nproj, h->sym_u,
                                                                                       h->sym_ldu, 2 * nb, h->sym_m, h->sym_kchunk,
                                                                                       h->sym_partial, h->sym_ldc2, nullptr, h->sym_cls);
    };
    if (h->sym_tma && h->sym_tail && 2 * nb <= ZgV0::BN) {  // at most 32 bands: one 64-column tile instead of a half-empty 128-column one
      const int mt = (h->nproj + ZgV0::BM - 1) / ZgV0::BM;
      k_becp_tma<ZgV0, ZF_SYM><<<dim3(mt, h->sym_nsplit), ZgV0::NT, ZgV0::SMEM_BECP + 1024, st>>>(
          h->tm_a6_beta, h->tm_a6_u64, h->nproj, 2 * nb, h->sym_m, h->sym_kchunk, h->sym_partial, h->sym_ldc2, h->sym_cls, nullptr,
          h->sym_dead0, h->sym_dead1);
    } else if (h->sym_tma) {
      const int mt = (h->nproj + ZgS::BM - 1) / ZgS::BM, nt = (2 * nb + ZgS::BN - 1) / ZgS::BN;
      k_becp_tma<ZgS, ZF_SYM><<<dim3(mt * nt, h->sym_nsplit), ZgS::NT, ZgS::SMEM_BECP + 1024, st>>>(
          h->tm_a6_beta, h->tm_a6_u, h->nproj, 2 * nb, h->sym_m, h->sym_kchunk, h->sym_partial, h->sym_ldc2, h->sym_cls, nullptr,
          h->sym_dead0, h->sym_dead1);
    } else if (h->sym_wide) go(ZgS{}); else go(ZgV0{});
  } else
    becp_fp64(h, psi, ldpsi, nb, st, h->partial, nullptr);
  const size_t t1 = prof_mark(h, st);
  prof_span(h, ts, t1, SLOT_BECP);
  const dim3 rg((nb + 127) / 128, h->nproj);
  if (h->sym)
    sym::k_sym_reduce<<<rg, 128, 0, st>>>(h->oz_s ? h->oz_partial : h->sym_partial, h->oz_s ? h->oz_nsplit : h->sym_nsplit, h->nproj,
                                          h->sym_ldc2, nb, h->sym_cls, h->becp, h->ldc);
  else if (h->gamma)
    k_becp_reduce_gamma<<<rg, 128, 0, st>>>(h->oz_s ? h->oz_partial : h->partial, h->oz_s ? h->oz_nsplit : h->nsplit, h->nproj, h->ldc, nb,
                                            h->beta, h->ldbeta, psi, ldpsi,
                                            h->becp);
  else if (h->oz_s && h->oz_3m)
    oz::k_oz_reduce3<<<rg, 128, 0, st>>>(h->oz_partial, h->oz_nsplit, h->nproj, h->ldc, nb, h->becp);
  else
    k_becp_reduce<<<rg, 128, 0, st>>>(h->oz_s ? h->oz_partial : h->partial, h->oz_s ? h->oz_nsplit : h->nsplit, h->nproj, h->ldc, nb,
                                      h->becp);
  k_dmul<<<rg, 128, 0, st>>>(h->becp, h->nproj, h->ldc, nb, h->proj_blk0, h->proj_nh, h->proj_doff, h->dpk, h->dbecp,
                            h->dbT, h->ldp);
  if (h->sym)  // real coefficient rows (Re e, Im e) of the symmetric a8
    sym::k_sym_coef<<<rg, 128, 0, st>>>(h->dbecp, h->nproj, h->ldc, nb, h->sym_cls, h->sym_e, h->ldp);
  prof_span(h, t1, prof_mark(h, st), SLOT_DMUL);
  h->nb_last = nb;
  CU_TRY(h, cudaGetLastError());
  return QE_HPSI_OK;
}

// symmetric a8 on the TMA kernels: number of live row tiles the 64 x 128 launch takes; the rest (the last, partly filled wave)
// goes to a second launch on 64 x 64 tiles.  All of them when there is no tail worth splitting off.
int sym_a8_main_tiles(qe_hpsi_t h, int nb) {
  if (h->sym_tail && 2 * nb <= ZgV0::BN) return 0;  // at most 32 bands: every tile on 64 x 64
  const int nt = (2 * nb + ZgS::BN - 1) / ZgS::BN;
  const long long units = (long long)h->sym_nlive * nt;
  const long long full = units / h->num_sms * h->num_sms, rem = units - full;
  if (!h->sym_tail || full < 4LL * h->num_sms || rem == 0 || rem * 10 > 7LL * h->num_sms) return h->sym_nlive;
  return (int)(full / nt);
}

// a8
int launch_vnl_add(qe_hpsi_t h, const double2* bT, double2* hpsi, long long ldh, int nb, cudaStream_t st) {
  // Gamma-symmetric mode: the real coefficient rows of D becp are in sym_e already (launch_becp); for the q-term of
  // qe_hpsi_apply_hs they are rebuilt from qbecp when q couples equal classes only (else: general contraction, FP64 path only)
  bool use_sym = h->sym && bT == h->dbT;
  if (h->sym && bT == h->qbT && h->sym_q_ok) {
    sym::k_sym_coef<<<dim3((nb + 127) / 128, h->nproj), 128, 0, st>>>(h->qbecp, h->nproj, h->ldc, nb, h->sym_cls, h->sym_e, h->ldp);
    use_sym = true;
  }
  if (h->sym && h->oz_s && !use_sym) return QE_HPSI_ESTATE;  // the int8 planes of a symmetric handle hold the real forms only
  if (h->oz_s) {
    const size_t t0 = prof_mark(h, st);
#define OZ_CALL(S_) oz_vnl_slice_t<S_>(h, bT, nb, st)
    OZ_DISPATCH(h->oz_s, OZ_CALL)
#undef OZ_CALL
    const size_t ts = prof_mark(h, st);
    prof_span(h, t0, ts, SLOT_OZ_SLICE);
#define OZ_CALL(S_) oz_vnl_gemm_t<S_>(h, hpsi, ldh, nb, st)
    OZ_DISPATCH(h->oz_s, OZ_CALL)
#undef OZ_CALL
    prof_span(h, ts, prof_mark(h, st), SLOT_VNL);
  } else if (h->gamma) {
    auto go = [&](auto cfg) {
      using Cfg = decltype(cfg);
      if (vnl_tma_launch<Cfg, ZF_GAMMA>(h, bT, hpsi, ldh, nb, st, nullptr)) return;
      const int mt = (h->npw + Cfg::BM - 1) / Cfg::BM, nt = (nb + Cfg::BN - 1) / Cfg::BN;
      if (mt > 0)
        k_vnl_add<Cfg, true><<<(unsigned)(mt * nt), Cfg::NT, Cfg::SMEM_VNL, st>>>(h->beta, h->ldbeta, h->nproj, h->npw, bT,
                                                                                  h->ldp, nb, hpsi, ldh);
    };
    // 64 x 128 tiles from 65 bands on; a partly filled last wave of them runs on 64 x 64 tiles (see the symmetric form below)
    const int mtg = (h->npw + ZgS::BM - 1) / ZgS::BM, ntg = (nb + ZgS::BN - 1) / ZgS::BN;
    const long long ug = (long long)mtg * ntg, fullg = ug / h->num_sms * h->num_sms, remg = ug - fullg;
    if (nb > 64 && h->zg_tma && fullg >= 4LL * h->num_sms && remg > 0 && remg * 10 <= 7LL * h->num_sms &&
        vnl_tma_launch<ZgS, ZF_GAMMA>(h, bT, hpsi, ldh, nb, st, nullptr, 0, (int)(fullg / ntg))) {
      if (!vnl_tma_launch<ZgV0, ZF_GAMMA>(h, bT, hpsi, ldh, nb, st, nullptr, (int)(fullg / ntg), mtg)) return QE_HPSI_ECUDA;
    } else if (nb > 64) go(ZgS{}); else go(ZgV0{});
  } else if (use_sym) {
    // symmetric a8: X = sum_p b_p Re e_p, Y = sum_p b_p Im e_p over the half sphere; hpsi(G) += X + iY, hpsi(-G) += conj X + i conj Y
    auto go = [&](auto cfg) {
      using Cfg = decltype(cfg);
      const int mt = (h->sym_m + Cfg::BM - 1) / Cfg::BM, nt = (2 * nb + Cfg::BN - 1) / Cfg::BN;
      if (mt > 0)
        k_vnl_add<Cfg, true, true><<<(unsigned)(mt * nt), Cfg::NT, Cfg::SMEM_VNL, st>>>(h->beta, h->ldbeta, h->nproj, h->sym_m,
                                                                                        h->sym_e, h->ldp, 2 * nb, hpsi, ldh, nullptr,
                                                                                        h->sym_cmask, h->sym_minus);
    };
    if (h->sym_tma) {
      // live row tiles only; the last, partly filled wave of 64 x 128 tiles runs as 64 x 64 tiles instead (same sums, half the
      // time of that round)
      const int nt = (2 * nb + ZgS::BN - 1) / ZgS::BN;
      const int ma = sym_a8_main_tiles(h, nb);
      if (ma > 0)
        k_vnl_tma<ZgS, ZF_SYM><<<(unsigned)(ma * nt), ZgS::NT, ZgS::SMEM_VNL, st>>>(h->tm_a8_beta, h->tm_a8_e, h->nproj, h->sym_m, 2 * nb,
                                                                                    hpsi, ldh, nullptr, h->sym_cmask, h->sym_minus, 0,
                                                                                    h->sym_live, 0);
      if (ma < h->sym_nlive) {
        const int nt64 = (2 * nb + ZgV0::BN - 1) / ZgV0::BN;
        k_vnl_tma<ZgV0, ZF_SYM><<<(unsigned)((h->sym_nlive - ma) * nt64), ZgV0::NT, ZgV0::SMEM_VNL, st>>>(
            h->tm_a8_beta, h->tm_a8_e64, h->nproj, h->sym_m, 2 * nb, hpsi, ldh, nullptr, h->sym_cmask, h->sym_minus, 0, h->sym_live, ma);
      }
    } else if (h->sym_wide) go(ZgS{}); else go(ZgV0{});
  } else
    vnl_fp64(h, bT, hpsi, ldh, nb, st, nullptr);
  CU_TRY(h, cudaGetLastError());
  return QE_HPSI_OK;
}

// QE_HPSI_PROJ_CERTIFY, after a6-a7 of the int8 path: a8 into the scratch v8, the check, the FP64 re-computation of the bands
// that fail it, and hpsi[b] += (FP64 result or int8 result).  DESIGN.md section 5.7; kernels in cert_kernels.cuh.
int launch_vnl_certified(qe_hpsi_t h, const double2* psi, long long ldpsi, double2* hpsi, long long ldh, int nb, cudaStream_t st) {
  const long long ld = h->cert_ld;
  CU_TRY(h, cudaMemsetAsync(h->cert_v8, 0, sizeof(double2) * (size_t)nb * ld, st));
  int rc = launch_vnl_add(h, h->dbT, h->cert_v8, ld, nb, st);
  if (rc) return rc;
  const size_t t0 = prof_mark(h, st);
  const int gchunk = (int)((h->npw + h->cert_nch - 1) / h->cert_nch);
  cert::k_cert_probe<<<dim3(h->cert_nch, nb), cert::NT, 0, st>>>(h->cert_v8, ld, psi, ldpsi, h->cert_y, ld, h->npw, gchunk, h->cert_part,
                                                               h->cert_nch);
  cert::k_cert_decide<<<1, cert::NT, 0, st>>>(h->cert_part, h->cert_nch, nb, h->cert_tol, h->cert_rel, h->cert_redo, h->cert_slot,
                                            h->cert_list, h->cert_count);
  const unsigned gx = (unsigned)std::min<long long>((h->npw + 255) / 256, 64);
  cert::k_cert_gather<<<dim3(gx, nb), 256, 0, st>>>(psi, ldpsi, h->npw, h->cert_list, h->cert_count, h->cert_psif, h->cert_vf, ld);
  const NlBufs B{h->partial_f, h->becp_f, h->dbecp_f, h->dbT_f};
  nonlocal_fp64(h, h->cert_psif, ld, h->cert_vf, ld, nb, st, B, h->cert_count);
  cert::k_cert_commit<<<dim3(gx, nb), 256, 0, st>>>(h->cert_v8, h->cert_vf, ld, h->cert_redo, h->cert_slot, h->npw, hpsi, ldh);
  prof_span(h, t0, prof_mark(h, st), SLOT_CERT);
  CU_TRY(h, cudaGetLastError());
  return QE_HPSI_OK;
}

int apply_chunk(qe_hpsi_t h, const double2* psi, long long ldpsi, double2* hpsi, long long ldh, int nb, cudaStream_t st,
                bool local, bool nonlocal) {
  int rc = QE_HPSI_OK;
  const bool nl = nonlocal && h->nproj > 0 && h->npw > 0;
  if (h->prof_mode && h->prof_used + 24 > 16384) prof_drain(h);
  // a6-a7 and a1-a5 are independent (both only read psi): with QE_HPSI_OVERLAP=1 the FFT chain runs on an internal
  // stream forked from the caller's stream while the projector ZGEMM runs on the caller's stream; joined before a8.
  const bool fork = nl && local && h->overlap && h->st_fft && !h->prof_mode;
  if (fork) {
    CU_TRY(h, cudaEventRecord(h->ev_fork, st));
    CU_TRY(h, cudaStreamWaitEvent(h->st_fft, h->ev_fork, 0));
    rc = launch_local(h, psi, ldpsi, hpsi, ldh, nb, h->st_fft);
    if (rc) return rc;
    CU_TRY(h, cudaEventRecord(h->ev_join, h->st_fft));
  }
  if (nl) {
    rc = launch_becp(h, psi, ldpsi, nb, st);
    if (rc) return rc;
  }
  if (fork) {
    CU_TRY(h, cudaStreamWaitEvent(st, h->ev_join, 0));
  } else if (local) {
    const size_t t0 = h->prof_mode == 1 ? prof_mark(h, st) : (size_t)-1;
    rc = launch_local(h, psi, ldpsi, hpsi, ldh, nb, st);
    if (rc) return rc;
    if (h->prof_mode == 1) prof_span(h, t0, prof_mark(h, st), SLOT_FFT);
  }
  if (nl) {
    if (h->certify) return launch_vnl_certified(h, psi, ldpsi, hpsi, ldh, nb, st);
    const size_t t0 = h->oz_s ? (size_t)-1 : prof_mark(h, st);  // the int8 path records its own spans (slices | GEMM)
    rc = launch_vnl_add(h, h->dbT, hpsi, ldh, nb, st);
    if (!h->oz_s) prof_span(h, t0, prof_mark(h, st), SLOT_VNL);
  }
  return rc;
}

int apply_impl(qe_hpsi_t h, const void* psi_dev, int64_t ldpsi, void* hpsi_dev, int64_t ldhpsi, int nbands,
               void* cuda_stream, bool local, bool nonlocal) {
  int rc = check_apply_args(h, psi_dev, ldpsi, hpsi_dev, ldhpsi, nbands);
  if (rc || nbands == 0) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const double2* psi = static_cast<const double2*>(psi_dev);
  double2* hpsi = static_cast<double2*>(hpsi_dev);
  for (int b0 = 0; b0 < nbands; b0 += h->max_batch) {
    const int nb = std::min(h->max_batch, nbands - b0);
    rc = apply_chunk(h, psi + (size_t)b0 * ldpsi, ldpsi, hpsi + (size_t)b0 * ldhpsi, ldhpsi, nb, st, local, nonlocal);
    if (rc) return rc;
  }
  return QE_HPSI_OK;
}

}  // namespace

extern "C" int qe_hpsi_apply(qe_hpsi_t h, const void* psi_dev, int64_t ldpsi, void* hpsi_dev, int64_t ldhpsi, int nbands,
                             void* cuda_stream) {
  return apply_impl(h, psi_dev, ldpsi, hpsi_dev, ldhpsi, nbands, cuda_stream, true, true);
}
extern "C" int qe_hpsi_fft_local(qe_hpsi_t h, const void* psi_dev, int64_t ldpsi, void* hpsi_dev, int64_t ldhpsi,
                                 int nbands, void* cuda_stream) {
  return apply_impl(h, psi_dev, ldpsi, hpsi_dev, ldhpsi, nbands, cuda_stream, true, false);
}
extern "C" int qe_hpsi_nonlocal(qe_hpsi_t h, const void* psi_dev, int64_t ldpsi, void* hpsi_dev, int64_t ldhpsi,
                                int nbands, void* cuda_stream) {
  return apply_impl(h, psi_dev, ldpsi, hpsi_dev, ldhpsi, nbands, cuda_stream, false, true);
}

// ---------------------------------------------------------------------------------------------------------
// NEXT-2: overlap operator S = 1 + beta q beta^H, sharing becp with H (include/qe_hpsi.h)
// ---------------------------------------------------------------------------------------------------------
extern "C" int qe_hpsi_set_s(qe_hpsi_t h, const double* q_host) {
  if (!h) return QE_HPSI_ESTATE;
  if (h->nproj == 0) return QE_HPSI_OK;
  if (!q_host) return QE_HPSI_EINVAL;
  CU_TRY(h, cudaSetDevice(h->device));
  if (!h->qpk) {
    const size_t pc = (size_t)h->nproj * h->ldc * sizeof(double2);
    CU_TRY(h, guarded_malloc(h, &h->qpk, sizeof(double) * (size_t)std::max<long long>(h->d_total, 1)));
    CU_TRY(h, guarded_malloc(h, &h->qbecp, pc));
    CU_TRY(h, guarded_malloc(h, &h->qbT, (size_t)h->max_batch * h->ldp * sizeof(double2)));
    CU_TRY(h, cudaMemset(h->qbT, 0, (size_t)h->max_batch * h->ldp * sizeof(double2)));
    h->workspace_bytes += pc + (size_t)h->max_batch * h->ldp * sizeof(double2);
  }
  if (h->sym) {  // does q couple projectors of equal class only?  (needed by the symmetric real forms)
    bool ok = true;
    long long off = 0;
    for (size_t a = 0; a + 1 < h->blk_off.size() && ok; ++a) {
      const int q0 = h->blk_off[a], nh = h->blk_off[a + 1] - q0;
      for (int i = 0; i < nh && ok; ++i)
        for (int j = 0; j < nh; ++j)
          if (q_host[off + (long long)i * nh + j] != 0.0 && h->sym_cls_host[(size_t)q0 + i] != h->sym_cls_host[(size_t)q0 + j]) {
            ok = false;
            break;
          }
      off += (long long)nh * nh;
    }
    if (!ok && h->oz_s) return QE_HPSI_EINVAL;  // see include/qe_hpsi.h: create such a handle with QE_HPSI_NO_GAMMA_SYM
    h->sym_q_ok = ok;
  }
  CU_TRY(h, cudaMemcpy(h->qpk, q_host, sizeof(double) * (size_t)h->d_total, cudaMemcpyHostToDevice));
  return QE_HPSI_OK;
}

extern "C" int qe_hpsi_apply_hs(qe_hpsi_t h, const void* psi_dev, int64_t ldpsi, void* hpsi_dev, int64_t ldhpsi,
                                void* spsi_dev, int64_t ldspsi, int nbands, void* cuda_stream) {
  if (!h) return QE_HPSI_ESTATE;
  if (h->certify) return QE_HPSI_ESTATE;  // the a-posteriori check covers qe_hpsi_apply / qe_hpsi_apply_host only
  if (!spsi_dev) return QE_HPSI_EINVAL;
  int rc = check_apply_args(h, psi_dev, ldpsi, spsi_dev, ldspsi, nbands);
  if (rc) return rc;
  if (hpsi_dev) {
    rc = check_apply_args(h, psi_dev, ldpsi, hpsi_dev, ldhpsi, nbands);
    if (rc) return rc;
    rc = check_apply_args(h, hpsi_dev, ldhpsi, spsi_dev, ldspsi, nbands);  // hpsi and spsi must not overlap either
    if (rc) return rc;
  }
  if (nbands == 0) return QE_HPSI_OK;
  const bool nl = h->nproj > 0 && h->npw > 0;
  if (nl && !h->qpk) return QE_HPSI_ESTATE;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const double2* psi = static_cast<const double2*>(psi_dev);
  double2* hpsi = static_cast<double2*>(hpsi_dev);
  double2* spsi = static_cast<double2*>(spsi_dev);
  for (int b0 = 0; b0 < nbands; b0 += h->max_batch) {
    const int nb = std::min(h->max_batch, nbands - b0);
    const double2* p = psi + (size_t)b0 * ldpsi;
    double2* sp = spsi + (size_t)b0 * ldspsi;
    if (nl) {
      rc = launch_becp(h, p, ldpsi, nb, st);  // becp, dbecp = D becp, dbT
      if (rc) return rc;
      const dim3 rg((nb + 127) / 128, h->nproj);
      k_dmul<<<rg, 128, 0, st>>>(h->becp, h->nproj, h->ldc, nb, h->proj_blk0, h->proj_nh, h->proj_doff, h->qpk, h->qbecp,
                                h->qbT, h->ldp);  // qbecp = q becp, qbT
    }
    if (hpsi) {
      double2* hp = hpsi + (size_t)b0 * ldhpsi;
      rc = launch_local(h, p, ldpsi, hp, ldhpsi, nb, st);
      if (rc) return rc;
      if (nl) {
        rc = launch_vnl_add(h, h->dbT, hp, ldhpsi, nb, st);
        if (rc) return rc;
      }
    }
    if (h->npw > 0)
      CU_TRY(h, cudaMemcpy2DAsync(sp, sizeof(double2) * (size_t)ldspsi, p, sizeof(double2) * (size_t)ldpsi,
                                  sizeof(double2) * (size_t)h->npw, (size_t)nb, cudaMemcpyDeviceToDevice, st));
    if (nl) {
      rc = launch_vnl_add(h, h->qbT, sp, ldspsi, nb, st);  // spsi = psi + beta (q becp)
      if (rc) return rc;
    }
  }
  CU_TRY(h, cudaGetLastError());
  return QE_HPSI_OK;
}

// ---------------------------------------------------------------------------------------------------------
// NEXT-3: reduced matrices out[i][j] = <a_i|b_j> with the split-K DMMA kernel of a6
// ---------------------------------------------------------------------------------------------------------
extern "C" int qe_hpsi_overlap(qe_hpsi_t h, const void* a_dev, int64_t lda, int na, const void* b_dev, int64_t ldb,
                               int nb, void* out_dev, int64_t ldo, void* cuda_stream) {
  if (!h) return QE_HPSI_ESTATE;
  if (na < 0 || nb < 0) return QE_HPSI_EINVAL;
  if (na == 0 || nb == 0) return QE_HPSI_OK;
  if (!a_dev || !b_dev || !out_dev || lda < h->npw || ldb < h->npw || ldo < nb) return QE_HPSI_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const double2* a = static_cast<const double2*>(a_dev);
  const double2* b = static_cast<const double2*>(b_dev);
  double2* out = static_cast<double2*>(out_dev);
  if (h->npw == 0) {
    CU_TRY(h, cudaMemset2DAsync(out, sizeof(double2) * (size_t)ldo, 0, sizeof(double2) * (size_t)nb, (size_t)na, st));
    return QE_HPSI_OK;
  }
  // K slices depend on npw only (plan and workspace made at create), so an element's bits do not depend on how many
  // rows / columns the call has, and the call allocates and synchronises nothing
  constexpr int MA = 512, NB = 128, LDC = 128;
  const int ns = h->ovl_ns, kchunk = h->ovl_kchunk;
  for (int a0 = 0; a0 < na; a0 += MA) {
    const int ma = std::min(MA, na - a0);
    for (int b0 = 0; b0 < nb; b0 += NB) {
      const int nbc = std::min(NB, nb - b0);
      const int mt = (ma + ZgV0::BM - 1) / ZgV0::BM, nt = (nbc + ZgV0::BN - 1) / ZgV0::BN;
      k_becp<ZgV0><<<dim3(mt * nt, ns), ZgV0::NT, ZgV0::SMEM_BECP, st>>>(a + (size_t)a0 * lda, lda, ma, b + (size_t)b0 * ldb,
                                                                         ldb, nbc, h->npw, kchunk, h->ovl_partial, LDC);
      k_ovl_reduce<<<dim3((nbc + 127) / 128, ma), 128, 0, st>>>(h->ovl_partial, ns, ma, LDC, nbc,
                                                                out + (size_t)a0 * ldo + b0, ldo);
    }
  }
  CU_TRY(h, cudaGetLastError());
  return QE_HPSI_OK;
}

// ---------------------------------------------------------------------------------------------------------
// qe_hpsi_overlap_static: the same reduced matrix without a handle and without any allocation (qe_hpsi.h).  The split-K
// partials live in a file-scope device array that every GPU loading the library holds until exit.
// ---------------------------------------------------------------------------------------------------------
namespace {
constexpr int OVS_MAX_N = QE_HPSI_OVERLAP_STATIC_MAX;  // rows and columns of one call
constexpr int OVS_MAX_SPLIT = 32, OVS_LDC = 128;
static __device__ __align__(256) double2 g_ovs_scratch[(size_t)OVS_MAX_SPLIT * OVS_MAX_N * OVS_LDC];  // 8 MiB
// In host code g_ovs_scratch is only a stand-in for the symbol: the device address is asked for once per device, with that
// device current, and that pointer is what the kernels get
double2* g_ovs_ptr[MAX_DEVICES] = {};
std::mutex g_ovs_mutex;
int ovs_setup(double2** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess && (dev < 0 || dev >= MAX_DEVICES)) return QE_HPSI_EINVAL;
  if (e == cudaSuccess) e = set_kernel_attrs();  // per device, allocates nothing
  if (e == cudaSuccess) {
    std::lock_guard<std::mutex> lock(g_ovs_mutex);
    if (!g_ovs_ptr[dev]) {
      double2* ptr = nullptr;
      e = cudaGetSymbolAddress((void**)&ptr, g_ovs_scratch);
      if (e == cudaSuccess) g_ovs_ptr[dev] = ptr;
    }
    if (e == cudaSuccess) *out = g_ovs_ptr[dev];
  }
  if (e != cudaSuccess) {
    g_last_cuda = (int)e;
    return QE_HPSI_ECUDA;
  }
  return QE_HPSI_OK;
}
}  // namespace

extern "C" int qe_hpsi_overlap_static_init(void) {
  double2* ptr = nullptr;
  return ovs_setup(&ptr);
}

extern "C" int qe_hpsi_overlap_static(const void* a_dev, int64_t lda, int na, const void* b_dev, int64_t ldb, int nb, int64_t npw,
                                      void* out_dev, int64_t ldo, void* cuda_stream) {
  if (na < 0 || nb < 0 || npw < 0) return QE_HPSI_EINVAL;
  if (na > OVS_MAX_N || nb > OVS_MAX_N || npw > (int64_t)INT32_MAX - 4096) return QE_HPSI_EINVAL;  // beyond the static scratch
  if (na == 0 || nb == 0) return QE_HPSI_OK;
  if (!a_dev || !b_dev || !out_dev || lda < npw || ldb < npw || ldo < nb) return QE_HPSI_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  double2* out = static_cast<double2*>(out_dev);
  qe_hpsi_handle* h = nullptr;
  if (npw == 0) {
    CU_TRY(h, cudaMemset2DAsync(out, sizeof(double2) * (size_t)ldo, 0, sizeof(double2) * (size_t)nb, (size_t)na, st));
    return QE_HPSI_OK;
  }
  double2* scratch = nullptr;
  const int rc = ovs_setup(&scratch);
  if (rc != QE_HPSI_OK) return rc;
  // the K slices of qe_hpsi_overlap (a function of npw only): the two entry points give the same bits
  const int ns0 = std::max(1, std::min(OVS_MAX_SPLIT, (int)(npw / 2048)));
  int kchunk = (int)((npw + ns0 - 1) / ns0);
  kchunk = std::max(ZgV0::BK, (kchunk + ZgV0::BK - 1) / ZgV0::BK * ZgV0::BK);
  const int ns = std::max(1, (int)((npw + kchunk - 1) / kchunk));
  const int mt = (na + ZgV0::BM - 1) / ZgV0::BM, nt = (nb + ZgV0::BN - 1) / ZgV0::BN;
  // every partial the reduction reads is written by this call's k_becp (slices are never empty), so nothing has to be cleared
  k_becp<ZgV0><<<dim3(mt * nt, ns), ZgV0::NT, ZgV0::SMEM_BECP, st>>>(static_cast<const double2*>(a_dev), lda, na,
                                                                     static_cast<const double2*>(b_dev), ldb, nb, (int)npw, kchunk,
                                                                     scratch, OVS_LDC);
  k_ovl_reduce<<<dim3((nb + 127) / 128, na), 128, 0, st>>>(scratch, ns, na, OVS_LDC, nb, out, ldo);
  CU_TRY(h, cudaGetLastError());
  return QE_HPSI_OK;
}

// NEXT-3, rest of the Davidson step: preconditioner diagonals, preconditioner, basis rotation (a8's kernel)
extern "C" int qe_hpsi_hdiag(qe_hpsi_t h, double vbar, double* hdiag_dev, double* sdiag_dev, void* cuda_stream) {
  if (!h) return QE_HPSI_ESTATE;
  if (!hdiag_dev && !sdiag_dev) return QE_HPSI_EINVAL;
  if (h->npw == 0) return QE_HPSI_OK;
  if (sdiag_dev && h->nproj > 0 && !h->qpk) return QE_HPSI_ESTATE;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const unsigned nblk = (unsigned)((h->npw + 127) / 128);
  if (hdiag_dev)
    k_proj_diag<<<nblk, 128, 0, st>>>(h->beta, h->ldbeta, h->nproj, h->npw, h->proj_doff, h->proj_blk0, h->proj_nh, h->dpk,
                                      h->g2kin, vbar, hdiag_dev);
  if (sdiag_dev)
    k_proj_diag<<<nblk, 128, 0, st>>>(h->beta, h->ldbeta, h->nproj, h->npw, h->proj_doff, h->proj_blk0, h->proj_nh, h->qpk,
                                      nullptr, 0.0, sdiag_dev);
  CU_TRY(h, cudaGetLastError());
  return QE_HPSI_OK;
}

extern "C" int qe_hpsi_precond(qe_hpsi_t h, void* r_dev, int64_t ldr, int nb, const double* e_dev, const double* hdiag_dev,
                               const double* sdiag_dev, void* cuda_stream) {
  if (!h) return QE_HPSI_ESTATE;
  if (nb < 0) return QE_HPSI_EINVAL;
  if (nb == 0 || h->npw == 0) return QE_HPSI_OK;
  if (!r_dev || !e_dev || !hdiag_dev || ldr < h->npw) return QE_HPSI_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  k_precond<<<dim3((h->npw + 255) / 256, nb), 256, 0, st>>>(static_cast<double2*>(r_dev), ldr, nb, h->npw, e_dev, hdiag_dev,
                                                            sdiag_dev);
  CU_TRY(h, cudaGetLastError());
  return QE_HPSI_OK;
}

extern "C" int qe_hpsi_rotate(qe_hpsi_t h, const void* x_dev, int64_t ldx, int nx, const void* coef_dev, int64_t ldcoef,
                              void* y_dev, int64_t ldy, int ny, int accumulate, void* cuda_stream) {
  if (!h) return QE_HPSI_ESTATE;
  if (nx < 0 || ny < 0) return QE_HPSI_EINVAL;
  if (ny == 0 || h->npw == 0) return QE_HPSI_OK;
  if (!y_dev || ldy < h->npw) return QE_HPSI_EINVAL;
  if (nx > 0 && (!x_dev || !coef_dev || ldx < h->npw || ldcoef < nx)) return QE_HPSI_EINVAL;  // before anything is written
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  double2* y = static_cast<double2*>(y_dev);
  if (!accumulate && nx == 0)
    CU_TRY(h, cudaMemset2DAsync(y, sizeof(double2) * (size_t)ldy, 0, sizeof(double2) * (size_t)h->npw, (size_t)ny, st));
  if (nx == 0) return QE_HPSI_OK;
  using Cfg = ZgV0;
  const int mt = (h->npw + Cfg::BM - 1) / Cfg::BM, nt = (ny + Cfg::BN - 1) / Cfg::BN;
  // y[k][g] += sum_j x[j][g] coef[k][j]: the a8 kernel with A = x (M-contiguous) and B = coef (K-contiguous)
  k_vnl_add<Cfg><<<(unsigned)(mt * nt), Cfg::NT, Cfg::SMEM_VNL, st>>>(static_cast<const double2*>(x_dev), ldx, nx, h->npw,
                                                                    static_cast<const double2*>(coef_dev), (int)ldcoef, ny, y,
                                                                    ldy, nullptr, nullptr, nullptr, accumulate ? 0 : 1);
  CU_TRY(h, cudaGetLastError());
  return QE_HPSI_OK;
}

extern "C" int qe_hpsi_residual(qe_hpsi_t h, const void* hx_dev, int64_t ldh, const void* sx_dev, int64_t lds,
                                const double* e_dev, void* r_dev, int64_t ldr, int nb, double* rnorm2_dev, void* cuda_stream) {
  if (!h) return QE_HPSI_ESTATE;
  if (nb < 0) return QE_HPSI_EINVAL;
  if (nb == 0) return QE_HPSI_OK;
  if (!hx_dev || !sx_dev || !e_dev || !r_dev || ldh < h->npw || lds < h->npw || ldr < h->npw) return QE_HPSI_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  k_residual<<<nb, 1024, 0, st>>>(static_cast<const double2*>(hx_dev), ldh, static_cast<const double2*>(sx_dev), lds, e_dev,
                                  static_cast<double2*>(r_dev), ldr, h->npw, rnorm2_dev);
  CU_TRY(h, cudaGetLastError());
  return QE_HPSI_OK;
}

extern "C" int qe_hpsi_scale(qe_hpsi_t h, void* x_dev, int64_t ldx, int nb, const double* fac_dev, void* cuda_stream) {
  if (!h) return QE_HPSI_ESTATE;
  if (nb < 0) return QE_HPSI_EINVAL;
  if (nb == 0 || h->npw == 0) return QE_HPSI_OK;
  if (!x_dev || !fac_dev || ldx < h->npw) return QE_HPSI_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  k_scale_rows<<<dim3((unsigned)((h->npw + 255) / 256), nb), 256, 0, st>>>(static_cast<double2*>(x_dev), ldx, h->npw, fac_dev);
  CU_TRY(h, cudaGetLastError());
  return QE_HPSI_OK;
}

// certified int8 projector path: tolerance and the check results of the last chunk (include/qe_hpsi.h)
extern "C" int qe_hpsi_set_proj_tolerance(qe_hpsi_t h, double tol) {
  if (!h) return QE_HPSI_ESTATE;
  if (!(tol >= 0.0)) return QE_HPSI_EINVAL;
  if (!h->certify) return QE_HPSI_ESTATE;
  h->cert_tol = tol;
  return QE_HPSI_OK;
}
extern "C" int qe_hpsi_get_proj_check(qe_hpsi_t h, double* rel_dev, int32_t* redo_dev, void* cuda_stream) {
  if (!h) return QE_HPSI_ESTATE;
  if (!h->certify) return QE_HPSI_ESTATE;
  if (h->nb_last == 0) return QE_HPSI_OK;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (rel_dev) CU_TRY(h, cudaMemcpyAsync(rel_dev, h->cert_rel, sizeof(double) * (size_t)h->nb_last, cudaMemcpyDeviceToDevice, st));
  if (redo_dev) CU_TRY(h, cudaMemcpyAsync(redo_dev, h->cert_redo, sizeof(int) * (size_t)h->nb_last, cudaMemcpyDeviceToDevice, st));
  return QE_HPSI_OK;
}

// ---------------------------------------------------------------------------------------------------------
// NEXT-4: charge density rho += scale * sum_b occ[b] |psi_b(r)|^2 from steps a1, a2 and the inverse half of a3
// ---------------------------------------------------------------------------------------------------------
extern "C" int qe_hpsi_density(qe_hpsi_t h, const void* psi_dev, int64_t ldpsi, int nbands, const double* occ_dev,
                               double scale, double* rho_dev, void* cuda_stream) {
  if (!h) return QE_HPSI_ESTATE;
  if (nbands < 0) return QE_HPSI_EINVAL;
  if (nbands == 0 || h->npw == 0) return QE_HPSI_OK;
  if (!psi_dev || !occ_dev || !rho_dev || ldpsi < h->npw) return QE_HPSI_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const double2* psi = static_cast<const double2*>(psi_dev);
  const FftGeom& g = h->geom;
  const unsigned zt = (unsigned)((g.S + FFT_C - 1) / FFT_C);
  const unsigned yt = (unsigned)(g.P * g.ntz);
  const unsigned xt = (unsigned)(g.n2 * g.ntz);
  const bool fast = h->f2p[0] != nullptr;
  const Fft2pEntry *ex = h->f2p[0], *ey = h->f2p[1], *ez = h->f2p[2];
  if (fast && !h->rho_attr_done) {
    CU_TRY(h, cudaFuncSetAttribute((const void*)ex->rho, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ex->smem_x));
    h->rho_attr_done = true;
  }
  for (int b0 = 0; b0 < nbands; b0 += h->fft_nb) {
    const int n = std::min(h->fft_nb, nbands - b0);
    const double2* p = psi + (size_t)b0 * ldpsi;
    if (fast) {
      if (h->z_tma_inv)  // the bulk-staged a1 of the hot path
        h->z_tma_inv<<<dim3(zt, n), ez->nthreads, h->smem_zt, st>>>(g, h->g2p, p, ldpsi, h->w1);
      else
        ez->zinv<<<dim3(zt, n), ez->nthreads, ez->smem_zy, st>>>(g, h->g2p, p, ldpsi, h->w1);
      ey->yinv<<<dim3(yt, n), ey->nthreads, ey->smem_zy, st>>>(g, h->g2p, h->w1, h->w2);
      if (h->rho_tma)
        h->rho_tma<<<dim3(xt, 1), ex->nthreads, h->smem_rho, st>>>(g, h->g2p, h->tmap_w2, n, occ_dev + b0, scale, rho_dev);
      else
        ex->rho<<<dim3(xt, 1), ex->nthreads, ex->smem_x, st>>>(g, h->g2p, h->w2, n, occ_dev + b0, scale, rho_dev);
    } else {
      k_scatter_zinv<<<dim3(zt, n), FFT_NT, h->smem_z, st>>>(g, p, ldpsi, h->w1);
      k_yinv<<<dim3(yt, n), FFT_NT, h->smem_y, st>>>(g, h->w1, h->w2);
      k_x_rho<<<dim3(xt, 1), FFT_NT, h->smem_x, st>>>(g, h->w2, n, occ_dev + b0, scale, rho_dev);
    }
  }
  CU_TRY(h, cudaGetLastError());
  return QE_HPSI_OK;
}

// ---------------------------------------------------------------------------------------------------------
// NEXT-1: Gamma-only path (k = 0, real wavefunctions, half sphere; "Gamma-point specific algorithms").
// A Gamma handle = a full-sphere local handle (nproj = 0) that transforms TWO real bands per complex FFT
// (Phi = c1 + i c2 on the full sphere), a half-sphere nonlocal handle (real becp, two real DMMAs per 8x8x4 block)
// and the index maps of G / -G.
// ---------------------------------------------------------------------------------------------------------
struct qe_hpsi_gamma_handle {
  qe_hpsi_handle* loc = nullptr;  // full sphere, local + kinetic only, max_batch = pairs
  qe_hpsi_handle* nl = nullptr;   // npw = ngw: nonlocal part only (may be null: no projectors)
  int ngw = 0, npw = 0, max_batch = 0, pairs = 0;
  long long ldf = 0;              // row stride of phi / hphi
  int *idx_plus = nullptr, *idx_minus = nullptr;  // [ngw] positions of G and -G in the full sphere
  double2 *phi = nullptr, *hphi = nullptr;        // [pairs][ldf]
};

namespace {

// does the Miller triple belong to the half sphere?  (n1 > 0) or (n1 == 0 and n2 > 0) or (n1 == n2 == 0 and n3 >= 0)
inline bool gamma_keep(const int* m) { return m[0] > 0 || (m[0] == 0 && (m[1] > 0 || (m[1] == 0 && m[2] >= 0))); }

// Phi[pair][G] = c1(G) + i c2(G), Phi[pair][-G] = conj(c1(G)) + i conj(c2(G)); band 2*pair+1 missing -> zero
__global__ void k_gamma_merge(const double2* __restrict__ psi, long long ldpsi, int nb, const int* __restrict__ idx_plus,
                              const int* __restrict__ idx_minus, int ngw, double2* __restrict__ phi, long long ldf) {
  const int ig = blockIdx.x * blockDim.x + threadIdx.x;
  const int pr = blockIdx.y;
  if (ig >= ngw) return;
  const int b1 = 2 * pr, b2 = 2 * pr + 1;
  const double2 c1 = psi[(size_t)b1 * ldpsi + ig];
  const double2 c2 = b2 < nb ? psi[(size_t)b2 * ldpsi + ig] : make_double2(0.0, 0.0);
  double2* row = phi + (size_t)pr * ldf;
  const int ip = idx_plus[ig], im = idx_minus[ig];
  if (im != ip) row[im] = make_double2(c1.x + c2.y, c2.x - c1.y);  // conj(c1) + i conj(c2)
  row[ip] = make_double2(c1.x - c2.y, c1.y + c2.x);                // c1 + i c2
}
// h1(G) = (X + conj(Y))/2, h2(G) = (X - conj(Y))/(2i) with X = Phi'(G), Y = Phi'(-G)
__global__ void k_gamma_split(const double2* __restrict__ hphi, long long ldf, const int* __restrict__ idx_plus,
                              const int* __restrict__ idx_minus, int ngw, double2* __restrict__ hpsi, long long ldh, int nb) {
  const int ig = blockIdx.x * blockDim.x + threadIdx.x;
  const int pr = blockIdx.y;
  if (ig >= ngw) return;
  const double2* row = hphi + (size_t)pr * ldf;
  const double2 x = row[idx_plus[ig]], y = row[idx_minus[ig]];
  const int b1 = 2 * pr, b2 = 2 * pr + 1;
  hpsi[(size_t)b1 * ldh + ig] = make_double2(0.5 * (x.x + y.x), 0.5 * (x.y - y.y));
  if (b2 < nb) hpsi[(size_t)b2 * ldh + ig] = make_double2(0.5 * (x.y + y.y), 0.5 * (y.x - x.x));
}

}  // namespace

extern "C" int qe_hpsi_gamma_gsphere(const double at[9], double ecutwfc, const int nr[3], int64_t* ngw,
                                     int32_t* miller_host) {
  if (!ngw) return QE_HPSI_EINVAL;
  const double xk[3] = {0.0, 0.0, 0.0};
  int64_t npw = 0;
  int rc = qe_hpsi_gsphere(at, xk, ecutwfc, nr, &npw, nullptr);
  if (rc) return rc;
  std::vector<int32_t> mil;
  try {
    mil.resize((size_t)std::max<int64_t>(npw, 1) * 3);
  } catch (const std::bad_alloc&) {
    return QE_HPSI_ENOMEM;
  }
  rc = qe_hpsi_gsphere(at, xk, ecutwfc, nr, &npw, mil.data());
  if (rc) return rc;
  int64_t n = 0;
  for (int64_t i = 0; i < npw; ++i)
    if (gamma_keep(&mil[3 * i])) {
      if (miller_host) {
        miller_host[3 * n] = mil[3 * i];
        miller_host[3 * n + 1] = mil[3 * i + 1];
        miller_host[3 * n + 2] = mil[3 * i + 2];
      }
      ++n;
    }
  *ngw = n;
  return QE_HPSI_OK;
}

extern "C" int qe_hpsi_gamma_destroy(qe_hpsi_gamma_t g) {
  if (!g) return QE_HPSI_OK;
  qe_hpsi_destroy(g->loc);
  qe_hpsi_destroy(g->nl);
  cudaFree(g->idx_plus);
  cudaFree(g->idx_minus);
  cudaFree(g->phi);
  cudaFree(g->hphi);
  delete g;
  return QE_HPSI_OK;
}

namespace {
int gamma_create_impl(qe_hpsi_gamma_t* out, qe_hpsi_gamma_handle** live, const double at[9], double ecutwfc, const int nr[3],
                      const double* vr_dev, int nproj, const void* beta_dev, int64_t ldbeta, int nblocks,
                      const int32_t* blk_off_host, const double* d_host, int max_batch, unsigned flags, void* cuda_stream) {
  if (!vr_dev || nproj < 0 || max_batch < 1) return QE_HPSI_EINVAL;
  {
    const int frc = validate_flags(flags, true);
    if (frc) return frc;
  }
  long long d_total = 0;
  if (nproj > 0) {
    if (!beta_dev || !blk_off_host || !d_host || nblocks < 1) return QE_HPSI_EINVAL;
    if (blk_off_host[0] != 0 || blk_off_host[nblocks] != nproj) return QE_HPSI_EINVAL;
    for (int a = 0; a < nblocks; ++a) {
      const long long nh = (long long)blk_off_host[a + 1] - blk_off_host[a];
      if (nh <= 0) return QE_HPSI_EINVAL;
      d_total += nh * nh;
    }
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  qe_hpsi_gamma_handle* g = new (std::nothrow) qe_hpsi_gamma_handle();
  if (!g) return QE_HPSI_ENOMEM;
  *live = g;  // on any failure below the caller (qe_hpsi_gamma_create) destroys it
  g->max_batch = max_batch;
  g->pairs = (max_batch + 1) / 2;
  const double xk[3] = {0.0, 0.0, 0.0};
  int rc = qe_hpsi_create(&g->loc, at, ecutwfc, xk, nr, vr_dev, 0, nullptr, 0, 0, nullptr, nullptr, g->pairs,
                          flags & QE_HPSI_GENERIC_FFT, cuda_stream);
  if (rc) return rc;
  g->npw = g->loc->npw;
#define CG_TRY(expr)                                                           \
  do {                                                                         \
    cudaError_t e__ = (expr);                                                  \
    if (e__ != cudaSuccess) {                                                  \
      g_last_cuda = (int)e__;                                                  \
      (void)cudaGetLastError();                                                \
      return e__ == cudaErrorMemoryAllocation ? QE_HPSI_ENOMEM : QE_HPSI_ECUDA; \
    }                                                                          \
  } while (0)
  // half-sphere maps from the device-built full sphere (host side: integer work, once per handle)
  std::vector<int> mil((size_t)std::max(g->npw, 1) * 3), fidx((size_t)std::max(g->npw, 1));
  if (g->npw) {
    CG_TRY(cudaMemcpy(mil.data(), g->loc->miller, sizeof(int) * 3 * (size_t)g->npw, cudaMemcpyDeviceToHost));
    CG_TRY(cudaMemcpy(fidx.data(), g->loc->fftidx, sizeof(int) * (size_t)g->npw, cudaMemcpyDeviceToHost));
  }
  std::vector<int> ip, im;
  for (int i = 0; i < g->npw; ++i) {
    if (!gamma_keep(&mil[3 * (size_t)i])) continue;
    // position of -G: wrapped linear index of the negated triple, binary search in the ascending fft_index
    long long lin = 0;
    for (int j = 0; j < 3; ++j) {
      const int n = -mil[3 * (size_t)i + j];
      lin = lin * nr[j] + ((n % nr[j]) + nr[j]) % nr[j];
    }
    auto it = std::lower_bound(fidx.begin(), fidx.begin() + g->npw, (int)lin);
    if (it == fidx.begin() + g->npw || *it != (int)lin) return QE_HPSI_ESTATE;  // cannot happen for a k = 0 sphere
    ip.push_back(i);
    im.push_back((int)(it - fidx.begin()));
  }
  g->ngw = (int)ip.size();
  if (nproj > 0 && ldbeta < g->ngw) return QE_HPSI_EINVAL;
  CG_TRY(upload(&g->idx_plus, ip, st));
  CG_TRY(upload(&g->idx_minus, im, st));
  g->ldf = ((long long)g->npw + 7) / 8 * 8;
  const size_t fb = sizeof(double2) * (size_t)g->pairs * (size_t)std::max<long long>(g->ldf, 1);
  CG_TRY(cudaMalloc(&g->phi, fb));
  CG_TRY(cudaMalloc(&g->hphi, fb));
  CG_TRY(cudaMemsetAsync(g->phi, 0, fb, st));
  CG_TRY(cudaMemsetAsync(g->hphi, 0, fb, st));
  if (nproj > 0 && g->ngw > 0) {
    g->nl = new (std::nothrow) qe_hpsi_handle();
    if (!g->nl) return QE_HPSI_ENOMEM;
    g->nl->device = g->loc->device;
    g->nl->num_sms = g->loc->num_sms;
    g->nl->npw = g->ngw;
    g->nl->nproj = nproj;
    g->nl->max_batch = max_batch;
    g->nl->gamma = true;
    CG_TRY(set_kernel_attrs());
    CG_TRY(setup_nonlocal(g->nl, nproj, beta_dev, ldbeta, nblocks, blk_off_host, d_host, d_total, max_batch, flags, st));
    if (flags & QE_HPSI_PROJ_INT8) CG_TRY(setup_ozaki(g->nl, max_batch, flags, st));
  }
  CG_TRY(cudaStreamSynchronize(st));
#undef CG_TRY
  *live = nullptr;
  *out = g;
  return QE_HPSI_OK;
}
}  // namespace

extern "C" int qe_hpsi_gamma_create(qe_hpsi_gamma_t* out, const double at[9], double ecutwfc, const int nr[3],
                                    const double* vr_dev, int nproj, const void* beta_dev, int64_t ldbeta, int nblocks,
                                    const int32_t* blk_off_host, const double* d_host, int max_batch, unsigned flags,
                                    void* cuda_stream) {
  if (!out) return QE_HPSI_EINVAL;
  *out = nullptr;
  qe_hpsi_gamma_handle* live = nullptr;
  int rc;
  try {
    rc = gamma_create_impl(out, &live, at, ecutwfc, nr, vr_dev, nproj, beta_dev, ldbeta, nblocks, blk_off_host, d_host, max_batch,
                           flags, cuda_stream);
  } catch (const std::bad_alloc&) {
    rc = QE_HPSI_ENOMEM;
  } catch (...) {
    rc = QE_HPSI_ESTATE;
  }
  if (rc != QE_HPSI_OK) {
    if (live) qe_hpsi_gamma_destroy(live);
    *out = nullptr;
  }
  return rc;
}


extern "C" int64_t qe_hpsi_gamma_ngw(qe_hpsi_gamma_t g) { return g ? g->ngw : (int64_t)QE_HPSI_ESTATE; }

extern "C" int qe_hpsi_gamma_apply(qe_hpsi_gamma_t g, const void* psi_dev, int64_t ldpsi, void* hpsi_dev, int64_t ldhpsi,
                                   int nbands, void* cuda_stream) {
  if (!g) return QE_HPSI_ESTATE;
  if (nbands < 0) return QE_HPSI_EINVAL;
  if (nbands == 0 || g->ngw == 0) return QE_HPSI_OK;
  if (!psi_dev || !hpsi_dev || ldpsi < g->ngw || ldhpsi < g->ngw) return QE_HPSI_EINVAL;
  {
    const char* a0 = static_cast<const char*>(psi_dev);
    const char* a1 = a0 + ((size_t)(nbands - 1) * ldpsi + g->ngw) * sizeof(double2);
    const char* b0 = static_cast<const char*>(hpsi_dev);
    const char* b1 = b0 + ((size_t)(nbands - 1) * ldhpsi + g->ngw) * sizeof(double2);
    if (a0 < b1 && b0 < a1) return QE_HPSI_EINVAL;
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const double2* psi = static_cast<const double2*>(psi_dev);
  double2* hpsi = static_cast<double2*>(hpsi_dev);
  qe_hpsi_handle* h = g->loc;
  for (int b0 = 0; b0 < nbands; b0 += g->max_batch) {
    const int nb = std::min(g->max_batch, nbands - b0);
    const int pairs = (nb + 1) / 2;
    const double2* p = psi + (size_t)b0 * ldpsi;
    double2* o = hpsi + (size_t)b0 * ldhpsi;
    if (g->nl) {
      const int rc = launch_becp(g->nl, p, ldpsi, nb, st);  // real becp over the half sphere, dbecp = D becp
      if (rc) return rc;
    }
    const dim3 grid((g->ngw + 255) / 256, pairs);
    k_gamma_merge<<<grid, 256, 0, st>>>(p, ldpsi, nb, g->idx_plus, g->idx_minus, g->ngw, g->phi, g->ldf);
    int rc = launch_local(h, g->phi, g->ldf, g->hphi, g->ldf, pairs, st);  // a1-a5 on pairs of bands, kinetic included
    if (rc) return rc;
    k_gamma_split<<<grid, 256, 0, st>>>(g->hphi, g->ldf, g->idx_plus, g->idx_minus, g->ngw, o, ldhpsi, nb);
    if (g->nl) {
      rc = launch_vnl_add(g->nl, g->nl->dbT, o, ldhpsi, nb, st);
      if (rc) return rc;
    }
  }
  CU_TRY(h, cudaGetLastError());
  return QE_HPSI_OK;
}

// ---------------------------------------------------------------------------------------------------------
// end-to-end variant with host buffers: H2D copy of chunk i+1 and D2H copy of chunk i-1 overlap the compute
// of chunk i (three internal streams, two staging buffers each for psi and hpsi)
// ---------------------------------------------------------------------------------------------------------
extern "C" int qe_hpsi_apply_host(qe_hpsi_t h, const void* psi_host, int64_t ldpsi, void* hpsi_host, int64_t ldhpsi,
                                  int nbands) {
  if (!h) return QE_HPSI_ESTATE;
  if (nbands < 0) return QE_HPSI_EINVAL;
  if (nbands == 0) return QE_HPSI_OK;
  if (!psi_host || !hpsi_host || ldpsi < h->npw || ldhpsi < h->npw) return QE_HPSI_EINVAL;
  if (!h->st_comp) {
    h->ldint = ((long long)h->npw + 7) / 8 * 8;
    const size_t bytes = std::max<size_t>(16, (size_t)h->max_batch * h->ldint * sizeof(double2));
    for (int i = 0; i < 2; ++i) {
      CU_TRY(h, guarded_malloc(h, &h->hbuf_psi[i], bytes));
      CU_TRY(h, guarded_malloc(h, &h->hbuf_h[i], bytes));
      CU_TRY(h, cudaEventCreateWithFlags(&h->ev_in[i], cudaEventDisableTiming));
      CU_TRY(h, cudaEventCreateWithFlags(&h->ev_comp[i], cudaEventDisableTiming));
      CU_TRY(h, cudaEventCreateWithFlags(&h->ev_out[i], cudaEventDisableTiming));
    }
    CU_TRY(h, cudaStreamCreateWithFlags(&h->st_in, cudaStreamNonBlocking));
    CU_TRY(h, cudaStreamCreateWithFlags(&h->st_out, cudaStreamNonBlocking));
    CU_TRY(h, cudaStreamCreateWithFlags(&h->st_comp, cudaStreamNonBlocking));
  }
  const double2* psi = static_cast<const double2*>(psi_host);
  double2* hpsi = static_cast<double2*>(hpsi_host);
  const size_t width = sizeof(double2) * (size_t)h->npw;
  // chunks of max_batch bands, except that the first and the last chunk are halved (down to a 64-band ZGEMM tile) when
  // there are several: the H2D copy of the first chunk and the D2H copy of the last one are the only transfers that do
  // not overlap compute
  // (32 bands where the projector kernels have a 64-column tile for them: the Gamma-symmetric TMA kernels; else 64)
  const int small = (h->sym_tma && h->sym_tail) ? 32 : 64;
  const int half = (h->max_batch >= 128 && nbands > h->max_batch) ? small : h->max_batch;
  int ci = 0;
  for (int b0 = 0, nb = 0; b0 < nbands; b0 += nb, ++ci) {
    const int left = nbands - b0;
    nb = std::min(h->max_batch, left);
    if (ci == 0) nb = std::min(half, left);
    else if (left > half && left < h->max_batch + half) nb = std::min(h->max_batch, left - half);  // leave exactly `half` for the last chunk
    const int u = ci & 1;
    if (ci >= 2) CU_TRY(h, cudaStreamWaitEvent(h->st_in, h->ev_comp[u], 0));  // compute of chunk ci-2 read psi buf u
    if (width)
      CU_TRY(h, cudaMemcpy2DAsync(h->hbuf_psi[u], sizeof(double2) * h->ldint, psi + (size_t)b0 * ldpsi,
                                  sizeof(double2) * (size_t)ldpsi, width, (size_t)nb, cudaMemcpyHostToDevice, h->st_in));
    CU_TRY(h, cudaEventRecord(h->ev_in[u], h->st_in));
    CU_TRY(h, cudaStreamWaitEvent(h->st_comp, h->ev_in[u], 0));
    if (ci >= 2) CU_TRY(h, cudaStreamWaitEvent(h->st_comp, h->ev_out[u], 0));  // D2H of chunk ci-2 read hpsi buf u
    int rc = apply_chunk(h, h->hbuf_psi[u], h->ldint, h->hbuf_h[u], h->ldint, nb, h->st_comp, true, true);
    if (rc) return rc;
    CU_TRY(h, cudaEventRecord(h->ev_comp[u], h->st_comp));
    CU_TRY(h, cudaStreamWaitEvent(h->st_out, h->ev_comp[u], 0));
    if (width)
      CU_TRY(h, cudaMemcpy2DAsync(hpsi + (size_t)b0 * ldhpsi, sizeof(double2) * (size_t)ldhpsi, h->hbuf_h[u],
                                  sizeof(double2) * h->ldint, width, (size_t)nb, cudaMemcpyDeviceToHost, h->st_out));
    CU_TRY(h, cudaEventRecord(h->ev_out[u], h->st_out));
  }
  CU_TRY(h, cudaStreamSynchronize(h->st_out));
  CU_TRY(h, cudaStreamSynchronize(h->st_comp));
  return QE_HPSI_OK;
}

// ---------------------------------------------------------------------------------------------------------
// accessors
// ---------------------------------------------------------------------------------------------------------
extern "C" int64_t qe_hpsi_npw(qe_hpsi_t h) { return h ? h->npw : (int64_t)QE_HPSI_ESTATE; }
extern "C" int64_t qe_hpsi_nsticks(qe_hpsi_t h) { return h ? h->S : (int64_t)QE_HPSI_ESTATE; }
extern "C" int64_t qe_hpsi_nplanes(qe_hpsi_t h) { return h ? h->P : (int64_t)QE_HPSI_ESTATE; }

extern "C" int qe_hpsi_get_maps(qe_hpsi_t h, int32_t* miller_dev, int32_t* fftidx_dev, double* g2kin_dev,
                                void* cuda_stream) {
  if (!h) return QE_HPSI_ESTATE;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const size_t n = (size_t)h->npw;
  if (n == 0) return QE_HPSI_OK;
  if (miller_dev) CU_TRY(h, cudaMemcpyAsync(miller_dev, h->miller, sizeof(int) * 3 * n, cudaMemcpyDeviceToDevice, st));
  if (fftidx_dev) CU_TRY(h, cudaMemcpyAsync(fftidx_dev, h->fftidx, sizeof(int) * n, cudaMemcpyDeviceToDevice, st));
  if (g2kin_dev) CU_TRY(h, cudaMemcpyAsync(g2kin_dev, h->g2kin, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
  return QE_HPSI_OK;
}

extern "C" int qe_hpsi_get_becp(qe_hpsi_t h, void* becp_dev, void* dbecp_dev, void* cuda_stream) {
  if (!h) return QE_HPSI_ESTATE;
  if (h->nproj == 0 || h->nb_last == 0) return QE_HPSI_OK;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const size_t w = sizeof(double2) * (size_t)h->nb_last, sp = sizeof(double2) * (size_t)h->ldc;
  if (becp_dev) CU_TRY(h, cudaMemcpy2DAsync(becp_dev, w, h->becp, sp, w, (size_t)h->nproj, cudaMemcpyDeviceToDevice, st));
  if (dbecp_dev) CU_TRY(h, cudaMemcpy2DAsync(dbecp_dev, w, h->dbecp, sp, w, (size_t)h->nproj, cudaMemcpyDeviceToDevice, st));
  return QE_HPSI_OK;
}

extern "C" int64_t qe_hpsi_launch_count(qe_hpsi_t h, int nbands) {
  if (!h) return QE_HPSI_ESTATE;
  if (nbands <= 0 || h->npw == 0) return 0;
  int64_t total = 0;
  for (int b0 = 0; b0 < nbands; b0 += h->max_batch) {
    const int nb = std::min(h->max_batch, nbands - b0);
    total += 5 * (int64_t)((nb + h->fft_nb - 1) / h->fft_nb);
    if (h->nproj > 0) total += h->oz_s ? 7 + (h->oz_3m ? 2 : 0) + (h->oz_3m8 ? 1 : (int)((h->oz_k2 / oz::KB + h->oz_kchunk2 - 1) / h->oz_kchunk2)) : (h->sym ? 6 + (h->sym_tma && sym_a8_main_tiles(h, nb) > 0 && sym_a8_main_tiles(h, nb) < h->sym_nlive ? 1 : 0) : 4);
    if (h->nproj > 0 && h->oz_s && h->sym) total += 2;  // merge and coefficient kernels of the symmetric real forms
    if (h->certify) total += 8;  // probe, decide, gather, the four FP64 kernels (empty grids when nothing failed), commit
  }
  return total;
}

extern "C" int qe_hpsi_info(qe_hpsi_t h, int64_t info[16]) {
  if (!h) return QE_HPSI_ESTATE;
  if (!info) return QE_HPSI_EINVAL;
  for (int i = 0; i < 16; ++i) info[i] = 0;
  info[0] = h->npw;
  info[1] = h->S;
  info[2] = h->P;
  info[3] = h->fft_nb;
  info[4] = h->nsplit;
  info[5] = (int64_t)h->workspace_bytes;
  info[6] = h->geom.ax1.npass;
  info[7] = h->geom.ax2.npass;
  info[8] = h->geom.ax3.npass;
  info[9] = h->kchunk;
  info[10] = h->x_split;
  info[11] = h->num_sms;
  info[12] = (h->f2p[0] ? 1 : 0) | (h->sym ? 2 : 0) | (h->x_half ? 4 : 0);
  info[13] = h->oz_s;
  info[14] = h->oz_nsplit;
  info[15] = (h->oz_3m ? (h->oz_3m8 ? 2 : 1) : 0) + (h->certify ? 4 : 0);
  return QE_HPSI_OK;
}

extern "C" int qe_hpsi_profile(qe_hpsi_t h, int mode) {
  if (!h) return QE_HPSI_ESTATE;
  if (mode < 0 || mode > 2) return QE_HPSI_EINVAL;
  prof_drain(h);
  for (int i = 0; i < 16; ++i) {
    h->prof_ms[i] = 0.0;
    h->prof_cnt[i] = 0;
  }
  h->prof_mode = mode;
  return QE_HPSI_OK;
}
extern "C" int qe_hpsi_profile_read(qe_hpsi_t h, double ms[16], int64_t count[16]) {
  if (!h) return QE_HPSI_ESTATE;
  if (!ms || !count) return QE_HPSI_EINVAL;
  prof_drain(h);
  for (int i = 0; i < 16; ++i) {
    ms[i] = h->prof_ms[i];
    count[i] = h->prof_cnt[i];
  }
  return QE_HPSI_OK;
}

// ---------------------------------------------------------------------------------------------------------
// FP64 peak probe (measurement helper for the roofline denominator; not on the hot path)
// ---------------------------------------------------------------------------------------------------------
namespace {
__global__ void __launch_bounds__(256) k_probe_dmma(double* out, int iters, double a, double b) {
  double c[32][2];
#pragma unroll
  for (int i = 0; i < 32; ++i) {
    c[i][0] = (double)i;
    c[i][1] = (double)threadIdx.x;
  }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 32; ++i) dmma884(c[i][0], c[i][1], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 32; ++i) s += c[i][0] + c[i][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void __launch_bounds__(1024) k_probe_dfma(double* out, int iters, double a, double b) {
  double x[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = threadIdx.x * 1e-3 + i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = fma(x[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += x[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
}  // namespace

extern "C" int qe_hpsi_probe_fp64(double millis, double* dmma_tflops, double* dfma_tflops) {
  qe_hpsi_handle* h = nullptr;
  int dev = 0, nsm = 0;
  CU_TRY(h, cudaGetDevice(&dev));
  CU_TRY(h, cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
  double* out = nullptr;
  CU_TRY(h, cudaMalloc(&out, sizeof(double) * (size_t)nsm * 1024));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  int rc = QE_HPSI_OK;
  for (int which = 0; which < 2 && rc == QE_HPSI_OK; ++which) {
    const int iters = which == 0 ? 4000 : 16000;
    const double flop_per_launch =
        which == 0 ? 2.0 * 256 * 32 * iters * 8.0 * nsm : 2.0 * 16 * iters * 1024.0 * nsm;
    double best = 0.0, spent = 0.0;
    for (int rep = 0; rep < 1000 && (rep < 3 || spent < millis); ++rep) {
      cudaEventRecord(e0);
      if (which == 0)
        k_probe_dmma<<<nsm, 256>>>(out, iters, 1.0000001, 1e-9);
      else
        k_probe_dfma<<<nsm, 1024>>>(out, iters, 1.0000001, 1e-9);
      cudaEventRecord(e1);
      cudaError_t e = cudaEventSynchronize(e1);
      if (e != cudaSuccess) {
        g_last_cuda = (int)e;
        rc = QE_HPSI_ECUDA;
        break;
      }
      float ms = 0.f;
      cudaEventElapsedTime(&ms, e0, e1);
      spent += ms;
      if (rep >= 1) best = std::max(best, flop_per_launch / (ms * 1e-3) * 1e-12);
    }
    if (which == 0 && dmma_tflops) *dmma_tflops = best;
    if (which == 1 && dfma_tflops) *dfma_tflops = best;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(out);
  return rc;
}
