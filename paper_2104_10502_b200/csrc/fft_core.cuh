// fft_core.cuh -- FP64 complex radix-2/3/5 pencil FFT building blocks (shared-memory Stockham passes with
// register-resident radix-R butterflies, R <= 16).  Part of libqe_hpsi (steps a1-a5 of DESIGN.md; the paper only
// says the local term goes through 1-D and 2-D FFTs, PAPER.md:L215 -- the decomposition here is this build's).
//
// Tile layout.  A CTA transforms C pencils ("columns", C = 8) of length N held in shared memory as
// tile[n][c] complex128 with the column index XOR-swizzled by the row:  phys(n,c) = n*C + (c ^ (n & 7)).
//   * butterflies: lanes run over c at fixed n  -> 8 consecutive lanes cover one 128-byte row: conflict free;
//   * transposing loads/stores (z passes; lanes run over n at fixed c) -> 8 consecutive n give 8 distinct
//     16-byte bank groups: conflict free as well.
// Passes ping-pong between two such tiles (Stockham autosort, natural order in and out).
#pragma once
#include <cuda_runtime.h>
#include <type_traits>
#include <utility>

namespace qehpsi {

constexpr int FFT_C = 8;          // pencils per tile
constexpr int FFT_MAX_PASS = 12;  // N <= 720: at most 9 passes even with radices 2..5 only (512 = 2^9 -> 4,4,4,4,2)

struct FftAxis {
  int n;                      // length
  int npass;                  // number of passes
  int radix[FFT_MAX_PASS];    // radix of each pass (product = n)
  const double2* tw;          // device table tw[k] = exp(+2 pi i k / n), k = 0..n-1
};

__device__ __forceinline__ int fft_phys(int n, int c) { return n * FFT_C + (c ^ (n & 7)); }

// ---------------------------------------------------------------------------------------------------------
// compile-time twiddles exp(2 pi i m / R): exact quadrant reduction with integers, then Taylor series on
// |delta| <= pi/4 (error ~1e-16).  Evaluated by the front end (constexpr), so butterflies carry literals.
// ---------------------------------------------------------------------------------------------------------
constexpr double kPi = 3.141592653589793238462643383279502884;

__host__ __device__ constexpr double ct_sin(double x) {
  double x2 = x * x, term = x, sum = x;
  for (int i = 1; i <= 12; ++i) {
    term *= -x2 / double((2 * i) * (2 * i + 1));
    sum += term;
  }
  return sum;
}
__host__ __device__ constexpr double ct_cos(double x) {
  double x2 = x * x, term = 1.0, sum = 1.0;
  for (int i = 1; i <= 12; ++i) {
    term *= -x2 / double((2 * i - 1) * (2 * i));
    sum += term;
  }
  return sum;
}
struct cpx_ct {
  double re, im;
};
// exp(2 pi i m / R), any integer m
__host__ __device__ constexpr cpx_ct ct_twiddle(int m, int R) {
  m %= R;
  if (m < 0) m += R;
  int q = (8 * m + R) / (2 * R);  // nearest quarter turn
  int num = 4 * m - q * R;        // delta = pi * num / (2 R), |delta| <= pi/4
  double d = kPi * double(num) / double(2 * R);
  double c = (num == 0) ? 1.0 : ct_cos(d);
  double s = (num == 0) ? 0.0 : ct_sin(d);
  q &= 3;
  if (q == 0) return {c, s};
  if (q == 1) return {-s, c};
  if (q == 2) return {-c, -s};
  return {s, -c};
}

// ---------------------------------------------------------------------------------------------------------
// small complex helpers
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
// a * conj(b)
__device__ __forceinline__ double2 cmulc(double2 a, double2 b) {
  return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
// multiply by DIR*i
template <int DIR>
__device__ __forceinline__ double2 cmul_i(double2 a) {
  return DIR > 0 ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x);
}

// v * exp(DIR * 2 pi i M / R) with compile-time M, R; trivial factors cost nothing
template <int M_, int R, int DIR>
__device__ __forceinline__ double2 cmul_tw(double2 v) {
  constexpr int M = ((DIR > 0 ? M_ : -M_) % R + R) % R;
  if constexpr (M == 0) {
    return v;
  } else if constexpr (4 * M == R) {
    return make_double2(-v.y, v.x);
  } else if constexpr (2 * M == R) {
    return make_double2(-v.x, -v.y);
  } else if constexpr (4 * M == 3 * R) {
    return make_double2(v.y, -v.x);
  } else if constexpr (8 * M == R || 8 * M == 3 * R || 8 * M == 5 * R || 8 * M == 7 * R) {
    constexpr double h = 0.70710678118654752440;
    constexpr cpx_ct w = ct_twiddle(M, R);
    constexpr double sr = w.re > 0 ? h : -h, si = w.im > 0 ? h : -h;
    return make_double2(sr * v.x - si * v.y, si * v.x + sr * v.y);
  } else {
    constexpr cpx_ct w = ct_twiddle(M, R);
    return make_double2(v.x * w.re - v.y * w.im, v.x * w.im + v.y * w.re);
  }
}

template <int I>
using ic = std::integral_constant<int, I>;
template <typename F, int... Is>
__device__ __forceinline__ void static_for_impl(F&& f, std::integer_sequence<int, Is...>) {
  (f(ic<Is>{}), ...);
}
template <int N, typename F>
__device__ __forceinline__ void static_for(F&& f) {
  static_for_impl(static_cast<F&&>(f), std::make_integer_sequence<int, N>{});
}

// ---------------------------------------------------------------------------------------------------------
// register DFTs, natural order in and out:  X[k] = sum_n x[n] exp(DIR 2 pi i n k / R)
// ---------------------------------------------------------------------------------------------------------
template <int R, int DIR>
struct Dft;

template <int DIR>
struct Dft<1, DIR> {
  __device__ __forceinline__ static void run(double2 (&)[1]) {}
};
template <int DIR>
struct Dft<2, DIR> {
  __device__ __forceinline__ static void run(double2 (&v)[2]) {
    double2 a = v[0], b = v[1];
    v[0] = cadd(a, b);
    v[1] = csub(a, b);
  }
};
template <int DIR>
struct Dft<3, DIR> {
  __device__ __forceinline__ static void run(double2 (&v)[3]) {
    constexpr double s = 0.86602540378443864676;  // sin(2 pi/3)
    double2 t = cadd(v[1], v[2]);
    double2 d = csub(v[1], v[2]);
    double2 m = make_double2(v[0].x - 0.5 * t.x, v[0].y - 0.5 * t.y);
    double2 r = cmul_i<DIR>(make_double2(s * d.x, s * d.y));
    v[0] = cadd(v[0], t);
    v[1] = cadd(m, r);
    v[2] = csub(m, r);
  }
};
template <int DIR>
struct Dft<4, DIR> {
  __device__ __forceinline__ static void run(double2 (&v)[4]) {
    double2 a = cadd(v[0], v[2]), b = csub(v[0], v[2]);
    double2 c = cadd(v[1], v[3]), d = cmul_i<DIR>(csub(v[1], v[3]));
    v[0] = cadd(a, c);
    v[1] = cadd(b, d);
    v[2] = csub(a, c);
    v[3] = csub(b, d);
  }
};
template <int DIR>
struct Dft<5, DIR> {
  __device__ __forceinline__ static void run(double2 (&v)[5]) {
    constexpr double c1 = 0.30901699437494742410;   // cos(2 pi/5)
    constexpr double c2 = -0.80901699437494742410;  // cos(4 pi/5)
    constexpr double s1 = 0.95105651629515357212;   // sin(2 pi/5)
    constexpr double s2 = 0.58778525229247312917;   // sin(4 pi/5)
    double2 a1 = cadd(v[1], v[4]), b1 = csub(v[1], v[4]);
    double2 a2 = cadd(v[2], v[3]), b2 = csub(v[2], v[3]);
    double2 m1 = make_double2(v[0].x + c1 * a1.x + c2 * a2.x, v[0].y + c1 * a1.y + c2 * a2.y);
    double2 m2 = make_double2(v[0].x + c2 * a1.x + c1 * a2.x, v[0].y + c2 * a1.y + c1 * a2.y);
    double2 r1 = cmul_i<DIR>(make_double2(s1 * b1.x + s2 * b2.x, s1 * b1.y + s2 * b2.y));
    double2 r2 = cmul_i<DIR>(make_double2(s2 * b1.x - s1 * b2.x, s2 * b1.y - s1 * b2.y));
    v[0] = make_double2(v[0].x + a1.x + a2.x, v[0].y + a1.y + a2.y);
    v[1] = cadd(m1, r1);
    v[4] = csub(m1, r1);
    v[2] = cadd(m2, r2);
    v[3] = csub(m2, r2);
  }
};

// composite R = P*Q (P a primitive radix): x[Q a + b] -> P-point DFTs over a, twiddle W_R^{b c}, Q-point DFTs
// over b, X[c + P d].
template <int R>
constexpr int first_factor() {
  return (R % 4 == 0) ? 4 : (R % 2 == 0) ? 2 : (R % 3 == 0) ? 3 : (R % 5 == 0) ? 5 : R;
}
template <int R, int DIR>
struct Dft {
  static constexpr int P = first_factor<R>();
  static constexpr int Q = R / P;
  static_assert(P != R, "unsupported radix");
  __device__ __forceinline__ static void run(double2 (&v)[R]) {
    double2 y[Q][P];
    static_for<Q>([&](auto b_) {
      constexpr int b = decltype(b_)::value;
      double2 t[P];
      static_for<P>([&](auto a_) {
        constexpr int a = decltype(a_)::value;
        t[a] = v[Q * a + b];
      });
      Dft<P, DIR>::run(t);
      static_for<P>([&](auto c_) {
        constexpr int c = decltype(c_)::value;
        y[b][c] = cmul_tw<b * c, R, DIR>(t[c]);
      });
    });
    static_for<P>([&](auto c_) {
      constexpr int c = decltype(c_)::value;
      double2 u[Q];
      static_for<Q>([&](auto b_) {
        constexpr int b = decltype(b_)::value;
        u[b] = y[b][c];
      });
      Dft<Q, DIR>::run(u);
      static_for<Q>([&](auto d_) {
        constexpr int d = decltype(d_)::value;
        v[c + P * d] = u[d];
      });
    });
  }
};

// ---------------------------------------------------------------------------------------------------------
// one Stockham pass over a [N][FFT_C] tile:  out = pass_R(in),  Ns = product of the radices already applied
// ---------------------------------------------------------------------------------------------------------
template <int R, int DIR>
__device__ __forceinline__ void fft_pass(const double2* __restrict__ in, double2* __restrict__ out, int N, int Ns,
                                         const double2* __restrict__ tw, int tid, int nthreads) {
  const int M = N / R;
  const int tasks = M * FFT_C;
  const int twstep = M / Ns;
  for (int t = tid; t < tasks; t += nthreads) {
    const int c = t & (FFT_C - 1);
    const int j = t / FFT_C;
    const int k = j % Ns;
    double2 v[R];
#pragma unroll
    for (int q = 0; q < R; ++q) v[q] = in[fft_phys(j + q * M, c)];
    if (Ns > 1) {
      const int e = k * twstep;
#pragma unroll
      for (int q = 1; q < R; ++q) {
        double2 w = __ldg(&tw[q * e]);
        v[q] = DIR > 0 ? cmul(v[q], w) : cmulc(v[q], w);
      }
    }
    Dft<R, DIR>::run(v);
    const int j0 = (j - k) * R + k;
#pragma unroll
    for (int q = 0; q < R; ++q) out[fft_phys(j0 + q * Ns, c)] = v[q];
  }
}

// all passes of one axis; returns the buffer holding the result.  Caller must __syncthreads() before (tile
// complete) -- this function syncs after every pass, so the result is visible to all threads on return.
template <int DIR>
__device__ __forceinline__ double2* fft_tile(double2* a, double2* b, const FftAxis& ax, int tid, int nthreads) {
  int Ns = 1;
  for (int p = 0; p < ax.npass; ++p) {
    const int R = ax.radix[p];
    switch (R) {
      case 2: fft_pass<2, DIR>(a, b, ax.n, Ns, ax.tw, tid, nthreads); break;
      case 3: fft_pass<3, DIR>(a, b, ax.n, Ns, ax.tw, tid, nthreads); break;
      case 4: fft_pass<4, DIR>(a, b, ax.n, Ns, ax.tw, tid, nthreads); break;
      case 5: fft_pass<5, DIR>(a, b, ax.n, Ns, ax.tw, tid, nthreads); break;
      case 6: fft_pass<6, DIR>(a, b, ax.n, Ns, ax.tw, tid, nthreads); break;
      case 8: fft_pass<8, DIR>(a, b, ax.n, Ns, ax.tw, tid, nthreads); break;
      case 9: fft_pass<9, DIR>(a, b, ax.n, Ns, ax.tw, tid, nthreads); break;
      case 10: fft_pass<10, DIR>(a, b, ax.n, Ns, ax.tw, tid, nthreads); break;
      case 12: fft_pass<12, DIR>(a, b, ax.n, Ns, ax.tw, tid, nthreads); break;
      case 16: fft_pass<16, DIR>(a, b, ax.n, Ns, ax.tw, tid, nthreads); break;
      default: break;
    }
    __syncthreads();
    Ns *= R;
    double2* t = a;
    a = b;
    b = t;
  }
  return a;
}

}  // namespace qehpsi
