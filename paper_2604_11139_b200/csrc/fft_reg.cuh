// fft_reg.cuh -- register-resident small DFTs (radix 2..16) with compile-time twiddles.
//
// The local-potential kernels factor every axis length n = r1 * r2 (r1, r2 <= 16) and run each 1-D transform as
// two passes in which one thread holds a whole radix-r sub-transform in registers, so a line crosses shared memory
// twice per transform instead of once per radix-2/4 level (the batched FFT pair around the
// pointwise V_loc multiply).  Composite radices are Cooley-Tukey products of the 2/3/4/5 butterflies, fully
// unrolled; their internal twiddles are constexpr (evaluated by the compiler from a Taylor series on an argument
// reduced to the first octant, so they are correct to about one ulp).
#pragma once
#include "common.cuh"

namespace pwh {

// ---- constexpr cos/sin of 2 pi k / n ---------------------------------------------------------------------------
constexpr double kPi = 3.14159265358979323846264338327950288;

__host__ __device__ constexpr double taylor_cos(double x) {  // |x| <= pi/4
  const double x2 = x * x;
  double term = 1.0, sum = 0.0;
  double terms[14] = {0};
  for (int i = 0; i < 14; ++i) {
    terms[i] = term;
    term = -term * x2 / ((2 * i + 1) * (2 * i + 2));
  }
  for (int i = 13; i >= 0; --i) sum += terms[i];
  return sum;
}
__host__ __device__ constexpr double taylor_sin(double x) {  // |x| <= pi/4
  const double x2 = x * x;
  double term = x, sum = 0.0;
  double terms[14] = {0};
  for (int i = 0; i < 14; ++i) {
    terms[i] = term;
    term = -term * x2 / ((2 * i + 2) * (2 * i + 3));
  }
  for (int i = 13; i >= 0; --i) sum += terms[i];
  return sum;
}
// cos(2 pi k / n), exact symmetries first: work in units of 1/(8n) of a turn so that octants are integers
__host__ __device__ constexpr double cos_turn(long k, long n) {
  k %= n;
  if (k < 0) k += n;
  long e = 8 * k;          // angle = 2 pi e / (8 n); octant boundaries at multiples of n
  if (e > 4 * n) e = 8 * n - e;                 // cos(2pi - a) = cos a        -> [0, pi]
  bool neg = false;
  if (e > 2 * n) { e = 4 * n - e; neg = true; } // cos(pi - a) = -cos a        -> [0, pi/2]
  double r = 0.0;
  if (e == 0) r = 1.0;
  else if (e == 2 * n) r = 0.0;
  else if (e == n) r = 0.70710678118654752440084436210485;
  else if (e < n) r = taylor_cos(2.0 * kPi * (double)e / (8.0 * (double)n));
  else r = taylor_sin(2.0 * kPi * (double)(2 * n - e) / (8.0 * (double)n));   // cos a = sin(pi/2 - a)
  return neg ? -r : r;
}
__host__ __device__ constexpr double sin_turn(long k, long n) { return cos_turn(4 * k - n, 4 * n); }   // sin a = cos(a - pi/2)

// v *= exp(DIR * 2 pi i K / N) with K, N compile-time; trivial rotations cost no multiply
template <int K, int N, int DIR>
__device__ __forceinline__ c128 rot(c128 v) {
  constexpr int k = ((K % N) + N) % N;
  if constexpr (k == 0) return v;
  else if constexpr (4 * k == N) return DIR > 0 ? cmake(-v.y, v.x) : cmake(v.y, -v.x);
  else if constexpr (2 * k == N) return cmake(-v.x, -v.y);
  else if constexpr (4 * k == 3 * N) return DIR > 0 ? cmake(v.y, -v.x) : cmake(-v.y, v.x);
  else {
    constexpr double c = cos_turn(k, N);
    constexpr double s = (DIR > 0 ? 1.0 : -1.0) * sin_turn(k, N);
    if constexpr (8 * k == N || 8 * k == 3 * N || 8 * k == 5 * N || 8 * k == 7 * N) {
      // |c| == |s| == 1/sqrt2: two adds and two multiplies
      constexpr double h = 0.70710678118654752440084436210485;
      constexpr double sc = c > 0 ? 1.0 : -1.0, ss = s > 0 ? 1.0 : -1.0;
      // (x + i y)(sc + i ss) h = h (sc x - ss y) + i h (ss x + sc y)
      return cmake(h * (sc * v.x - ss * v.y), h * (ss * v.x + sc * v.y));
    } else {
      return cmake(fma(c, v.x, -s * v.y), fma(c, v.y, s * v.x));
    }
  }
}

template <int R, int DIR>
struct Dft;   // in place on v[0..R-1], natural order in and out: v[k] <- sum_n v[n] exp(DIR 2 pi i n k / R)

template <int DIR>
struct Dft<1, DIR> {
  __device__ __forceinline__ static void run(c128*) {}
};
template <int DIR>
struct Dft<2, DIR> {
  __device__ __forceinline__ static void run(c128* v) {
    const c128 a = v[0], b = v[1];
    v[0] = cadd(a, b);
    v[1] = csub(a, b);
  }
};
template <int DIR>
struct Dft<3, DIR> {
  __device__ __forceinline__ static void run(c128* v) {
    constexpr double S3 = 0.86602540378443864676372317075294 * (DIR > 0 ? 1.0 : -1.0);
    const c128 t = cadd(v[1], v[2]);
    const c128 d = csub(v[1], v[2]);
    const c128 mid = cmake(fma(-0.5, t.x, v[0].x), fma(-0.5, t.y, v[0].y));
    v[0] = cadd(v[0], t);
    // i * S3 * d = (-S3 d.y, S3 d.x)
    v[1] = cmake(fma(-S3, d.y, mid.x), fma(S3, d.x, mid.y));
    v[2] = cmake(fma(S3, d.y, mid.x), fma(-S3, d.x, mid.y));
  }
};
template <int DIR>
struct Dft<4, DIR> {
  __device__ __forceinline__ static void run(c128* v) {
    const c128 t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
    const c128 t2 = cadd(v[1], v[3]), d = csub(v[1], v[3]);
    const c128 t3 = DIR > 0 ? cmake(-d.y, d.x) : cmake(d.y, -d.x);
    v[0] = cadd(t0, t2);
    v[2] = csub(t0, t2);
    v[1] = cadd(t1, t3);
    v[3] = csub(t1, t3);
  }
};
template <int DIR>
struct Dft<5, DIR> {
  __device__ __forceinline__ static void run(c128* v) {
    constexpr double C1 = 0.30901699437494742410229341718282;
    constexpr double C2 = -0.80901699437494742410229341718282;
    constexpr double S1 = 0.95105651629515357211643933337938 * (DIR > 0 ? 1.0 : -1.0);
    constexpr double S2 = 0.58778525229247312916870595463907 * (DIR > 0 ? 1.0 : -1.0);
    const c128 t1 = cadd(v[1], v[4]), t2 = cadd(v[2], v[3]);
    const c128 d1 = csub(v[1], v[4]), d2 = csub(v[2], v[3]);
    const c128 m1 = cmake(fma(C1, t1.x, fma(C2, t2.x, v[0].x)), fma(C1, t1.y, fma(C2, t2.y, v[0].y)));
    const c128 m2 = cmake(fma(C2, t1.x, fma(C1, t2.x, v[0].x)), fma(C2, t1.y, fma(C1, t2.y, v[0].y)));
    const c128 n1 = cmake(fma(S1, d1.x, S2 * d2.x), fma(S1, d1.y, S2 * d2.y));    // to be multiplied by i
    const c128 n2 = cmake(fma(S2, d1.x, -S1 * d2.x), fma(S2, d1.y, -S1 * d2.y));
    v[0] = cadd(v[0], cadd(t1, t2));
    v[1] = cmake(m1.x - n1.y, m1.y + n1.x);
    v[4] = cmake(m1.x + n1.y, m1.y - n1.x);
    v[2] = cmake(m2.x - n2.y, m2.y + n2.x);
    v[3] = cmake(m2.x + n2.y, m2.y - n2.x);
  }
};

// Cooley-Tukey product R = A * B in registers: n = a*B + b, k = ka + A*kb.
template <int A, int B, int DIR>
struct DftCT {
  template <int Bi, int Ka>
  __device__ __forceinline__ static void twiddle_row(c128* u) {
    if constexpr (Ka < A) {
      u[Ka] = rot<Bi * Ka, A * B, DIR>(u[Ka]);
      twiddle_row<Bi, Ka + 1>(u);
    }
  }
  template <int Bi>
  __device__ __forceinline__ static void first(const c128* v, c128 (*t)[A]) {
    if constexpr (Bi < B) {
      c128 u[A];
#pragma unroll
      for (int a = 0; a < A; ++a) u[a] = v[a * B + Bi];
      Dft<A, DIR>::run(u);
      twiddle_row<Bi, 0>(u);
#pragma unroll
      for (int a = 0; a < A; ++a) t[Bi][a] = u[a];
      first<Bi + 1>(v, t);
    }
  }
  __device__ __forceinline__ static void run(c128* v) {
    c128 t[B][A];
    first<0>(v, t);
#pragma unroll
    for (int ka = 0; ka < A; ++ka) {
      c128 u[B];
#pragma unroll
      for (int b = 0; b < B; ++b) u[b] = t[b][ka];
      Dft<B, DIR>::run(u);
#pragma unroll
      for (int kb = 0; kb < B; ++kb) v[ka + A * kb] = u[kb];
    }
  }
};

template <int DIR> struct Dft<6, DIR> { __device__ __forceinline__ static void run(c128* v) { DftCT<2, 3, DIR>::run(v); } };
template <int DIR> struct Dft<8, DIR> { __device__ __forceinline__ static void run(c128* v) { DftCT<2, 4, DIR>::run(v); } };
template <int DIR> struct Dft<9, DIR> { __device__ __forceinline__ static void run(c128* v) { DftCT<3, 3, DIR>::run(v); } };
template <int DIR> struct Dft<10, DIR> { __device__ __forceinline__ static void run(c128* v) { DftCT<2, 5, DIR>::run(v); } };
template <int DIR> struct Dft<12, DIR> { __device__ __forceinline__ static void run(c128* v) { DftCT<3, 4, DIR>::run(v); } };
template <int DIR> struct Dft<15, DIR> { __device__ __forceinline__ static void run(c128* v) { DftCT<3, 5, DIR>::run(v); } };
template <int DIR> struct Dft<16, DIR> { __device__ __forceinline__ static void run(c128* v) { DftCT<4, 4, DIR>::run(v); } };

}  // namespace pwh
