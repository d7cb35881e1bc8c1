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

// ---- pruned transforms -------------------------------------------------------------------------------------------------
// The sphere occupies a prefix of every spectral axis once the axis is indexed from its lowest touched line (a shift of the
// spectral index is a phase in real space, which cancels between the inverse and the forward transform around the real,
// pointwise V_loc multiply).  In the strided-role pass of n = R * r2 the inputs of one radix-R transform are the lines
// s + r2 q: only q < L = ceil(touched / r2) can be non-zero on the way in, and only those outputs are wanted on the way out.

// v0 + exp(DIR 2 pi i K / N) v1 with compile-time K, N
template <int K, int N, int DIR>
__device__ __forceinline__ c128 add_rot(c128 v0, c128 v1) {
  constexpr int k = ((K % N) + N) % N;
  if constexpr (k == 0 || 4 * k == N || 2 * k == N || 4 * k == 3 * N) return cadd(v0, rot<K, N, DIR>(v1));
  else {
    constexpr double c = cos_turn(k, N);
    constexpr double s = (DIR > 0 ? 1.0 : -1.0) * sin_turn(k, N);
    return cmake(fma(c, v1.x, fma(-s, v1.y, v0.x)), fma(c, v1.y, fma(s, v1.x, v0.y)));
  }
}

// DFT of length A whose inputs v[LA..A-1] are zero (they are neither read nor assumed initialised); all A outputs
template <int A, int DIR, int LA>
struct DftIn {
  template <int K>
  __device__ __forceinline__ static void two(c128 v0, c128 v1, c128* v) {
    if constexpr (K < A) {
      v[K] = add_rot<K, A, DIR>(v0, v1);
      two<K + 1>(v0, v1, v);
    }
  }
  __device__ __forceinline__ static void run(c128* v) {
    if constexpr (LA <= 0) {
#pragma unroll
      for (int k = 0; k < A; ++k) v[k] = cmake(0.0, 0.0);
    } else if constexpr (LA == 1) {
#pragma unroll
      for (int k = 1; k < A; ++k) v[k] = v[0];
    } else if constexpr (LA == 2 && A > 2) {
      const c128 v0 = v[0], v1 = v[1];
      two<0>(v0, v1, v);
    } else {
#pragma unroll
      for (int a = (LA < A ? LA : A); a < A; ++a) v[a] = cmake(0.0, 0.0);
      Dft<A, DIR>::run(v);
    }
  }
};

// Cooley-Tukey product R = A * B (n = a*B + b, k = ka + A*kb) with inputs n >= L zero: the first-stage transforms over a
// see only the a with a*B + b < L
template <int A, int B, int DIR, int L>
struct DftCTIn {
  template <int Bi>
  __device__ __forceinline__ static void first(const c128* v, c128 (*t)[A]) {
    if constexpr (Bi < B) {
      constexpr int LA = (L - Bi + B - 1) / B < 0 ? 0 : ((L - Bi + B - 1) / B > A ? A : (L - Bi + B - 1) / B);
      c128 u[A];
#pragma unroll
      for (int a = 0; a < LA; ++a) u[a] = v[a * B + Bi];
      DftIn<A, DIR, LA>::run(u);
      if constexpr (LA > 0) DftCT<A, B, DIR>::template twiddle_row<Bi, 0>(u);
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

// v[0..R-1] <- DFT_R(v) where v[L..R-1] are zero on entry (not read)
template <int R, int DIR, int L>
struct DftPrunedIn {
  __device__ __forceinline__ static void run(c128* v) {
    if constexpr (L >= R) Dft<R, DIR>::run(v);
    else if constexpr (R == 6) DftCTIn<2, 3, DIR, L>::run(v);
    else if constexpr (R == 8) DftCTIn<2, 4, DIR, L>::run(v);
    else if constexpr (R == 9) DftCTIn<3, 3, DIR, L>::run(v);
    else if constexpr (R == 10) DftCTIn<2, 5, DIR, L>::run(v);
    else if constexpr (R == 12) DftCTIn<3, 4, DIR, L>::run(v);
    else if constexpr (R == 15) DftCTIn<3, 5, DIR, L>::run(v);
    else if constexpr (R == 16) DftCTIn<4, 4, DIR, L>::run(v);
    else DftIn<R, DIR, L>::run(v);
  }
};

}  // namespace pwh
