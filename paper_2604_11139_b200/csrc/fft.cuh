// fft.cuh -- in-place mixed-radix complex-FP64 FFT on lines held in shared memory.
//
// Inverse transforms (G -> r, exp(+i)) run decimation-in-frequency and leave their output in digit-permuted
// positions; forward transforms (r -> G, exp(-i)) run decimation-in-time and consume exactly that permuted
// order, so no reordering pass exists anywhere: the pointwise V_loc multiply between them simply uses a copy of
// V_loc stored in permuted positions (built once in pwh_ham_setup).  This is the local-potential step of
// PAPER.md:67, 165, 327 (batched FFT -> pointwise multiply -> FFT), re-designed for shared-memory residency.
#pragma once
#include "common.cuh"

namespace pwh {

// a * (DIR * i)
template <int DIR>
__device__ __forceinline__ c128 mul_i(c128 a) {
  return DIR > 0 ? cmake(-a.y, a.x) : cmake(a.y, -a.x);
}

template <int R, int DIR>
struct Bfly;

template <int DIR>
struct Bfly<2, DIR> {
  __device__ __forceinline__ static void run(c128* v) {
    c128 a = v[0], b = v[1];
    v[0] = cadd(a, b);
    v[1] = csub(a, b);
  }
};

template <int DIR>
struct Bfly<3, DIR> {
  __device__ __forceinline__ static void run(c128* v) {
    const double S3 = 0.86602540378443864676372317075294;  // sqrt(3)/2
    c128 t = cadd(v[1], v[2]);
    c128 d = mul_i<DIR>(cscale(S3, csub(v[1], v[2])));
    c128 mid = cmake(fma(-0.5, t.x, v[0].x), fma(-0.5, t.y, v[0].y));
    v[0] = cadd(v[0], t);
    v[1] = cadd(mid, d);
    v[2] = csub(mid, d);
  }
};

template <int DIR>
struct Bfly<4, DIR> {
  __device__ __forceinline__ static void run(c128* v) {
    c128 t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
    c128 t2 = cadd(v[1], v[3]), t3 = mul_i<DIR>(csub(v[1], v[3]));
    v[0] = cadd(t0, t2);
    v[2] = csub(t0, t2);
    v[1] = cadd(t1, t3);
    v[3] = csub(t1, t3);
  }
};

template <int DIR>
struct Bfly<5, DIR> {
  __device__ __forceinline__ static void run(c128* v) {
    const double C1 = 0.30901699437494742410229341718282;   // cos(2 pi/5)
    const double C2 = -0.80901699437494742410229341718282;  // cos(4 pi/5)
    const double S1 = 0.95105651629515357211643933337938;   // sin(2 pi/5)
    const double S2 = 0.58778525229247312916870595463907;   // sin(4 pi/5)
    c128 t1 = cadd(v[1], v[4]), t2 = cadd(v[2], v[3]);
    c128 d1 = csub(v[1], v[4]), d2 = csub(v[2], v[3]);
    c128 m1 = cmake(fma(C1, t1.x, fma(C2, t2.x, v[0].x)), fma(C1, t1.y, fma(C2, t2.y, v[0].y)));
    c128 m2 = cmake(fma(C2, t1.x, fma(C1, t2.x, v[0].x)), fma(C2, t1.y, fma(C1, t2.y, v[0].y)));
    c128 n1 = mul_i<DIR>(cmake(fma(S1, d1.x, S2 * d2.x), fma(S1, d1.y, S2 * d2.y)));
    c128 n2 = mul_i<DIR>(cmake(fma(S2, d1.x, -S1 * d2.x), fma(S2, d1.y, -S1 * d2.y)));
    v[0] = cadd(v[0], cadd(t1, t2));
    v[1] = cadd(m1, n1);
    v[4] = csub(m1, n1);
    v[2] = cadd(m2, n2);
    v[3] = csub(m2, n2);
  }
};

template <int DIR>
struct Bfly<8, DIR> {
  __device__ __forceinline__ static void run(c128* v) {
    const double H = 0.70710678118654752440084436210485;  // 1/sqrt(2)
    c128 e[4] = {v[0], v[2], v[4], v[6]};
    c128 o[4] = {v[1], v[3], v[5], v[7]};
    Bfly<4, DIR>::run(e);
    Bfly<4, DIR>::run(o);
    // w8^1 = (1 + DIR i)/sqrt2, w8^2 = DIR i, w8^3 = (-1 + DIR i)/sqrt2
    c128 o1 = cscale(H, cadd(o[1], mul_i<DIR>(o[1])));
    c128 o2 = mul_i<DIR>(o[2]);
    c128 o3 = cscale(H, csub(mul_i<DIR>(o[3]), o[3]));
    v[0] = cadd(e[0], o[0]);
    v[4] = csub(e[0], o[0]);
    v[1] = cadd(e[1], o1);
    v[5] = csub(e[1], o1);
    v[2] = cadd(e[2], o2);
    v[6] = csub(e[2], o2);
    v[3] = cadd(e[3], o3);
    v[7] = csub(e[3], o3);
  }
};

// One stage over `nlines` lines: work item i -> (butterfly j = i / nlines, line = i % nlines), so the lanes of a
// warp sit on different lines (odd line stride => conflict-free 16-byte accesses) and share one twiddle.
template <int R, int DIR, bool DIT>
__device__ __forceinline__ void fft_stage(c128* base, int nlines, FastDiv div_lines, int lstride, int n, int m,
                                          FastDiv div_m, const c128* tw, int tid, int nthr) {
  const int total = nlines * (n / R);
  const bool has_tw = m > 1;
  for (int i = tid; i < total; i += nthr) {
    uint32_t j, line, blk, n2;
    div_lines.divmod((uint32_t)i, j, line);
    div_m.divmod(j, blk, n2);
    c128* p = base + line * lstride + blk * (R * m) + n2;
    c128 v[R];
#pragma unroll
    for (int q = 0; q < R; ++q) v[q] = p[q * m];
    if (DIT && has_tw) {
#pragma unroll
      for (int q = 1; q < R; ++q) {
        c128 t = tw[(q - 1) * m + n2];
        v[q] = DIR > 0 ? cmul(v[q], t) : cmulc(v[q], t);
      }
    }
    Bfly<R, DIR>::run(v);
    if (!DIT && has_tw) {
#pragma unroll
      for (int q = 1; q < R; ++q) {
        c128 t = tw[(q - 1) * m + n2];
        v[q] = DIR > 0 ? cmul(v[q], t) : cmulc(v[q], t);
      }
    }
#pragma unroll
    for (int q = 0; q < R; ++q) p[q * m] = v[q];
  }
}

// Transform `nlines` lines of length pl.n (stride lstride) in shared memory; ends with __syncthreads().
// DIR=+1: exp(+i), DIF, natural -> permuted.   DIR=-1: exp(-i), DIT, permuted -> natural.
template <int DIR>
__device__ __forceinline__ void fft_lines(c128* base, int nlines, FastDiv div_lines, int lstride, const AxisPlan& pl,
                                          const c128* tw, int tid, int nthr) {
  constexpr bool DIT = DIR < 0;
  for (int si = 0; si < pl.nstages; ++si) {
    const int s = DIT ? pl.nstages - 1 - si : si;
    const int r = pl.radix[s], m = pl.m[s];
    const c128* t = tw + pl.tw_off[s];
    switch (r) {
      case 8: fft_stage<8, DIR, DIT>(base, nlines, div_lines, lstride, pl.n, m, pl.div_m[s], t, tid, nthr); break;
      case 5: fft_stage<5, DIR, DIT>(base, nlines, div_lines, lstride, pl.n, m, pl.div_m[s], t, tid, nthr); break;
      case 4: fft_stage<4, DIR, DIT>(base, nlines, div_lines, lstride, pl.n, m, pl.div_m[s], t, tid, nthr); break;
      case 3: fft_stage<3, DIR, DIT>(base, nlines, div_lines, lstride, pl.n, m, pl.div_m[s], t, tid, nthr); break;
      default: fft_stage<2, DIR, DIT>(base, nlines, div_lines, lstride, pl.n, m, pl.div_m[s], t, tid, nthr); break;
    }
    __syncthreads();
  }
}

}  // namespace pwh
