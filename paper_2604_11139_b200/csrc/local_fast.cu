// local_fast.cu -- the local-potential part of H psi with register-resident two-pass transforms (fft_reg.cuh).
//
//   w_loc = gather( FFT( V_loc(r) . iFFT( scatter(psi) ) ) )
//   out   = alpha * ((kin - c) . y + w_loc) - beta * y_prev
//
// Every axis length is factored n = r1 * r2 with r1 <= 16, r2 <= 12.  A 1-D transform is two passes over a line held
// in shared memory, each thread owning one radix-r1 ("strided role": elements q*r2 + sub) or radix-r2 ("contiguous
// role": elements sub*r2 + q) sub-transform in registers; both passes are in place, so the real-space data sit in
// "slot" order  slot s  <->  position (s / r2) + r1 * (s % r2)  and the forward transforms undo it.  V_loc/F is stored
// once in that slot order (and with y fastest) by pwh_ham_setup, so no reordering pass exists.  Lanes of a warp sit on
// different lines (odd line strides => conflict-free 16-byte shared accesses) and share their twiddles.
//
// Three kernels per group of bands; the n1*n2*n3 box never exists in HBM:
//   kf_scatter_zinv : sphere -> touched z-columns, inverse z transform, store plane-major  [band][zslot][column]
//   kf_plane        : per (band, z-plane): disc -> shared memory, inverse y on the touched x-lines, then per batch of
//                     y-slots: inverse x, multiply by V_loc/F in registers, forward x, keep the touched x-lines;
//                     forward y; store the disc back in place
//   kf_zfwd_gather  : forward z transform of the columns, gather the sphere, fused kinetic + three-term recurrence
#include <type_traits>

#include "fft_reg.cuh"
#include "launch.h"

namespace pwh {

namespace {

constexpr int ZT = 256;        // threads of the z kernels
constexpr int PT_MAX = 512;    // threads of the plane kernel (256 when two CTAs fit on an SM)

template <int R>
using RC = std::integral_constant<int, R>;

// call f(RC<r>) for the runtime radix r; `BIG` also instantiates the radices only used as r1
template <bool BIG, class F>
__device__ __forceinline__ void with_radix(int r, F&& f) {
  switch (r) {
    case 1: f(RC<1>()); break;
    case 2: f(RC<2>()); break;
    case 3: f(RC<3>()); break;
    case 4: f(RC<4>()); break;
    case 5: f(RC<5>()); break;
    case 6: f(RC<6>()); break;
    case 8: f(RC<8>()); break;
    case 9: f(RC<9>()); break;
    case 10: f(RC<10>()); break;
    case 12: f(RC<12>()); break;
    case 15: if constexpr (BIG) f(RC<15>()); break;
    case 16: if constexpr (BIG) f(RC<16>()); break;
    default: break;
  }
}

// One pass over `nsub * nlines` work items: item -> (sub, line); v[q] = ld(sub, q, line); DFT_R; optional twiddle
// v[q] *= exp(DIR 2 pi i sub q / n) (table tw[t] = exp(+2 pi i t / n)); st(sub, q, line, v[q]).
template <int R, int DIR, bool TW, class LD, class ST>
__device__ __forceinline__ void run_pass(int nsub, int nlines, FastDiv div_lines, const c128* __restrict__ tw, int tid,
                                         int nthr, LD ld, ST st) {
  const int total = nsub * nlines;
  for (int i = tid; i < total; i += nthr) {
    uint32_t sub, line;
    div_lines.divmod((uint32_t)i, sub, line);
    c128 v[R];
#pragma unroll
    for (int q = 0; q < R; ++q) v[q] = ld((int)sub, q, (int)line);
    Dft<R, DIR>::run(v);
    if (TW) {
#pragma unroll
      for (int q = 1; q < R; ++q) {
        const c128 t = tw[sub * q];
        v[q] = DIR > 0 ? cmul(v[q], t) : cmulc(v[q], t);
      }
    }
#pragma unroll
    for (int q = 0; q < R; ++q) st((int)sub, q, (int)line, v[q]);
  }
}

__device__ __forceinline__ void copy_tw(c128* dst, const c128* __restrict__ src, int n, int tid, int nthr) {
  for (int i = tid; i < n; i += nthr) dst[i] = src[i];
}

// ---------------------------------------------------------------------------------------------------------------
// z kernels
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(ZT) kf_scatter_zinv(const FastPlan P, const c128* __restrict__ psi, int64_t ldpsi,
                                                      c128* __restrict__ colbuf) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128* lines = reinterpret_cast<c128*>(smem_raw);   // [colgrp][zstride]
  c128* tw = lines + P.colgrp * P.zstride;
  const int tid = threadIdx.x, grp = blockIdx.x, band = blockIdx.y;
  const int nline = P.colgrp * P.zstride;
  for (int i = tid; i < nline; i += ZT) lines[i] = cmake(0.0, 0.0);
  copy_tw(tw, P.tw[2], P.n3, tid, ZT);
  __syncthreads();
  const c128* src = psi + (int64_t)band * ldpsi;
  const int e0 = P.grp_ptr[grp], e1 = P.grp_ptr[grp + 1];
  for (int e = e0 + tid; e < e1; e += ZT) lines[P.ent_off[e]] = src[P.ent_pw[e]];
  __syncthreads();
  const int r1 = P.r1[2], r2 = P.r2[2], zs = P.zstride;
  c128* dst = colbuf + (int64_t)band * P.n3 * P.ncols_pad + grp * P.colgrp;
  const int64_t pstride = P.ncols_pad;
  if (r2 == 1) {
    with_radix<true>(r1, [&](auto rc) {
      constexpr int R = decltype(rc)::value;
      run_pass<R, +1, false>(1, P.colgrp, P.div_colgrp, tw, tid, ZT,
                             [&](int, int q, int c) { return lines[c * zs + q]; },
                             [&](int, int q, int c, c128 v) { dst[(int64_t)q * pstride + c] = v; });
    });
    return;
  }
  with_radix<true>(r1, [&](auto rc) {
    constexpr int R = decltype(rc)::value;
    run_pass<R, +1, true>(r2, P.colgrp, P.div_colgrp, tw, tid, ZT,
                          [&](int sub, int q, int c) { return lines[c * zs + q * r2 + sub]; },
                          [&](int sub, int q, int c, c128 v) { lines[c * zs + q * r2 + sub] = v; });
  });
  __syncthreads();
  with_radix<false>(r2, [&](auto rc) {
    constexpr int R = decltype(rc)::value;
    run_pass<R, +1, false>(r1, P.colgrp, P.div_colgrp, tw, tid, ZT,
                           [&](int sub, int q, int c) { return lines[c * zs + sub * r2 + q]; },
                           [&](int sub, int q, int c, c128 v) { dst[(int64_t)(sub * r2 + q) * pstride + c] = v; });
  });
}

// `out` may alias `y` or `yprev`: entry g of the three is read and written by the same thread, in that order.
__global__ void __launch_bounds__(ZT) kf_zfwd_gather(const FastPlan P, const c128* __restrict__ colbuf,
                                                     const c128* y, int64_t ldy,
                                                     const c128* yprev, int64_t ldprev,
                                                     c128* out, int64_t ldout, double alpha, double cshift,
                                                     double beta) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128* lines = reinterpret_cast<c128*>(smem_raw);
  c128* tw = lines + P.colgrp * P.zstride;
  const int tid = threadIdx.x, grp = blockIdx.x, band = blockIdx.y;
  copy_tw(tw, P.tw[2], P.n3, tid, ZT);
  __syncthreads();
  const c128* src = colbuf + (int64_t)band * P.n3 * P.ncols_pad + grp * P.colgrp;
  const int64_t pstride = P.ncols_pad;
  const int r1 = P.r1[2], r2 = P.r2[2], zs = P.zstride;
  if (r2 == 1) {
    with_radix<true>(r1, [&](auto rc) {
      constexpr int R = decltype(rc)::value;
      run_pass<R, -1, false>(1, P.colgrp, P.div_colgrp, tw, tid, ZT,
                             [&](int, int q, int c) { return src[(int64_t)q * pstride + c]; },
                             [&](int, int q, int c, c128 v) { lines[c * zs + q] = v; });
    });
  } else {
    with_radix<false>(r2, [&](auto rc) {
      constexpr int R = decltype(rc)::value;
      run_pass<R, -1, true>(r1, P.colgrp, P.div_colgrp, tw, tid, ZT,
                            [&](int sub, int q, int c) { return src[(int64_t)(sub * r2 + q) * pstride + c]; },
                            [&](int sub, int q, int c, c128 v) { lines[c * zs + sub * r2 + q] = v; });
    });
    __syncthreads();
    with_radix<true>(r1, [&](auto rc) {
      constexpr int R = decltype(rc)::value;
      run_pass<R, -1, false>(r2, P.colgrp, P.div_colgrp, tw, tid, ZT,
                             [&](int sub, int q, int c) { return lines[c * zs + q * r2 + sub]; },
                             [&](int sub, int q, int c, c128 v) { lines[c * zs + q * r2 + sub] = v; });
    });
  }
  __syncthreads();
  const c128* yb = y + (int64_t)band * ldy;
  const c128* pb = (beta != 0.0) ? yprev + (int64_t)band * ldprev : nullptr;
  c128* ob = out + (int64_t)band * ldout;
  const int e0 = P.grp_ptr[grp], e1 = P.grp_ptr[grp + 1];
  for (int e = e0 + tid; e < e1; e += ZT) {
    const int g = P.ent_pw[e];
    const c128 w = lines[P.ent_off[e]];
    const c128 yv = yb[g];
    const double k = P.kin[g] - cshift;
    c128 r = cmake(alpha * fma(k, yv.x, w.x), alpha * fma(k, yv.y, w.y));
    if (pb) {
      const c128 pv = pb[g];
      r.x = fma(-beta, pv.x, r.x);
      r.y = fma(-beta, pv.y, r.y);
    }
    ob[g] = r;
  }
}

// ---------------------------------------------------------------------------------------------------------------
// plane kernel
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(PT_MAX, 1) kf_plane(const FastPlan P, c128* __restrict__ colbuf) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128* half = reinterpret_cast<c128*>(smem_raw);       // [nxl][ystride]   touched x-lines x all y
  c128* T = half + P.nxl * P.ystride;                   // [n1][yb]         one batch of full-length x-lines
  c128* twx = T + P.tsize;
  c128* twy = twx + P.n1;
  short* xl_of_x = reinterpret_cast<short*>(twy + P.n2);  // [n1]
  const int tid = threadIdx.x, nthr = blockDim.x, zslot = blockIdx.x, band = blockIdx.y;
  const int ys = P.ystride, nxl = P.nxl, YB = P.yb;
  const int r1x = P.r1[0], r2x = P.r2[0], r1y = P.r1[1], r2y = P.r2[1];

  const int nhalf = nxl * ys;
  for (int i = tid; i < nhalf; i += nthr) half[i] = cmake(0.0, 0.0);
  copy_tw(twx, P.tw[0], P.n1, tid, nthr);
  copy_tw(twy, P.tw[1], P.n2, tid, nthr);
  for (int i = tid; i < P.n1; i += nthr) xl_of_x[i] = P.xl_of_x[i];
  __syncthreads();
  c128* plane = colbuf + ((int64_t)band * P.n3 + zslot) * P.ncols_pad;
  for (int c = tid; c < P.ncols; c += nthr) half[P.col_hp[c]] = plane[c];
  __syncthreads();

  // ---- inverse y on the touched x-lines (in place; output in y-slot order)
  with_radix<true>(r1y, [&](auto rc) {
    constexpr int R = decltype(rc)::value;
    if (r2y == 1)
      run_pass<R, +1, false>(1, nxl, P.div_nxl, twy, tid, nthr,
                             [&](int, int q, int l) { return half[l * ys + q]; },
                             [&](int, int q, int l, c128 v) { half[l * ys + q] = v; });
    else
      run_pass<R, +1, true>(r2y, nxl, P.div_nxl, twy, tid, nthr,
                            [&](int sub, int q, int l) { return half[l * ys + q * r2y + sub]; },
                            [&](int sub, int q, int l, c128 v) { half[l * ys + q * r2y + sub] = v; });
  });
  __syncthreads();
  if (r2y > 1) {
    with_radix<false>(r2y, [&](auto rc) {
      constexpr int R = decltype(rc)::value;
      run_pass<R, +1, false>(r1y, nxl, P.div_nxl, twy, tid, nthr,
                             [&](int sub, int q, int l) { return half[l * ys + sub * r2y + q]; },
                             [&](int sub, int q, int l, c128 v) { half[l * ys + sub * r2y + q] = v; });
    });
    __syncthreads();
  }

  // ---- x direction, one batch of YB y-slots at a time
  const double* __restrict__ vz = P.vslot + (int64_t)zslot * P.n1 * P.n2;   // [xslot][yslot]
  const int n2 = P.n2;
  for (int y0 = 0; y0 < n2; y0 += YB) {
    if (r2x == 1) {
      // single-pass x transform: inverse, multiply, forward, all in registers
      with_radix<true>(r1x, [&](auto rc) {
        constexpr int R = decltype(rc)::value;
        for (int yb = tid; yb < YB; yb += nthr) {
          c128 v[R];
#pragma unroll
          for (int q = 0; q < R; ++q) {
            const int xl = xl_of_x[q];
            v[q] = xl >= 0 ? half[xl * ys + y0 + yb] : cmake(0.0, 0.0);
          }
          Dft<R, +1>::run(v);
#pragma unroll
          for (int q = 0; q < R; ++q) v[q] = cscale(vz[(int64_t)q * n2 + y0 + yb], v[q]);
          Dft<R, -1>::run(v);
#pragma unroll
          for (int q = 0; q < R; ++q) {
            const int xl = xl_of_x[q];
            if (xl >= 0) half[xl * ys + y0 + yb] = v[q];
          }
        }
      });
      continue;   // different y-slots never interact: no barrier needed between batches
    }
    // (a) strided role: radix r1x over i1, twiddle, into T
    with_radix<true>(r1x, [&](auto rc) {
      constexpr int R = decltype(rc)::value;
      run_pass<R, +1, true>(r2x, YB, P.div_yb, twx, tid, nthr,
                            [&](int sub, int q, int yb) {
                              const int xl = xl_of_x[q * r2x + sub];
                              return xl >= 0 ? half[xl * ys + y0 + yb] : cmake(0.0, 0.0);
                            },
                            [&](int sub, int q, int yb, c128 v) { T[(q * r2x + sub) * YB + yb] = v; });
    });
    __syncthreads();
    // (b) contiguous role: radix r2x inverse -> real space, multiply by V_loc/F, radix r2x forward, twiddle
    with_radix<false>(r2x, [&](auto rc) {
      constexpr int R = decltype(rc)::value;
      const int total = r1x * YB;
      for (int i = tid; i < total; i += nthr) {
        uint32_t k1, yb;
        P.div_yb.divmod((uint32_t)i, k1, yb);
        c128* t = T + (k1 * r2x) * YB + yb;
        c128 v[R];
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = t[q * YB];
        Dft<R, +1>::run(v);
        const double* vv = vz + (int64_t)(k1 * r2x) * n2 + y0 + yb;
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = cscale(vv[(int64_t)q * n2], v[q]);
        Dft<R, -1>::run(v);
#pragma unroll
        for (int q = 1; q < R; ++q) v[q] = cmulc(v[q], twx[k1 * q]);
#pragma unroll
        for (int q = 0; q < R; ++q) t[q * YB] = v[q];
      }
    });
    __syncthreads();
    // (c) strided role: radix r1x forward over k1, keep the touched x-lines
    with_radix<true>(r1x, [&](auto rc) {
      constexpr int R = decltype(rc)::value;
      run_pass<R, -1, false>(r2x, YB, P.div_yb, twx, tid, nthr,
                             [&](int sub, int q, int yb) { return T[(q * r2x + sub) * YB + yb]; },
                             [&](int sub, int q, int yb, c128 v) {
                               const int xl = xl_of_x[q * r2x + sub];
                               if (xl >= 0) half[xl * ys + y0 + yb] = v;
                             });
    });
    __syncthreads();
  }
  if (r2x == 1) __syncthreads();

  // ---- forward y (in place; back to natural order)
  if (r2y > 1) {
    with_radix<false>(r2y, [&](auto rc) {
      constexpr int R = decltype(rc)::value;
      run_pass<R, -1, true>(r1y, nxl, P.div_nxl, twy, tid, nthr,
                            [&](int sub, int q, int l) { return half[l * ys + sub * r2y + q]; },
                            [&](int sub, int q, int l, c128 v) { half[l * ys + sub * r2y + q] = v; });
    });
    __syncthreads();
  }
  with_radix<true>(r1y, [&](auto rc) {
    constexpr int R = decltype(rc)::value;
    if (r2y == 1)
      run_pass<R, -1, false>(1, nxl, P.div_nxl, twy, tid, nthr,
                             [&](int, int q, int l) { return half[l * ys + q]; },
                             [&](int, int q, int l, c128 v) { half[l * ys + q] = v; });
    else
      run_pass<R, -1, false>(r2y, nxl, P.div_nxl, twy, tid, nthr,
                             [&](int sub, int q, int l) { return half[l * ys + q * r2y + sub]; },
                             [&](int sub, int q, int l, c128 v) { half[l * ys + q * r2y + sub] = v; });
  });
  __syncthreads();
  for (int c = tid; c < P.ncols; c += nthr) plane[c] = half[P.col_hp[c]];
}


// ---------------------------------------------------------------------------------------------------------------
// density accumulation (Algorithm 3 step 10)
// ---------------------------------------------------------------------------------------------------------------
// One CTA per z-slot walks over the bands of the group in order: disc -> inverse y -> inverse x (the first half of
// kf_plane), then acc[zslot][xslot][yslot] += occ[band] |u|^2.  A real-space point is owned by one thread of one CTA and
// the bands come in a fixed order, so the sum is deterministic.  acc is in slot order; kf_density_unslot adds it to the
// caller's array in natural order.
__global__ void __launch_bounds__(PT_MAX, 1) kf_density_plane(const FastPlan P, const c128* __restrict__ colbuf, int nb,
                                                              const double* __restrict__ occ, double* __restrict__ acc) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128* half = reinterpret_cast<c128*>(smem_raw);
  c128* T = half + P.nxl * P.ystride;
  c128* twx = T + P.tsize;
  c128* twy = twx + P.n1;
  short* xl_of_x = reinterpret_cast<short*>(twy + P.n2);
  const int tid = threadIdx.x, nthr = blockDim.x, zslot = blockIdx.x;
  const int ys = P.ystride, nxl = P.nxl, YB = P.yb;
  const int r1x = P.r1[0], r2x = P.r2[0], r1y = P.r1[1], r2y = P.r2[1];
  const int n2 = P.n2;
  copy_tw(twx, P.tw[0], P.n1, tid, nthr);
  copy_tw(twy, P.tw[1], P.n2, tid, nthr);
  for (int i = tid; i < P.n1; i += nthr) xl_of_x[i] = P.xl_of_x[i];
  double* __restrict__ az = acc + (int64_t)zslot * P.n1 * P.n2;   // [xslot][yslot]
  const int nhalf = nxl * ys;
  for (int band = 0; band < nb; ++band) {
    const double f = occ[band];
    __syncthreads();
    for (int i = tid; i < nhalf; i += nthr) half[i] = cmake(0.0, 0.0);
    __syncthreads();
    const c128* plane = colbuf + ((int64_t)band * P.n3 + zslot) * P.ncols_pad;
    for (int c = tid; c < P.ncols; c += nthr) half[P.col_hp[c]] = plane[c];
    __syncthreads();
    with_radix<true>(r1y, [&](auto rc) {
      constexpr int R = decltype(rc)::value;
      if (r2y == 1)
        run_pass<R, +1, false>(1, nxl, P.div_nxl, twy, tid, nthr,
                               [&](int, int q, int l) { return half[l * ys + q]; },
                               [&](int, int q, int l, c128 v) { half[l * ys + q] = v; });
      else
        run_pass<R, +1, true>(r2y, nxl, P.div_nxl, twy, tid, nthr,
                              [&](int sub, int q, int l) { return half[l * ys + q * r2y + sub]; },
                              [&](int sub, int q, int l, c128 v) { half[l * ys + q * r2y + sub] = v; });
    });
    __syncthreads();
    if (r2y > 1) {
      with_radix<false>(r2y, [&](auto rc) {
        constexpr int R = decltype(rc)::value;
        run_pass<R, +1, false>(r1y, nxl, P.div_nxl, twy, tid, nthr,
                               [&](int sub, int q, int l) { return half[l * ys + sub * r2y + q]; },
                               [&](int sub, int q, int l, c128 v) { half[l * ys + sub * r2y + q] = v; });
      });
      __syncthreads();
    }
    for (int y0 = 0; y0 < n2; y0 += YB) {
      if (r2x == 1) {
        with_radix<true>(r1x, [&](auto rc) {
          constexpr int R = decltype(rc)::value;
          for (int yb = tid; yb < YB; yb += nthr) {
            c128 v[R];
#pragma unroll
            for (int q = 0; q < R; ++q) {
              const int xl = xl_of_x[q];
              v[q] = xl >= 0 ? half[xl * ys + y0 + yb] : cmake(0.0, 0.0);
            }
            Dft<R, +1>::run(v);
            double old[R];
#pragma unroll
            for (int q = 0; q < R; ++q) old[q] = az[(int64_t)q * n2 + y0 + yb];
#pragma unroll
            for (int q = 0; q < R; ++q)
              az[(int64_t)q * n2 + y0 + yb] = fma(f, fma(v[q].x, v[q].x, v[q].y * v[q].y), old[q]);
          }
        });
        continue;
      }
      with_radix<true>(r1x, [&](auto rc) {
        constexpr int R = decltype(rc)::value;
        run_pass<R, +1, true>(r2x, YB, P.div_yb, twx, tid, nthr,
                              [&](int sub, int q, int yb) {
                                const int xl = xl_of_x[q * r2x + sub];
                                return xl >= 0 ? half[xl * ys + y0 + yb] : cmake(0.0, 0.0);
                              },
                              [&](int sub, int q, int yb, c128 v) { T[(q * r2x + sub) * YB + yb] = v; });
      });
      __syncthreads();
      with_radix<false>(r2x, [&](auto rc) {
        constexpr int R = decltype(rc)::value;
        const int total = r1x * YB;
        for (int i = tid; i < total; i += nthr) {
          uint32_t k1, yb;
          P.div_yb.divmod((uint32_t)i, k1, yb);
          const c128* t = T + (k1 * r2x) * YB + yb;
          c128 v[R];
#pragma unroll
          for (int q = 0; q < R; ++q) v[q] = t[q * YB];
          Dft<R, +1>::run(v);
          double* a = az + (int64_t)(k1 * r2x) * n2 + y0 + yb;
          // read-modify-write of R entries through one pointer: all loads first, or each load waits for the store before it
          double old[R];
#pragma unroll
          for (int q = 0; q < R; ++q) old[q] = a[(int64_t)q * n2];
#pragma unroll
          for (int q = 0; q < R; ++q) a[(int64_t)q * n2] = fma(f, fma(v[q].x, v[q].x, v[q].y * v[q].y), old[q]);
        }
      });
      __syncthreads();
    }
  }
}

// rho[x + n1 (y + n2 z)] += weight * acc[(zs n1 + xs) n2 + ys]  with the slot maps of k_slot_vloc (pwham.cu)
__global__ void kf_density_unslot(int n1, int n2, int n3, int r1x, int r2x, int r1y, int r2y, int r1z, int r2z,
                                  const double* __restrict__ acc, double weight, double* __restrict__ rho) {
  const int64_t total = (int64_t)n1 * n2 * n3;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int ys = (int)(i % n2);
    const int xs = (int)((i / n2) % n1);
    const int zs = (int)(i / ((int64_t)n1 * n2));
    const int x = xs / r2x + r1x * (xs % r2x), y = ys / r2y + r1y * (ys % r2y), z = zs / r2z + r1z * (zs % r2z);
    double* r = rho + x + (int64_t)n1 * (y + (int64_t)n2 * z);
    *r = fma(weight, acc[i], *r);
  }
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------------
size_t fast_zkernel_smem(const FastPlan& P) { return sizeof(c128) * ((size_t)P.colgrp * P.zstride + P.n3); }
size_t fast_plane_smem(const FastPlan& P) {
  return sizeof(c128) * ((size_t)P.nxl * P.ystride + (size_t)P.tsize + P.n1 + P.n2) + sizeof(short) * P.n1;
}

cudaError_t fast_kernels_init(const FastPlan& P) {
  cudaError_t e;
  e = set_max_dyn_smem(reinterpret_cast<const void*>(&kf_scatter_zinv));
  if (e != cudaSuccess) return e;
  e = set_max_dyn_smem(reinterpret_cast<const void*>(&kf_zfwd_gather));
  if (e != cudaSuccess) return e;
  e = set_max_dyn_smem(reinterpret_cast<const void*>(&kf_plane));
  if (e != cudaSuccess) return e;
  return set_max_dyn_smem(reinterpret_cast<const void*>(&kf_density_plane));
}

void launch_fast_scatter_zinv(const FastPlan& P, const c128* psi, int64_t ldpsi, c128* colbuf, int nb, cudaStream_t st) {
  dim3 grid(P.ngrp, nb);
  ScopedLaunch sl(ST_SCATTER_ZINV, st);
  kf_scatter_zinv<<<grid, ZT, fast_zkernel_smem(P), st>>>(P, psi, ldpsi, colbuf);
}

void launch_fast_plane(const FastPlan& P, c128* colbuf, int nb, cudaStream_t st) {
  dim3 grid(P.n3, nb);
  ScopedLaunch sl(ST_PLANE, st);
  kf_plane<<<grid, P.plane_threads, fast_plane_smem(P), st>>>(P, colbuf);
}

void launch_fast_density_plane(const FastPlan& P, const c128* colbuf, int nb, const double* occ, double* acc, cudaStream_t st) {
  ScopedLaunch sl(ST_PLANE, st);
  kf_density_plane<<<P.n3, P.plane_threads, fast_plane_smem(P), st>>>(P, colbuf, nb, occ, acc);
}

void launch_fast_density_unslot(const FastPlan& P, const double* acc, double weight, double* rho, cudaStream_t st) {
  ScopedLaunch sl(ST_AXPY, st);
  kf_density_unslot<<<148 * 4, 256, 0, st>>>(P.n1, P.n2, P.n3, P.r1[0], P.r2[0], P.r1[1], P.r2[1], P.r1[2], P.r2[2], acc, weight,
                                             rho);
}

void launch_fast_zfwd_gather(const FastPlan& P, const c128* colbuf, const c128* y, int64_t ldy, const c128* yprev,
                             int64_t ldprev, c128* out, int64_t ldout, double alpha, double cshift, double beta, int nb,
                             cudaStream_t st) {
  dim3 grid(P.ngrp, nb);
  ScopedLaunch sl(ST_ZFWD_GATHER, st);
  kf_zfwd_gather<<<grid, ZT, fast_zkernel_smem(P), st>>>(P, colbuf, y, ldy, yprev, ldprev, out, ldout, alpha, cshift, beta);
}

}  // namespace pwh
