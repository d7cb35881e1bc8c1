// local_z.cu -- warp-private z transforms of the local-potential part of H psi.
//
//   kz_scatter_zinv : sphere -> touched z-columns, inverse z transform, store plane-major [band][z-slot][column]
//
//   kz_zfwd_gather  : forward z transform of the columns, gather the sphere, fused kinetic + three-term recurrence
//                     out = alpha * ((kin - c) . y + w_loc) - beta * y_prev
//
// Same arithmetic as kf_scatter_zinv / kf_zfwd_gather in local_fast.cu (two-pass register-resident transforms,
// n3 = r1 * r2), re-organised around what the ncu capture of those kernels showed (profiles/r01c: 21 % of the warp
// slots, 5-11 long-scoreboard stalls per issue, every phase -- zero-fill, index loads, gather, two passes -- ended by a
// CTA-wide barrier with all warps in the same phase):
//   * a work item is (cw columns, one band), owned by ONE warp; its two passes meet in a warp-private shared-memory
//     buffer with __syncwarp only, so the 16 warps of an SM drift apart and one warp's global-load latency is covered
//     by the others' butterflies.  Warps walk over the items of the whole band group (persistent grid);
//   * there is no zero-fill, no staging of the sphere and no index indirection through shared memory: the first pass
//     of the inverse transform takes its radix-r1 inputs straight from psi through a table of plane-wave indices laid
//     out in the order the lanes read it (-1 = outside the sphere: the input is zero and is not loaded), and the last
//     pass of the forward transform holds the r1 outputs of a column in registers and applies the recurrence epilogue
//     to those that are inside the sphere.  Every global load of a pass is independent of the others (up to 16 + 16
//     in flight per thread).
#include <type_traits>

#include "fft_reg.cuh"
#include "launch.h"

namespace pwh {

namespace {

constexpr int ZW = 8;   // warps per CTA; two CTAs per SM
#ifndef PWH_Z_GATHER_BATCH
#define PWH_Z_GATHER_BATCH 3
#endif
constexpr int ZGB = PWH_Z_GATHER_BATCH;   // entries of the gather epilogue whose loads are issued together

template <int R>
using RC = std::integral_constant<int, R>;

// the pruned instantiation of a radix-R strided-role pass: a cutoff sphere in a box of twice its diameter touches just over
// half of an axis, i.e. R/2 + 1 of the R rows q r2 + sub
__host__ __device__ constexpr int pruned_len(int R) { return R >= 4 ? R / 2 + 1 : R; }
// columns per work item for a contiguous-role radix r2 (the rule of pwh_ham_setup), and log2 of a power of two
__host__ __device__ constexpr int cw_of(int r2) { return r2 >= 6 ? 4 : (r2 >= 4 ? 8 : (r2 >= 2 ? 16 : 32)); }
__host__ __device__ constexpr int log2_of(int v) { return v <= 1 ? 0 : 1 + log2_of(v / 2); }

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

// the R plane-wave indices of work-item element i = sub*cw + c (R padded to a multiple of 4): int4 number j of element i
// sits at tab4[j * nelem + i], so one load instruction of a warp reads 512 contiguous bytes
template <int R>
__device__ __forceinline__ void load_idx(const int4* __restrict__ tab4, int nelem, int i, int* idx) {
  constexpr int R4 = (R + 3) / 4;   // R = number of table entries per element (the L of a pruned transform)
  const int4* r4 = tab4 + i;
#pragma unroll
  for (int j = 0; j < R4; ++j) {
    const int4 t = __ldg(r4 + (int64_t)j * nelem);
    if (4 * j + 0 < R) idx[4 * j + 0] = t.x;
    if (4 * j + 1 < R) idx[4 * j + 1] = t.y;
    if (4 * j + 2 < R) idx[4 * j + 2] = t.z;
    if (4 * j + 3 < R) idx[4 * j + 3] = t.w;
  }
}

// pass 1 of kz_scatter_zinv for one work item: radix R over the z-rows q r2 + sub of which only q < L can be inside the sphere
template <int R, int L>
__device__ __forceinline__ void scatter_pass1(const int4* __restrict__ tab4, const c128* __restrict__ src,
                                              c128* __restrict__ dst, c128* __restrict__ buf, const c128* __restrict__ tw,
                                              int64_t pstride, int r2, int cw, int lcw, int zs, int lane) {
  for (int i = lane; i < r2 * cw; i += 32) {
    const int sub = i >> lcw, c = i & (cw - 1);
    int idx[L];
    load_idx<L>(tab4, r2 * cw, i, idx);
    c128 v[R];
#pragma unroll
    for (int q = 0; q < L; ++q) v[q] = idx[q] >= 0 ? src[idx[q]] : cmake(0.0, 0.0);
    DftPrunedIn<R, +1, L>::run(v);
    if (r2 == 1) {
#pragma unroll
      for (int q = 0; q < R; ++q) dst[(int64_t)q * pstride + c] = v[q];
    } else {
      c128* b = buf + c * zs + sub;
      b[0] = v[0];
#pragma unroll
      for (int q = 1; q < R; ++q) b[q * (r2 + 1)] = cmul(v[q], tw[sub * q]);
    }
  }
}

// pass 2 of kz_zfwd_gather for one work item: radix R over positions q r2 + sub, outputs q < L, recurrence epilogue
template <int R, int L, int GB>
__device__ __forceinline__ void gather_pass2(const int4* __restrict__ tab4, const c128* __restrict__ src,
                                             const c128* __restrict__ buf, int64_t pstride, int r2, int cw, int lcw, int zs,
                                             int lane, const c128* yb, const c128* pb, c128* ob,
                                             const double* __restrict__ kin, double alpha, double cshift, double beta) {
  for (int i = lane; i < r2 * cw; i += 32) {
    const int sub = i >> lcw, c = i & (cw - 1);
    int idx[L];
    load_idx<L>(tab4, r2 * cw, i, idx);
    c128 v[R];
    if (r2 == 1) {
#pragma unroll
      for (int q = 0; q < R; ++q) v[q] = src[(int64_t)q * pstride + c];
    } else {
      const c128* b = buf + c * zs + sub;
#pragma unroll
      for (int q = 0; q < R; ++q) v[q] = b[q * (r2 + 1)];
    }
    Dft<R, -1>::run(v);
    // `out` may be the buffer of y or y_prev, so the compiler cannot move the loads of one entry above the store of the one
    // before: entries are handled GB at a time, all loads of a batch first (a thread only ever reads the entries it writes).
    // GB = 3 in the kernels specialised for one factorisation (what their 128 registers hold), 1 in the generic kernel.
    if constexpr (GB <= 1) {
#pragma unroll
      for (int q = 0; q < L; ++q) {
        const int g = idx[q];
        if (g < 0) continue;
        const c128 yv = yb[g];
        const double k = kin[g] - cshift;
        c128 r = cmake(alpha * fma(k, yv.x, v[q].x), alpha * fma(k, yv.y, v[q].y));
        if (pb) {
          const c128 pv = pb[g];
          r.x = fma(-beta, pv.x, r.x);
          r.y = fma(-beta, pv.y, r.y);
        }
        ob[g] = r;
      }
    } else {
#pragma unroll
      for (int q0 = 0; q0 < L; q0 += GB) {
        c128 yv[GB], pv[GB];
        double kk[GB];
#pragma unroll
        for (int t = 0; t < GB; ++t) {
          const int g = q0 + t < L ? idx[q0 + t < L ? q0 + t : 0] : -1;
          if (g < 0) continue;
          yv[t] = yb[g];
          kk[t] = kin[g];
          if (pb) pv[t] = pb[g];
        }
#pragma unroll
        for (int t = 0; t < GB; ++t) {
          if (q0 + t >= L) continue;
          const int q = q0 + t < L ? q0 + t : 0;
          const int g = idx[q];
          if (g < 0) continue;
          const double k = kk[t] - cshift;
          c128 r = cmake(alpha * fma(k, yv[t].x, v[q].x), alpha * fma(k, yv[t].y, v[q].y));
          if (pb) {
            r.x = fma(-beta, pv[t].x, r.x);
            r.y = fma(-beta, pv[t].y, r.y);
          }
          ob[g] = r;
        }
      }
    }
  }
}

// PR: the pruned instantiation of pass 1 (P.lq == pruned_len(r1)).  R1C x R2C: the factorisation of n3 as compile-time
// constants for the box sides of the bench configs (0 = taken from the plan at run time, every radix instantiated).  One
// kernel per choice keeps each kernel's code small: with both pass-1 bodies of all twelve radices in one kernel the scatter
// ran 15 % slower (profiles/r02d).
template <int R1C, int R2C, bool PR>
__global__ void __launch_bounds__(ZW * 32, 2) kz_scatter_zinv(const ZPlan P, const c128* __restrict__ psi, int64_t ldpsi,
                                                              c128* __restrict__ colbuf, int nb) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128* tw = reinterpret_cast<c128*>(smem_raw);                       // [n3]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  c128* buf = tw + P.n3 + warp * (P.cw * P.zs);                       // [cw][zs], warp-private
  for (int i = tid; i < P.n3; i += ZW * 32) tw[i] = P.tw[i];
  __syncthreads();
  const int r1 = R1C > 0 ? R1C : P.r1, r2 = R2C > 0 ? R2C : P.r2;
  const int cw = R2C > 0 ? cw_of(R2C) : P.cw, lcw = R2C > 0 ? log2_of(cw_of(R2C)) : P.log2cw, zs = P.zs, lqp = P.lqp;
  const int64_t pstride = P.ncols_pad;
  const int nitems = P.nq * nb;
  for (int item = blockIdx.x * ZW + warp; item < nitems; item += gridDim.x * ZW) {
    const int quad = item % P.nq, band = item / P.nq;
    const c128* __restrict__ src = psi + (int64_t)band * ldpsi;
    c128* __restrict__ dst = colbuf + (int64_t)band * P.n3 * pstride + quad * cw;
    const int4* __restrict__ tab4 = reinterpret_cast<const int4*>(P.ztab + (int64_t)quad * (r2 * cw * lqp));
    // pass 1, strided role: radix r1 over the z-ROWS zl = q r2 + sub counted from the lowest touched z (a shift of the
    // spectral index is a phase per z-plane in real space, which the forward transform of kz_zfwd_gather takes out again):
    // only q < L = P.lq can be inside the sphere; inputs gathered from the sphere
    auto pass1 = [&](auto rc) {
      constexpr int R = decltype(rc)::value;
      scatter_pass1<R, PR ? pruned_len(R) : R>(tab4, src, dst, buf, tw, pstride, r2, cw, lcw, zs, lane);
    };
    if constexpr (R1C > 0) pass1(RC<R1C>()); else with_radix<true>(r1, pass1);
    if (r2 == 1) continue;
    __syncwarp();
    // pass 2, contiguous role: radix r2 over positions sub r2 + q; output z-slot sub r2 + q, plane-major
    auto pass2 = [&](auto rc) {
      constexpr int R = decltype(rc)::value;
      for (int i = lane; i < r1 * cw; i += 32) {
        const int sub = i >> lcw, c = i & (cw - 1);
        const c128* b = buf + c * zs + sub * (R + 1);
        c128 v[R];
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = b[q];
        Dft<R, +1>::run(v);
        c128* d = dst + (int64_t)(sub * R) * pstride + c;
#pragma unroll
        for (int q = 0; q < R; ++q) d[(int64_t)q * pstride] = v[q];
      }
    };
    if constexpr (R2C > 0) pass2(RC<R2C>()); else with_radix<false>(r2, pass2);
    __syncwarp();
  }
}

// `out` may alias `y` or `yprev`: entry g of the three is read and written by the same thread, in that order.
template <int R1C, int R2C, bool PR>
__global__ void __launch_bounds__(ZW * 32, 2) kz_zfwd_gather(const ZPlan P, const c128* __restrict__ colbuf,
                                                             const c128* y, int64_t ldy,
                                                             const c128* yprev, int64_t ldprev,
                                                             c128* out, int64_t ldout, double alpha,
                                                             double cshift, double beta, int nb) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128* tw = reinterpret_cast<c128*>(smem_raw);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  c128* buf = tw + P.n3 + warp * (P.cw * P.zs);
  for (int i = tid; i < P.n3; i += ZW * 32) tw[i] = P.tw[i];
  __syncthreads();
  const int r1 = R1C > 0 ? R1C : P.r1, r2 = R2C > 0 ? R2C : P.r2;
  const int cw = R2C > 0 ? cw_of(R2C) : P.cw, lcw = R2C > 0 ? log2_of(cw_of(R2C)) : P.log2cw, zs = P.zs, lqp = P.lqp;
  const int64_t pstride = P.ncols_pad;
  const double* __restrict__ kin = P.kin;
  const int nitems = P.nq * nb;
  for (int item = blockIdx.x * ZW + warp; item < nitems; item += gridDim.x * ZW) {
    const int quad = item % P.nq, band = item / P.nq;
    const c128* __restrict__ src = colbuf + (int64_t)band * P.n3 * pstride + quad * cw;
    const int4* __restrict__ tab4 = reinterpret_cast<const int4*>(P.ztab + (int64_t)quad * (r2 * cw * lqp));
    const c128* yb = y + (int64_t)band * ldy;
    const c128* pb = (beta != 0.0) ? yprev + (int64_t)band * ldprev : nullptr;
    c128* ob = out + (int64_t)band * ldout;
    // the epilogue's operands y[g], y_prev[g] come from HBM: start them towards L2 now, the transforms run meanwhile
    for (int i = lane; i < r2 * cw * (lqp / 4); i += 32) {
      const int4 t = __ldg(tab4 + i);
      const int gi[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (gi[k] >= 0) {
          asm volatile("prefetch.global.L2 [%0];\n" ::"l"(yb + gi[k]));
          if (pb) asm volatile("prefetch.global.L2 [%0];\n" ::"l"(pb + gi[k]));
        }
    }
    if (r2 > 1) {
      // pass 1, contiguous role: radix r2 over z-slots sub r2 + q, twiddle w^-(sub q)
      auto pass1 = [&](auto rc) {
        constexpr int R = decltype(rc)::value;
        for (int i = lane; i < r1 * cw; i += 32) {
          const int sub = i >> lcw, c = i & (cw - 1);
          const c128* s = src + (int64_t)(sub * R) * pstride + c;
          c128 v[R];
#pragma unroll
          for (int q = 0; q < R; ++q) v[q] = s[(int64_t)q * pstride];
          Dft<R, -1>::run(v);
          c128* b = buf + c * zs + sub * (R + 1);
          b[0] = v[0];
#pragma unroll
          for (int q = 1; q < R; ++q) b[q] = cmulc(v[q], tw[sub * q]);
        }
      };
      if constexpr (R2C > 0) pass1(RC<R2C>()); else with_radix<false>(r2, pass1);
      __syncwarp();
    }
    // pass 2, strided role: radix r1 over positions q r2 + sub; output = w_loc at z-row zl = q r2 + sub (q < L: the others
    // are outside the sphere, never used, and their butterflies are dropped); recurrence epilogue
    auto pass2 = [&](auto rc) {
      constexpr int R = decltype(rc)::value;
      gather_pass2<R, PR ? pruned_len(R) : R, (R1C > 0 ? ZGB : 1)>(tab4, src, buf, pstride, r2, cw, lcw, zs, lane, yb, pb, ob, kin, alpha, cshift, beta);
    };
    if constexpr (R1C > 0) pass2(RC<R1C>()); else with_radix<true>(r1, pass2);
    __syncwarp();
  }
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------------
int zw_pruned_len(int r) { return pruned_len(r); }

size_t zw_smem(const ZPlan& P) { return sizeof(c128) * ((size_t)P.n3 + (size_t)ZW * P.cw * P.zs); }

// the instantiation for a plan: the bench configs' factorisations of n3 as compile-time constants, anything else generic
template <class F>
static void zw_dispatch(const ZPlan& P, F&& f) {
  const bool pr = P.lq < P.r1;
  auto go = [&](auto r1c, auto r2c) {
    if (pr) f(r1c, r2c, std::true_type()); else f(r1c, r2c, std::false_type());
  };
  if (P.cw != cw_of(P.r2)) go(RC<0>(), RC<0>());
  else if (P.r1 == 16 && P.r2 == 8) go(RC<16>(), RC<8>());
  else if (P.r1 == 15 && P.r2 == 12) go(RC<15>(), RC<12>());
  else if (P.r1 == 12 && P.r2 == 8) go(RC<12>(), RC<8>());
  else if (P.r1 == 8 && P.r2 == 6) go(RC<8>(), RC<6>());
  else go(RC<0>(), RC<0>());
}

cudaError_t zw_kernels_init(const ZPlan& P) {
  cudaError_t e = cudaSuccess;
  zw_dispatch(P, [&](auto r1c, auto r2c, auto pr) {
    constexpr int A = decltype(r1c)::value, B = decltype(r2c)::value;
    constexpr bool PR = decltype(pr)::value;
    e = set_max_dyn_smem(reinterpret_cast<const void*>(&kz_scatter_zinv<A, B, PR>));
    if (e == cudaSuccess) e = set_max_dyn_smem(reinterpret_cast<const void*>(&kz_zfwd_gather<A, B, PR>));
  });
  return e;
}

static int zw_grid(const ZPlan& P, int nb) {
  const int64_t items = (int64_t)P.nq * nb;
  const int64_t ctas = (items + ZW - 1) / ZW;
  return (int)(ctas < 2 * 148 ? ctas : 2 * 148);     // persistent: two CTAs of 8 warps per SM
}

void launch_zw_scatter_zinv(const ZPlan& P, const c128* psi, int64_t ldpsi, c128* colbuf, int nb, cudaStream_t st) {
  ScopedLaunch sl(ST_SCATTER_ZINV, st);
  zw_dispatch(P, [&](auto r1c, auto r2c, auto pr) {
    kz_scatter_zinv<decltype(r1c)::value, decltype(r2c)::value, decltype(pr)::value>
        <<<zw_grid(P, nb), ZW * 32, zw_smem(P), st>>>(P, psi, ldpsi, colbuf, nb);
  });
}

void launch_zw_zfwd_gather(const ZPlan& P, const c128* colbuf, const c128* y, int64_t ldy, const c128* yprev,
                           int64_t ldprev, c128* out, int64_t ldout, double alpha, double cshift, double beta, int nb,
                           cudaStream_t st) {
  ScopedLaunch sl(ST_ZFWD_GATHER, st);
  zw_dispatch(P, [&](auto r1c, auto r2c, auto pr) {
    kz_zfwd_gather<decltype(r1c)::value, decltype(r2c)::value, decltype(pr)::value>
        <<<zw_grid(P, nb), ZW * 32, zw_smem(P), st>>>(P, colbuf, y, ldy, yprev, ldprev, out, ldout, alpha, cshift,
                                                      yprev ? beta : 0.0, nb);
  });
}

}  // namespace pwh
