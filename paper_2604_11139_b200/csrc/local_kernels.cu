// local_kernels.cu -- the local-potential part of H psi and the fused kinetic / recurrence epilogue.
//
//   w_loc = gather( FFT( V_loc(r) . iFFT( scatter(psi) ) ) )
//   out   = alpha * ((kin - c) . y + w_loc) - beta * y_prev
//
// Three kernels per group of bands, none of which ever materialises the n1*n2*n3 box:
//   k_scatter_zinv : sphere -> touched z-columns, inverse z transform, store plane-major  [band][z][column]
//   k_plane        : per (band, z-plane): load the disc of columns into shared memory, inverse y on the touched
//                    x-lines, then per batch of y-lines: inverse x, multiply by V_loc/F, forward x, keep the touched
//                    x-lines; forward y; store the disc back in place.  The full plane only ever exists in smem.
//   k_zfwd_gather  : forward z transform of the columns, gather the sphere, fused kinetic + three-term recurrence.
#include "fft.cuh"
#include "launch.h"

namespace pwh {

static constexpr int ZT = 256;  // threads of the z kernels
static constexpr int PT = 512;  // threads of the plane kernel

__device__ __forceinline__ void load_tw(c128* dst, const c128* src, int n, int tid, int nthr) {
  for (int i = tid; i < n; i += nthr) dst[i] = src[i];
}
// stage one AxisPlan from device memory into shared memory (the stage loop indexes it dynamically)
__device__ __forceinline__ void load_plan(AxisPlan* dst, const AxisPlan* src, int tid, int nthr) {
  constexpr int W = sizeof(AxisPlan) / sizeof(int);
  for (int i = tid; i < W; i += nthr) reinterpret_cast<int*>(dst)[i] = reinterpret_cast<const int*>(src)[i];
}

__global__ void __launch_bounds__(ZT) k_scatter_zinv(const LocalPlan P, const c128* __restrict__ psi, int64_t ldpsi,
                                                     c128* __restrict__ colbuf) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128* lines = reinterpret_cast<c128*>(smem_raw);
  c128* tw = lines + P.colgrp * P.zstride;
  __shared__ AxisPlan s_az;
  const int tid = threadIdx.x, grp = blockIdx.x, band = blockIdx.y;
  const int nline = P.colgrp * P.zstride;
  for (int i = tid; i < nline; i += ZT) lines[i] = cmake(0.0, 0.0);
  load_tw(tw, P.tw[2], P.ax[2].tw_len, tid, ZT);
  load_plan(&s_az, P.axp + 2, tid, ZT);
  __syncthreads();
  const c128* src = psi + (int64_t)band * ldpsi;
  const int e0 = P.grp_ptr[grp], e1 = P.grp_ptr[grp + 1];
  for (int e = e0 + tid; e < e1; e += ZT) lines[P.ent_off[e]] = src[P.ent_pw[e]];
  __syncthreads();
  fft_lines<+1>(lines, P.colgrp, P.div_colgrp, P.zstride, s_az, tw, tid, ZT);
  c128* dst = colbuf + (int64_t)band * P.n3 * P.ncols_pad + grp * P.colgrp;
  const int total = P.colgrp * P.n3;
  for (int i = tid; i < total; i += ZT) {
    uint32_t z, c;
    P.div_colgrp.divmod((uint32_t)i, z, c);
    dst[(int64_t)z * P.ncols_pad + c] = lines[c * P.zstride + z];
  }
}

// `out` may alias `y` or `yprev`: entry g of the three is read and written by the same thread, in that order.
__global__ void __launch_bounds__(ZT) k_zfwd_gather(const LocalPlan P, const c128* __restrict__ colbuf,
                                                    const c128* y, int64_t ldy,
                                                    const c128* yprev, int64_t ldprev,
                                                    c128* out, int64_t ldout, double alpha, double cshift,
                                                    double beta) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128* lines = reinterpret_cast<c128*>(smem_raw);
  c128* tw = lines + P.colgrp * P.zstride;
  __shared__ AxisPlan s_az;
  const int tid = threadIdx.x, grp = blockIdx.x, band = blockIdx.y;
  load_tw(tw, P.tw[2], P.ax[2].tw_len, tid, ZT);
  load_plan(&s_az, P.axp + 2, tid, ZT);
  const c128* src = colbuf + (int64_t)band * P.n3 * P.ncols_pad + grp * P.colgrp;
  const int total = P.colgrp * P.n3;
  for (int i = tid; i < total; i += ZT) {
    uint32_t z, c;
    P.div_colgrp.divmod((uint32_t)i, z, c);
    lines[c * P.zstride + z] = src[(int64_t)z * P.ncols_pad + c];
  }
  __syncthreads();
  fft_lines<-1>(lines, P.colgrp, P.div_colgrp, P.zstride, s_az, tw, tid, ZT);
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

__global__ void __launch_bounds__(PT) k_plane(const LocalPlan P, c128* __restrict__ colbuf) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128* half = reinterpret_cast<c128*>(smem_raw);      // [nxl][ystride]
  c128* work = half + P.nxl * P.ystride;               // [xbatch][xstride]
  c128* twx = work + P.xbatch * P.xstride;
  c128* twy = twx + P.ax[0].tw_len;
  __shared__ AxisPlan s_ax, s_ay;
  const int tid = threadIdx.x, pz = blockIdx.x, band = blockIdx.y;
  load_plan(&s_ax, P.axp + 0, tid, PT);
  load_plan(&s_ay, P.axp + 1, tid, PT);
  const int nhalf = P.nxl * P.ystride;
  for (int i = tid; i < nhalf; i += PT) half[i] = cmake(0.0, 0.0);
  load_tw(twx, P.tw[0], P.ax[0].tw_len, tid, PT);
  load_tw(twy, P.tw[1], P.ax[1].tw_len, tid, PT);
  __syncthreads();
  c128* plane = colbuf + ((int64_t)band * P.n3 + pz) * P.ncols_pad;
  for (int c = tid; c < P.ncols; c += PT) half[P.col_hp[c]] = plane[c];
  __syncthreads();
  fft_lines<+1>(half, P.nxl, P.div_nxl, P.ystride, s_ay, twy, tid, PT);
  const double* vplane = P.vperm + (int64_t)pz * P.n2 * P.n1;
  const int xb = P.xbatch;
  for (int y0 = 0; y0 < P.n2; y0 += xb) {
    // expand the touched x-lines of y-lines y0..y0+xb-1 into full-length lines (zero elsewhere)
    for (int i = tid; i < xb * P.n1; i += PT) {
      uint32_t x, yb;
      P.div_xbatch.divmod((uint32_t)i, x, yb);
      const int xl = P.xl_of_x[x];
      work[yb * P.xstride + x] = xl >= 0 ? half[xl * P.ystride + y0 + yb] : cmake(0.0, 0.0);
    }
    __syncthreads();
    fft_lines<+1>(work, xb, P.div_xbatch, P.xstride, s_ax, twx, tid, PT);
    for (int i = tid; i < xb * P.n1; i += PT) {
      uint32_t yb, px;
      P.div_n1.divmod((uint32_t)i, yb, px);
      const double v = vplane[(y0 + yb) * P.n1 + px];
      c128* p = work + yb * P.xstride + px;
      *p = cscale(v, *p);
    }
    __syncthreads();
    fft_lines<-1>(work, xb, P.div_xbatch, P.xstride, s_ax, twx, tid, PT);
    for (int i = tid; i < xb * P.nxl; i += PT) {
      uint32_t xl, yb;
      P.div_xbatch.divmod((uint32_t)i, xl, yb);
      half[xl * P.ystride + y0 + yb] = work[yb * P.xstride + P.x_of_xl[xl]];
    }
    __syncthreads();
  }
  fft_lines<-1>(half, P.nxl, P.div_nxl, P.ystride, s_ay, twy, tid, PT);
  for (int c = tid; c < P.ncols; c += PT) plane[c] = half[P.col_hp[c]];
}

// Density accumulation on the generic stage plan (Algorithm 3 step 10): one CTA per
// z position walks over the bands of the group in order: disc -> inverse y -> inverse x, acc[pz][py][px] += occ |u|^2 in
// digit-permuted positions (deterministic: one owner thread per point, bands in order); k_density_unpermute adds acc to
// the caller's array in natural order.
__global__ void __launch_bounds__(PT) k_density_plane(const LocalPlan P, const c128* __restrict__ colbuf, int nb,
                                                      const double* __restrict__ occ, double* __restrict__ acc) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128* half = reinterpret_cast<c128*>(smem_raw);
  c128* work = half + P.nxl * P.ystride;
  c128* twx = work + P.xbatch * P.xstride;
  c128* twy = twx + P.ax[0].tw_len;
  __shared__ AxisPlan s_ax, s_ay;
  const int tid = threadIdx.x, pz = blockIdx.x;
  load_plan(&s_ax, P.axp + 0, tid, PT);
  load_plan(&s_ay, P.axp + 1, tid, PT);
  load_tw(twx, P.tw[0], P.ax[0].tw_len, tid, PT);
  load_tw(twy, P.tw[1], P.ax[1].tw_len, tid, PT);
  const int nhalf = P.nxl * P.ystride;
  double* aplane = acc + (int64_t)pz * P.n2 * P.n1;
  const int xb = P.xbatch;
  for (int band = 0; band < nb; ++band) {
    const double f = occ[band];
    __syncthreads();
    for (int i = tid; i < nhalf; i += PT) half[i] = cmake(0.0, 0.0);
    __syncthreads();
    const c128* plane = colbuf + ((int64_t)band * P.n3 + pz) * P.ncols_pad;
    for (int c = tid; c < P.ncols; c += PT) half[P.col_hp[c]] = plane[c];
    __syncthreads();
    fft_lines<+1>(half, P.nxl, P.div_nxl, P.ystride, s_ay, twy, tid, PT);
    for (int y0 = 0; y0 < P.n2; y0 += xb) {
      for (int i = tid; i < xb * P.n1; i += PT) {
        uint32_t x, yb;
        P.div_xbatch.divmod((uint32_t)i, x, yb);
        const int xl = P.xl_of_x[x];
        work[yb * P.xstride + x] = xl >= 0 ? half[xl * P.ystride + y0 + yb] : cmake(0.0, 0.0);
      }
      __syncthreads();
      fft_lines<+1>(work, xb, P.div_xbatch, P.xstride, s_ax, twx, tid, PT);
      for (int i = tid; i < xb * P.n1; i += PT) {
        uint32_t yb, px;
        P.div_n1.divmod((uint32_t)i, yb, px);
        const c128 u = work[yb * P.xstride + px];
        double* a = aplane + (y0 + yb) * P.n1 + px;
        *a = fma(f, fma(u.x, u.x, u.y * u.y), *a);
      }
      __syncthreads();
    }
  }
}

// rho[natx[px] + n1 (naty[py] + n2 natz[pz])] += weight * acc[px + n1 (py + n2 pz)]   (inverse of k_permute_vloc, pwham.cu)
__global__ void k_density_unpermute(int n1, int n2, int n3, const double* __restrict__ acc, const int* __restrict__ natx,
                                    const int* __restrict__ naty, const int* __restrict__ natz, double weight,
                                    double* __restrict__ rho) {
  const int64_t total = (int64_t)n1 * n2 * n3;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int px = (int)(i % n1);
    const int py = (int)((i / n1) % n2);
    const int pz = (int)(i / ((int64_t)n1 * n2));
    double* r = rho + natx[px] + (int64_t)n1 * (naty[py] + (int64_t)n2 * natz[pz]);
    *r = fma(weight, acc[i], *r);
  }
}

size_t zkernel_smem(const LocalPlan& P) {
  return sizeof(c128) * ((size_t)P.colgrp * P.zstride + P.ax[2].tw_len);
}
size_t plane_smem(const LocalPlan& P) {
  return sizeof(c128) * ((size_t)P.nxl * P.ystride + (size_t)P.xbatch * P.xstride + P.ax[0].tw_len + P.ax[1].tw_len);
}

cudaError_t local_kernels_init(const LocalPlan& P) {
  cudaError_t e;
  e = set_max_dyn_smem(reinterpret_cast<const void*>(&k_scatter_zinv));
  if (e != cudaSuccess) return e;
  e = set_max_dyn_smem(reinterpret_cast<const void*>(&k_zfwd_gather));
  if (e != cudaSuccess) return e;
  e = set_max_dyn_smem(reinterpret_cast<const void*>(&k_plane));
  if (e != cudaSuccess) return e;
  return set_max_dyn_smem(reinterpret_cast<const void*>(&k_density_plane));
}

void launch_scatter_zinv(const LocalPlan& P, const c128* psi, int64_t ldpsi, c128* colbuf, int nb, cudaStream_t st) {
  dim3 grid(P.ngrp, nb);
  ScopedLaunch sl(ST_SCATTER_ZINV, st);
  k_scatter_zinv<<<grid, ZT, zkernel_smem(P), st>>>(P, psi, ldpsi, colbuf);
}

void launch_plane(const LocalPlan& P, c128* colbuf, int nb, cudaStream_t st) {
  dim3 grid(P.n3, nb);
  ScopedLaunch sl(ST_PLANE, st);
  k_plane<<<grid, PT, plane_smem(P), st>>>(P, colbuf);
}

void launch_density_plane(const LocalPlan& P, const c128* colbuf, int nb, const double* occ, double* acc, cudaStream_t st) {
  ScopedLaunch sl(ST_PLANE, st);
  k_density_plane<<<P.n3, PT, plane_smem(P), st>>>(P, colbuf, nb, occ, acc);
}

void launch_density_unpermute(const LocalPlan& P, const double* acc, const int* natx, const int* naty, const int* natz,
                              double weight, double* rho, cudaStream_t st) {
  ScopedLaunch sl(ST_AXPY, st);
  k_density_unpermute<<<148 * 4, 256, 0, st>>>(P.n1, P.n2, P.n3, acc, natx, naty, natz, weight, rho);
}

void launch_zfwd_gather(const LocalPlan& P, const c128* colbuf, const c128* y, int64_t ldy, const c128* yprev,
                        int64_t ldprev, c128* out, int64_t ldout, double alpha, double cshift, double beta, int nb,
                        cudaStream_t st) {
  dim3 grid(P.ngrp, nb);
  ScopedLaunch sl(ST_ZFWD_GATHER, st);
  k_zfwd_gather<<<grid, ZT, zkernel_smem(P), st>>>(P, colbuf, y, ldy, yprev, ldprev, out, ldout, alpha, cshift, beta);
}

}  // namespace pwh
