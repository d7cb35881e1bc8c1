// common.cuh -- shared declarations of the libpwham kernels (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pwh {

typedef double2 c128;  // {re, im}

__host__ __device__ inline c128 cmake(double x, double y) { c128 r; r.x = x; r.y = y; return r; }
__device__ __forceinline__ c128 cadd(c128 a, c128 b) { return cmake(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ c128 csub(c128 a, c128 b) { return cmake(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ c128 cmul(c128 a, c128 b) {
  return cmake(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}
// a * conj(b)
__device__ __forceinline__ c128 cmulc(c128 a, c128 b) {
  return cmake(fma(a.x, b.x, a.y * b.y), fma(a.y, b.x, -a.x * b.y));
}
__device__ __forceinline__ c128 cscale(double s, c128 a) { return cmake(s * a.x, s * a.y); }

// q = n / d for n*d < 2^32: one IMAD.HI.  (A 64-bit multiplier with `(uint64_t)n * mul >> 32` is miscompiled by
// ptxas 12.9 -O2/-O3 for sm_100a inside the strided stage loops -- observed on the B200, results depended on the
// optimisation level -- so the multiplier is kept to 32 bits and d == 1 is a special case.)
struct FastDiv {
  uint32_t mul;
  uint32_t d;
  __device__ __forceinline__ uint32_t div(uint32_t n) const { return d == 1 ? n : __umulhi(n, mul); }
  __device__ __forceinline__ void divmod(uint32_t n, uint32_t& q, uint32_t& r) const {
    q = div(n);
    r = n - q * d;
  }
};
inline FastDiv make_fastdiv(uint32_t d) {
  FastDiv f;
  f.d = d;
  f.mul = (d <= 1) ? 0u : (uint32_t)(((1ull << 32) + d - 1) / d);
  return f;
}

// One axis of the in-place mixed-radix FFT.  Stage s works on blocks of size radix[s]*m[s]:
//   decimation in frequency (natural -> digit-permuted):  stages 0..ns-1, butterfly then twiddle;
//   decimation in time      (digit-permuted -> natural):  stages ns-1..0, twiddle then butterfly.
// tw_off[s] indexes the per-axis twiddle table: tw[tw_off[s] + (k-1)*m + n2] = exp(+2 pi i n2 k / (radix*m)).
#define PWH_MAX_STAGES 8
struct AxisPlan {
  int n;
  int nstages;
  int radix[PWH_MAX_STAGES];
  int m[PWH_MAX_STAGES];
  int tw_off[PWH_MAX_STAGES];
  int tw_len;           // entries in the twiddle table
  FastDiv div_m[PWH_MAX_STAGES];
};

// Everything the local-potential kernels need (passed by value as a kernel parameter).
struct LocalPlan {
  AxisPlan ax[3];            // x, y, z (host copy; kernels only touch it with constant indices)
  const AxisPlan* axp;       // the same three plans in device memory (kernels stage them into shared memory)
  const c128* tw[3];         // device twiddle tables
  int n1, n2, n3;
  int ncols;                 // z-columns touched by the sphere
  int ncols_pad;             // padded to a multiple of the column-group size
  int nxl;                   // x-lines touched
  int colgrp;                // columns per CTA in the z kernels
  int ngrp;                  // number of column groups
  int zstride;               // smem line stride (elements) of a z-column, odd
  int ystride;               // smem line stride of an x-line (length n2), odd
  int xstride;               // smem line stride of a y-line (length n1), odd
  int xbatch;                // y-lines per x-pass batch in the plane kernel
  const int* grp_ptr;        // [ngrp+1] CSR over sphere entries sorted by column group
  const int* ent_pw;         // [npw] plane-wave index of each entry
  const int* ent_off;        // [npw] local smem offset: lcol*zstride + z
  const int* col_hp;         // [ncols_pad] half-plane offset xl*ystride + y of each column (-1 for padding)
  const short* xl_of_x;      // [n1] x-line index of each wrapped x, -1 if untouched
  const short* x_of_xl;      // [nxl] wrapped x of each x-line
  const double* vperm;       // [n3][n2][n1] V_loc/F in digit-permuted positions
  const double* kin;         // [npw]
  FastDiv div_colgrp, div_nxl, div_xbatch, div_n1, div_ncols_pad;
};

// Plan of the register-resident two-pass local kernels (local_fast.cu): every axis n = r1 * r2.
struct FastPlan {
  int n1, n2, n3;
  int r1[3], r2[3];          // x, y, z
  const c128* tw[3];         // tw[ax][t] = exp(+2 pi i t / n_ax), t < n_ax
  int ncols, ncols_pad, nxl;
  int colgrp, ngrp;          // columns per CTA of the z kernels, number of column groups
  int zstride, ystride;      // odd shared-memory line strides (elements)
  int yb;                    // y-slots per x batch in the plane kernel
  int tsize;                 // elements of the x-batch buffer T (0 when the x transform is a single pass)
  int plane_threads;         // block size of the plane kernel
  const int* grp_ptr;        // [ngrp+1] CSR over sphere entries sorted by column group
  const int* ent_pw;         // [npw] plane-wave index of each entry
  const int* ent_off;        // [npw] lcol*zstride + wrapped z
  const int* col_hp;         // [ncols_pad] xl*ystride + wrapped y of each column
  const short* xl_of_x;      // [n1] x-line index of each wrapped x, -1 if untouched
  const double* vslot;       // [n3 slots][n1 slots][n2 slots] V_loc/F, y-slot fastest
  const double* kin;         // [npw]
  FastDiv div_colgrp, div_nxl, div_yb;
};

// Plan of the size-specialised plane kernel (local_v2.cu).
struct V2Plan {
  int n1, n2, n3;
  int ncols_pad, nxl;
  int x0;                    // wrapped x of x-line 0: x-line of x is (x - x0) mod n1, touched iff < nxl
  int zcol;                  // first padding column (>= ncols): zero on input; zcol + 1 takes the stores outside the disc
  int variant;               // which template instantiation
  int r1[2], r2[2], nyb;     // x, y radices and y-slots per warp batch of that instantiation
  const int2* yrow;          // [n2] per y-row yl = (y - y0) mod n2, y0 the lowest touched row: .x = first column - xlmin,
                             // .y = xlmin | (count << 16)
  const c128* twA[2];        // x, y: [r2][r1+1]  exp(+2 pi i s k1 / n) at s (r1+1) + k1
  const c128* twB[2];        // x, y: [r1][r2+1]  the same value at k1 (r2+1) + s
  const double* vperm;       // V_loc/F in kernel read order (kv2_perm_vloc)
  FastDiv div_nxl;
};

// Plan of the warp-private z kernels (local_z.cu): n3 = r1 * r2, a work item is (cw columns, one band).
struct ZPlan {
  int n3, r1, r2;
  int lq;                    // z-rows zl = q r2 + sub with q >= lq are outside the sphere (lq = r1: no pruning)
  int lqp;                   // lq rounded up to a multiple of 4 (row length of ztab)
  int cw, log2cw;            // columns per work item (power of two: 4 when r2 >= 6), its log2
  int nq;                    // work items per band = ncols_pad / cw
  int ncols_pad;
  int zs;                    // elements per column of a warp buffer; position of z = q r2 + s is q (r2 + 1) + s
  const int* ztab;           // [nq][lqp/4][r2*cw][4]: plane-wave index of column quad*cw + c at z-row zl = q r2 + sub, counted
                             // from the lowest touched z: zl = (z - z0) mod n3 (element sub*cw + c, q = 4 j + k), -1 outside
                             // the sphere
  const c128* tw;            // tw[t] = exp(+2 pi i t / n3)
  const double* kin;         // [npw]
};

}  // namespace pwh
