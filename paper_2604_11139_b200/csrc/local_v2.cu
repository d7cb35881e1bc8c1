// local_v2.cu -- size-specialised plane kernel of the local-potential part of H psi.
//
//   per (band, z-plane):  disc of touched columns -> inverse y on the touched x-lines -> inverse x -> V_loc(r)/F ->
//                         forward x (touched x-lines only) -> forward y -> disc
//
// Same arithmetic as kf_plane in local_fast.cu (two-pass register-resident transforms, n = r1 * r2, real-space data in
// "slot" order, V_loc stored once in the order the kernel reads it), re-organised around what the ncu capture of
// kf_plane showed (profiles/r01a_*): 59 % of its instructions were integer/address work of the generic radix dispatch,
// its code did not fit the instruction cache, and every pass ended in a CTA-wide barrier with 16 warps resident.
//   * the box sides and radices are template parameters: every shared-memory access is base + immediate offset;
//   * the disc is read from and written to global memory directly by the first / last y pass (per-row range tables,
//     no zero-fill and no staging pass): valid when every y-row of the disc is a contiguous run of x-lines and the
//     touched x-lines are contiguous modulo n1 (true for any cutoff sphere; checked in pwh_ham_setup, otherwise the
//     generic kernels are used);
//   * the x direction is warp-private: a warp owns NYB y-slots at a time and carries them through inverse x,
//     V_loc multiply and forward x in its own padded buffer with __syncwarp only, so a plane needs 4 CTA barriers;
//   * V_loc/F is stored as [z-slot][y-batch][q][lane item] so that the multiply reads it fully coalesced.
//   * the inter-pass twiddles of the x direction are applied on both sides of the contiguous-role pass, where a lane keeps
//     the same k1 for all its items: they live in registers, and the strided-role passes are plain radix-r1 transforms;
//   * no load or store is predicated: x-lines outside the sphere are read from a zero line and stored to a dump line of
//     the half-plane, rows outside the disc are read from a zero padding column and stored to a dump padding column
//     (16 predicates per radix-16 item had to be packed into a register and unpacked again).
#include <type_traits>

#include "fft_reg.cuh"
#include "launch.h"

namespace pwh {

namespace {

template <int N1_, int R1X_, int R2X_, int N2_, int R1Y_, int R2Y_, int NW_, int NYB_, int MINB_ = 1, int LQX_ = R1X_>
struct PC {
  static constexpr int N1 = N1_, R1X = R1X_, R2X = R2X_, N2 = N2_, R1Y = R1Y_, R2Y = R2Y_, NW = NW_, NYB = NYB_;
  static_assert(R1X * R2X == N1 && R1Y * R2Y == N2, "axis factorisation");
  static_assert(N2 % NYB == 0, "y batches");
  static constexpr int NT = NW * 32;
  static constexpr int MINB = MINB_;                 // CTAs per SM the register budget is capped for
  static constexpr int LQX = LQX_;                   // x-lines l = s + R2X q with q >= LQX are untouched: nxl <= LQX * R2X
  static constexpr int LQY = LQX_ * R1Y_ >= R1X_ * R1Y_ ? R1Y_ : (LQX_ < R1Y_ ? LQX_ : R1Y_);   // the same for the y-rows: nyl <= LQY * R2Y
  static constexpr int YS = N2 | 1;                  // odd line stride of the half-plane (elements)
  static constexpr int XP = R1X * (R2X + 1);         // padded length of one x-line in a warp buffer
  static constexpr int TWA_X = R2X * (R1X + 1), TWB_X = R1X * (R2X + 1);
  static constexpr int TWA_Y = R2Y * (R1Y + 1), TWB_Y = R1Y * (R2Y + 1);
  static constexpr int NBATCH = N2 / NYB;
  static size_t smem_bytes(int nxl) {
    return sizeof(c128) * ((size_t)(nxl + 2) * YS + (size_t)NW * NYB * XP + TWA_X + TWB_X + TWA_Y + TWB_Y) + sizeof(int2) * N2;
  }
};

__device__ __forceinline__ c128 czero() { return cmake(0.0, 0.0); }

template <class C>
__global__ void __launch_bounds__(C::NT, C::MINB) kv2_plane(const V2Plan P, c128* __restrict__ colbuf) {
  constexpr int N1 = C::N1, R1X = C::R1X, R2X = C::R2X, N2 = C::N2, R1Y = C::R1Y, R2Y = C::R2Y;
  constexpr int NT = C::NT, YS = C::YS, XP = C::XP, NYB = C::NYB, LQX = C::LQX, LQY = C::LQY;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int nxl = P.nxl;
  c128* half = reinterpret_cast<c128*>(smem_raw);            // [nxl + 2][YS]: line nxl stays zero (read for the
                                                             // untouched x-lines), line nxl + 1 takes the stores to them
  c128* tbuf = half + (nxl + 2) * YS;                        // [NW][NYB][XP]
  c128* twAx = tbuf + C::NW * NYB * XP;                      // [R2X][R1X+1]  w^(s k1)
  c128* twBx = twAx + C::TWA_X;                              // [R1X][R2X+1]  w^(s k1)
  c128* twAy = twBx + C::TWB_X;
  c128* twBy = twAy + C::TWA_Y;
  int2* yrow = reinterpret_cast<int2*>(twBy + C::TWB_Y);     // [N2]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // CTAs are dispatched in increasing blockIdx.y: walk the bands of the group from the LAST to the first.  The scatter kernel
  // wrote the column buffer first band first, so what the L2 still holds of a buffer larger than itself is the last bands;
  // this kernel leaves the first bands in L2, which is where the gather kernel starts.
  const int zslot = blockIdx.x, band = (int)gridDim.y - 1 - (int)blockIdx.y;

  for (int i = tid; i < C::TWA_X; i += NT) twAx[i] = P.twA[0][i];
  for (int i = tid; i < C::TWB_X; i += NT) twBx[i] = P.twB[0][i];
  for (int i = tid; i < C::TWA_Y; i += NT) twAy[i] = P.twA[1][i];
  for (int i = tid; i < C::TWB_Y; i += NT) twBy[i] = P.twB[1][i];
  for (int i = tid; i < N2; i += NT) yrow[i] = P.yrow[i];
  for (int i = tid; i < YS; i += NT) half[nxl * YS + i] = czero();
  __syncthreads();

  c128* __restrict__ plane = colbuf + ((int64_t)band * P.n3 + zslot) * P.ncols_pad;
  const int zcol = P.zcol;

  // ---- y1: inverse y, strided role (radix R1Y over the y-ROWS yl = q R2Y + s, counted from the lowest touched row: the
  //      same index shift as in the x direction, so only q < LQY can hold a row of the disc), input straight from the disc
  {
    const int nitems = R2Y * nxl;
    // the disc comes from L2 / HBM: the loads of a thread's next item are issued before its current item is transformed
    auto load_item = [&](int i, c128* dstv) {
      uint32_t s, l;
      P.div_nxl.divmod((uint32_t)i, s, l);
      const int2* yr = yrow + s;
#pragma unroll
      for (int q = 0; q < LQY; ++q) {
        const int2 row = yr[q * R2Y];
        const uint32_t d = l - (uint32_t)(row.y & 0xffff);
        dstv[q] = plane[d < (uint32_t)(row.y >> 16) ? row.x + (int)l : zcol];   // zcol: a padding column, always zero
      }
    };
    c128 nxt[LQY];
    if (tid < nitems) load_item(tid, nxt);
    for (int i = tid; i < nitems; i += NT) {
      uint32_t s, l;
      P.div_nxl.divmod((uint32_t)i, s, l);
      c128 v[R1Y];
#pragma unroll
      for (int q = 0; q < LQY; ++q) v[q] = nxt[q];
      if (i + NT < nitems) load_item(i + NT, nxt);
      DftPrunedIn<R1Y, +1, LQY>::run(v);
      const c128* tw = twAy + s * (R1Y + 1);
      c128* dst = half + l * YS + s;
      dst[0] = v[0];
#pragma unroll
      for (int q = 1; q < R1Y; ++q) dst[q * R2Y] = cmul(v[q], tw[q]);
    }
  }
  __syncthreads();
  // ---- y2: inverse y, contiguous role (radix R2Y over positions k1 R2Y + s); output in y-slot order
  {
    const int nitems = R1Y * nxl;
    for (int i = tid; i < nitems; i += NT) {
      uint32_t k1, l;
      P.div_nxl.divmod((uint32_t)i, k1, l);
      c128* p = half + l * YS + k1 * R2Y;
      c128 v[R2Y];
#pragma unroll
      for (int q = 0; q < R2Y; ++q) v[q] = p[q];
      Dft<R2Y, +1>::run(v);
#pragma unroll
      for (int q = 0; q < R2Y; ++q) p[q] = v[q];
    }
  }
  __syncthreads();

  // ---- x direction, warp-private: NYB y-slots at a time
  {
    c128* tw_ = tbuf + warp * (NYB * XP);
    const double* __restrict__ vz = P.vperm + (int64_t)zslot * ((int64_t)N1 * N2);
    constexpr int XG = 32 / R1X;               // y-slots pass (b) handles per round: lane = xg * R1X + xk1
    static_assert(NYB % XG == 0, "pass (b) rounds");
    const int xk1 = lane % R1X, xg = lane / R1X;
    c128 xtw[R2X];
#pragma unroll
    for (int q = 0; q < R2X; ++q) xtw[q] = twBx[xk1 * (R2X + 1) + q];
    for (int b = warp; b < C::NBATCH; b += C::NW) {
      const int y0 = b * NYB;
      // V_loc/F of this batch: requested from L2 now, consumed in pass (b) after the radix-R1X transforms of pass (a)
      const double* __restrict__ vb = vz + (int64_t)b * (R2X * R1X * NYB);
      double vreg[NYB / XG][R2X];
#ifndef PWH_V2_NO_PREFETCH
      if (lane < XG * R1X) {
#pragma unroll
        for (int r = 0; r < NYB / XG; ++r)
#pragma unroll
          for (int q = 0; q < R2X; ++q) vreg[r][q] = __ldg(vb + q * (R1X * NYB) + xk1 + R1X * (xg + r * XG));
      }
#endif
      // (a) strided role: radix R1X over the x-LINES l = q R2X + s, twiddle, into the warp buffer at k1 (R2X+1) + s.
      //     The transform runs over the line index l = (x - x0) mod N1 instead of x: the shift is the phase w^(-x0 r) in real
      //     space, which the forward transform of pass (c) takes out again around the real, pointwise V_loc multiply -- so
      //     the touched lines are the prefix l < nxl, only the first LQX inputs of a radix-R1X transform can be non-zero
      //     and nothing wraps.
      for (int i = lane; i < R2X * NYB; i += 32) {
        const int s = i % R2X, yb = i / R2X;
        const c128* src = half + y0 + yb;
        c128 v[R1X];
#pragma unroll
        for (int q = 0; q < LQX; ++q) {
          const int l = s + q * R2X;
          v[q] = src[(l < nxl ? l : nxl) * YS];
        }
        DftPrunedIn<R1X, +1, LQX>::run(v);
        c128* dst = tw_ + yb * XP + s;
#pragma unroll
        for (int q = 0; q < R1X; ++q) dst[q * (R2X + 1)] = v[q];
      }
      __syncwarp();
      // (b) contiguous role: twiddle w^(s k1), radix R2X inverse -> real space, multiply by V_loc/F, radix R2X forward,
      //     twiddle w^-(s k1).  A lane keeps the same k1 for all its items, so its R2X-1 twiddles live in registers and
      //     passes (a) and (c) are plain radix-R1X transforms.
      if (lane < XG * R1X) {
#pragma unroll
        for (int r = 0; r < NYB / XG; ++r) {
          const int yb = xg + r * XG;
          c128* t = tw_ + yb * XP + xk1 * (R2X + 1);
          c128 v[R2X];
          v[0] = t[0];
#pragma unroll
          for (int q = 1; q < R2X; ++q) v[q] = cmul(t[q], xtw[q]);
          Dft<R2X, +1>::run(v);
#pragma unroll
#ifdef PWH_V2_NO_PREFETCH
          for (int q = 0; q < R2X; ++q) vreg[r][q] = vb[q * (R1X * NYB) + xk1 + R1X * yb];
#pragma unroll
#endif
          for (int q = 0; q < R2X; ++q) v[q] = cscale(vreg[r][q], v[q]);
          Dft<R2X, -1>::run(v);
          t[0] = v[0];
#pragma unroll
          for (int q = 1; q < R2X; ++q) t[q] = cmulc(v[q], xtw[q]);
        }
      }
      __syncwarp();
      // (c) strided role: radix R1X forward over k1; only the outputs q < LQX can be touched lines (the others are never
      //     stored, so the compiler drops the butterflies that feed only them)
      for (int i = lane; i < R2X * NYB; i += 32) {
        const int s = i % R2X, yb = i / R2X;
        const c128* src = tw_ + yb * XP + s;
        c128 v[R1X];
#pragma unroll
        for (int q = 0; q < R1X; ++q) v[q] = src[q * (R2X + 1)];
        Dft<R1X, -1>::run(v);
        c128* dst = half + y0 + yb;
#pragma unroll
        for (int q = 0; q < LQX; ++q) {
          const int l = s + q * R2X;
          dst[(l < nxl ? l : nxl + 1) * YS] = v[q];
        }
      }
      __syncwarp();
    }
  }
  __syncthreads();

  // ---- y2': forward y, contiguous role (radix R2Y over k2 at positions k1 R2Y + k2), twiddle w^-(s k1)
  {
    const int nitems = R1Y * nxl;
    for (int i = tid; i < nitems; i += NT) {
      uint32_t k1, l;
      P.div_nxl.divmod((uint32_t)i, k1, l);
      c128* p = half + l * YS + k1 * R2Y;
      c128 v[R2Y];
#pragma unroll
      for (int q = 0; q < R2Y; ++q) v[q] = p[q];
      Dft<R2Y, -1>::run(v);
      const c128* tw = twBy + k1 * (R2Y + 1);
      p[0] = v[0];
#pragma unroll
      for (int q = 1; q < R2Y; ++q) p[q] = cmulc(v[q], tw[q]);
    }
  }
  __syncthreads();
  // ---- y1': forward y, strided role (radix R1Y over k1 at positions k1 R2Y + s); output y = q R2Y + s to the disc
  {
    const int nitems = R2Y * nxl;
    for (int i = tid; i < nitems; i += NT) {
      uint32_t s, l;
      P.div_nxl.divmod((uint32_t)i, s, l);
      const c128* src = half + l * YS + s;
      c128 v[R1Y];
#pragma unroll
      for (int q = 0; q < R1Y; ++q) v[q] = src[q * R2Y];
      Dft<R1Y, -1>::run(v);
      const int2* yr = yrow + s;
#pragma unroll
      for (int q = 0; q < LQY; ++q) {      // rows q >= LQY are outside the disc: never stored, their butterflies are dropped
        const int2 row = yr[q * R2Y];
        const uint32_t d = l - (uint32_t)(row.y & 0xffff);
        plane[d < (uint32_t)(row.y >> 16) ? row.x + (int)l : zcol + 1] = v[q];   // zcol + 1: padding column nobody reads
      }
    }
  }
}

// V_loc/F in the order kv2_plane reads it:
//   out[((zs * NBATCH + b) * R2X + q) * (R1X*NYB) + i],  i = k1 + R1X * yb
//     = v[x + n1 * (y + n2 * z)] / F   with  x = k1 + R1X q,  y = slot(b NYB + yb; R1Y, R2Y),  z = slot(zs; r1z, r2z),
//   slot(p; r1, r2) = p / r2 + r1 * (p % r2)
__global__ void kv2_perm_vloc(int n1, int n2, int n3, int r1x, int r2x, int r1y, int r2y, int r1z, int r2z, int nyb,
                              const double* __restrict__ v, double inv_f, double* __restrict__ out) {
  const int64_t total = (int64_t)n1 * n2 * n3;
  const int per_q = r1x * nyb, per_b = r2x * per_q, nbatch = n2 / nyb;
  for (int64_t o = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; o < total; o += (int64_t)gridDim.x * blockDim.x) {
    const int i = (int)(o % per_q);
    const int q = (int)((o / per_q) % r2x);
    const int b = (int)((o / per_b) % nbatch);
    const int zs = (int)(o / ((int64_t)per_b * nbatch));
    const int k1 = i % r1x, yb = i / r1x;
    const int x = k1 + r1x * q;
    const int p = b * nyb + yb;
    const int y = p / r2y + r1y * (p % r2y);
    const int z = zs / r2z + r1z * (zs % r2z);
    out[o] = v[x + (int64_t)n1 * (y + (int64_t)n2 * z)] * inv_f;
  }
}

template <class C>
cudaError_t v2_init(int nxl) {
  return set_max_dyn_smem(reinterpret_cast<const void*>(&kv2_plane<C>));
}
template <class C>
void v2_launch(const V2Plan& P, c128* colbuf, int nb, cudaStream_t st) {
  dim3 grid(P.n3, nb);
  kv2_plane<C><<<grid, C::NT, C::smem_bytes(P.nxl), st>>>(P, colbuf);
}

// the specialisations: box side -> (r1, r2) and the (warps, y-slots per warp batch) variants tried in this order
using C48 = PC<48, 8, 6, 48, 8, 6, 8, 16>;
using C48b = PC<48, 8, 6, 48, 8, 6, 4, 8, 4>;     // small plane: 4 CTAs of 4 warps per SM instead of one of 8
using C96a = PC<96, 12, 8, 96, 12, 8, 16, 4>;
using C96b = PC<96, 12, 8, 96, 12, 8, 8, 4>;
using C96d = PC<96, 12, 8, 96, 12, 8, 4, 4, 2>;    // two CTAs of 4 warps per SM (113 KB each): independent phases overlap
using C96c = PC<96, 12, 8, 96, 12, 8, 12, 4>;    // 24 x batches = 2 per warp, 170 registers per thread
using C120a = PC<120, 15, 8, 120, 15, 8, 10, 4>;
using C120b = PC<120, 15, 8, 120, 15, 8, 8, 4>;
using C128a = PC<128, 16, 8, 128, 16, 8, 16, 4>;
using C128b = PC<128, 16, 8, 128, 16, 8, 8, 4>;
// the same shapes for spheres that touch at most LQX * R2X x-lines (a cutoff sphere in a box of twice its diameter touches
// about half of them): the strided-role x passes skip the lines that cannot be touched
using C48p = PC<48, 8, 6, 48, 8, 6, 4, 8, 4, 5>;        // nxl <= 30 (cfg 2: 25)
using C96p = PC<96, 12, 8, 96, 12, 8, 4, 4, 2, 7>;      // nxl <= 56 (cfg 3: 49)
using C120p = PC<120, 15, 8, 120, 15, 8, 8, 4, 1, 8>;   // nxl <= 64 (cfg 5: 64)
using C128p = PC<128, 16, 8, 128, 16, 8, 8, 4, 1, 9>;   // nxl <= 72 (cfg 4: 65)

template <class F>
bool v2_dispatch(int variant, F&& f) {
  switch (variant) {
    case 1: f(C48()); return true;
    case 2: f(C96a()); return true;
    case 3: f(C96b()); return true;
    case 4: f(C120a()); return true;
    case 5: f(C120b()); return true;
    case 6: f(C128a()); return true;
    case 7: f(C128b()); return true;
    case 8: f(C96c()); return true;
    case 9: f(C48b()); return true;
    case 10: f(C96d()); return true;
    case 11: f(C48p()); return true;
    case 12: f(C96p()); return true;
    case 13: f(C120p()); return true;
    case 14: f(C128p()); return true;
    default: return false;
  }
}

}  // namespace

// Picks the specialisation for an n1 x n2 plane with nxl touched x-lines and a disc spanning nyl y-rows that fits `smem_max` bytes of shared memory;
// fills the radices, NYB and the variant id of the plan.  Returns false when no specialisation applies.
bool v2_select(V2Plan& P, int n1, int n2, int nxl, int nyl, size_t smem_max, bool no_prune) {
  if (n1 != n2) return false;
  int order[5] = {0, 0, 0, 0, 0}, norder = 0;
  if (n1 == 48) { order[norder++] = 11; order[norder++] = 9; order[norder++] = 1; }
  else if (n1 == 96) { order[norder++] = 12; order[norder++] = 10; order[norder++] = 8; order[norder++] = 2; }
  else if (n1 == 120) { order[norder++] = 13; order[norder++] = 5; order[norder++] = 4; }   // 8 warps measured faster than 10 (12.4 vs 12.9 ms, cfg 5)
  else if (n1 == 128) { order[norder++] = 14; order[norder++] = 6; order[norder++] = 7; }
  if (no_prune && norder > 0) { for (int i = 1; i < norder; ++i) order[i - 1] = order[i]; --norder; }
  for (int oi = 0; oi < norder; ++oi) {
    const int var = order[oi];
    bool ok = false;
    v2_dispatch(var, [&](auto c) {
      using C = decltype(c);
      if (C::smem_bytes(nxl) <= smem_max && nxl <= C::LQX * C::R2X && nyl <= C::LQY * C::R2Y) {
        ok = true;
        P.variant = var;
        P.r1[0] = C::R1X; P.r2[0] = C::R2X; P.r1[1] = C::R1Y; P.r2[1] = C::R2Y;
        P.nyb = C::NYB;
      }
    });
    if (ok) return true;
  }
  return false;
}

cudaError_t v2_kernels_init(const V2Plan& P) {
  cudaError_t e = cudaErrorInvalidValue;
  v2_dispatch(P.variant, [&](auto c) { e = v2_init<decltype(c)>(P.nxl); });
  return e;
}

void launch_v2_perm_vloc(const V2Plan& P, int r1z, int r2z, const double* vloc, double* out, cudaStream_t st) {
  const double inv_f = 1.0 / ((double)P.n1 * P.n2 * P.n3);
  kv2_perm_vloc<<<148 * 4, 256, 0, st>>>(P.n1, P.n2, P.n3, P.r1[0], P.r2[0], P.r1[1], P.r2[1], r1z, r2z, P.nyb, vloc,
                                         inv_f, out);
}

void launch_v2_plane(const V2Plan& P, c128* colbuf, int nb, cudaStream_t st) {
  ScopedLaunch sl(ST_PLANE, st);
  v2_dispatch(P.variant, [&](auto c) { v2_launch<decltype(c)>(P, colbuf, nb, st); });
}

}  // namespace pwh
