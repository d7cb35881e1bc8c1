// zgemm.cu -- complex-FP64 GEMMs on the FP64 tensor pipe (DMMA, mma.sync.m8n8k4.f64) for the dense contractions
// of the path:
//   "CN":  C = A^H B   with K = npw   -> projector coefficients <p_i|psi_b> and the
//                                        Rayleigh-Ritz Gram product Psi^H (H Psi), split over K
//   "NN":  C += alpha A B with K = nproj -> P . (D . P^H psi) accumulated onto the recurrence term
// tcgen05 has no f64 kind, so FP64 contractions on sm_100a are warp-level DMMA with register accumulators
// (measured on B200: DMMA.8x8x4 peak 37.1 TFLOP/s == DFMA peak).  Two kernels live here:
//   k_zgemm3m_tma  (default)  3M complex product, operand slabs by TMA with 128-byte swizzle, mbarrier hand-over
//   k_zgemm3m      (fallback) 3M, slabs by cp.async into padded layouts, same mbarrier hand-over; used when the driver
//                             does not export cuTensorMapEncodeTiled or refuses an operand (PWH_ZGEMM_NO_TMA=1 forces it)
// Every shared-memory layout is chosen so that the 16-byte fragment loads of a quarter-warp are conflict-free.
#include <cuda.h>

#include <algorithm>
#include <atomic>
#include <cstdlib>
#include <cstring>

#include "launch.h"

namespace pwh {

namespace {

constexpr int BM = 128, BN = 64;                       // CTA tile (complex elements)

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}
// mbarrier helpers (shared-memory barriers that replace the CTA-wide __syncthreads() of the k loop)
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared.b64 [%0], %1;\n" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.shared.b64 st, [%0];\n}\n" ::"r"(bar) : "memory");
}
// arrive on `bar` once all cp.async issued so far by this thread have landed (does not change the pending count)
__device__ __forceinline__ void cp_async_arrive(uint32_t bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared.b64 [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n.reg .pred p;\nWAIT_%=:\n"
      "mbarrier.try_wait.parity.shared.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
      : "+d"(c0), "+d"(c1)
      : "d"(a), "d"(b));
}
__device__ __forceinline__ double2 lds128(uint32_t addr) {
  double2 v;
  asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "r"(addr));
  return v;
}

enum { EPI_PARTIAL = 0, EPI_ACC = 1, EPI_STORE = 2 };   // split-K partial | C += alpha AB | C = alpha AB

// Hermitian C = A^H B (Gram matrix Psi^H (H Psi)): only the 128 x 64 tiles with floor(m/128) <=
// floor(n/128) are computed; tile column tn holds tn/2 + 1 of them, so columns 2j and 2j+1 start at linear index
// j(j+1) and (j+1)^2.  The split-K reduction mirrors the rest.
__device__ __forceinline__ void herm_tile(int idx, int& tm, int& tn) {
  int j = (int)((sqrtf(4.f * (float)idx + 1.f) - 1.f) * 0.5f);
  while (j * (j + 1) > idx) --j;
  while ((j + 1) * (j + 2) <= idx) ++j;
  const int r = idx - j * (j + 1);
  if (r <= j) { tn = 2 * j; tm = r; } else { tn = 2 * j + 1; tm = r - (j + 1); }
}

// A_KMAJOR = true : op(A)[m,k] = conj(A[k + m*lda])  (CN);   false : op(A)[m,k] = A[m + k*lda]  (NN)
// ---------------------------------------------------------------------------------------------------------------
// 3M complex product: one complex product as THREE real DMMA products instead of four,
//     T1 = ar.br,  T2 = ai.bi,  T3 = (ar + ai).(br + bi)   =>   re = T1 - T2,  im = T3 - T1 - T2
// (for conj(a): ai -> -ai).  16 warps (4 x 4), warp tile 32 x 16 complex, three accumulator sets of 16 doubles;
// the sums ar+ai / br+bi are formed on the fragments (one DADD per fragment element).  The imaginary part carries a
// rounding error of order eps.(|ar|+|ai|).(|br|+|bi|), i.e. norm-wise the same as the 4M product.
//
// There is no CTA-wide barrier in the k loop: stage s is handed over through two shared-memory mbarriers, full[s]
// (all 512 threads' cp.async of the slab have landed; cp.async.mbarrier.arrive.noinc) and empty[s] (all 16 warps are
// done reading it), so warps drift by up to one k-slab instead of meeting at every slab (ncu, profiles/r01c: 13 % of
// the stall samples sat on that __syncthreads; measured CN 38.4 -> 41.3 TFLOP/s, NN 35.4 -> 38.2 at cfg 4).
// A persistent variant that walks over tiles with the pipeline running across tile boundaries was measured too and
// was no faster (NN 37.5 vs 38.1), so one CTA computes one tile.
// ---------------------------------------------------------------------------------------------------------------
constexpr int NT3 = 512;
constexpr int W3_M = 4;                                // 4 x 4 warps; warp tile 32 x 16

template <int BK_>
struct Tile3 {
  static constexpr int BK = BK_;
  static constexpr int KROW = BK * 16 + 64;            // bytes per row of a K-major tile (== 64 mod 128)
  static constexpr int MROW = BM * 16 + 32;            // bytes per k-row of an M-major A tile (== 32 mod 128)
  static constexpr int A_K = BM * KROW, A_M = BK * MROW, B_ = BN * KROW;
};

template <bool A_KMAJOR, int EPI, int BK_, int STAGES_>
__global__ void __launch_bounds__(NT3, 1)
k_zgemm3m(int M, int N, int64_t K, int tiles_m, int64_t k_per_split, const c128* __restrict__ A, int64_t lda,
          const c128* __restrict__ B, int64_t ldb, c128* __restrict__ C, int64_t ldc, double alpha, int herm) {
  using T = Tile3<BK_>;
  constexpr int BK = BK_, STAGES = STAGES_, KROW = T::KROW, MROW = T::MROW;
  extern __shared__ __align__(1024) unsigned char smem[];
  constexpr int A_BYTES = A_KMAJOR ? T::A_K : T::A_M;
  constexpr int STAGE_BYTES = A_BYTES + T::B_;
  const uint32_t smem_base = (uint32_t)__cvta_generic_to_shared(smem);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp % W3_M, wn = warp / W3_M;
  // CN: m-tile fastest (all tiles of one K split are co-resident and share the streamed K range through L2)
  // NN: n-tile fastest (the CTAs that share one slab of A rows run together)
  int tm, tn;
  if (A_KMAJOR) {
    if (herm) herm_tile((int)blockIdx.x, tm, tn);
    else { tm = blockIdx.x % tiles_m; tn = blockIdx.x / tiles_m; }
  } else { const int tiles_n = (N + BN - 1) / BN; tn = blockIdx.x % tiles_n; tm = blockIdx.x / tiles_n; }
  const int m0 = tm * BM, n0 = tn * BN;
  const int split = blockIdx.y;
  const int64_t kbeg = (int64_t)split * k_per_split;
  const int64_t kend = (kbeg + k_per_split < K) ? kbeg + k_per_split : K;
  const int nkt = (int)((kend - kbeg + BK - 1) / BK);

  auto load_stage = [&](int stage, int kt) {
    const uint32_t sa = smem_base + stage * STAGE_BYTES, sb = sa + A_BYTES;
    const int64_t k0 = kbeg + (int64_t)kt * BK;
    if (A_KMAJOR) {
#pragma unroll
      for (int i = 0; i < (BM * BK) / NT3; ++i) {
        const int idx = tid + i * NT3, r = idx / BK, kk = idx % BK;
        const bool ok = (m0 + r < M) && (k0 + kk < kend);
        const c128* src = ok ? A + (int64_t)(m0 + r) * lda + k0 + kk : A;
        cp_async16(sa + r * KROW + kk * 16, src, ok ? 16 : 0);
      }
    } else {
#pragma unroll
      for (int i = 0; i < (BM * BK) / NT3; ++i) {
        const int idx = tid + i * NT3, kk = idx / BM, r = idx % BM;
        const bool ok = (m0 + r < M) && (k0 + kk < kend);
        const c128* src = ok ? A + (int64_t)(k0 + kk) * lda + m0 + r : A;
        cp_async16(sa + kk * MROW + r * 16, src, ok ? 16 : 0);
      }
    }
#pragma unroll
    for (int i = 0; i < (BN * BK) / NT3; ++i) {
      const int idx = tid + i * NT3, r = idx / BK, kk = idx % BK;
      const bool ok = (n0 + r < N) && (k0 + kk < kend);
      const c128* src = ok ? B + (int64_t)(n0 + r) * ldb + k0 + kk : B;
      cp_async16(sb + r * KROW + kk * 16, src, ok ? 16 : 0);
    }
  };

  double t1[4][2][2], t2[4][2][2], t3[4][2][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
      for (int h = 0; h < 2; ++h) { t1[i][j][h] = 0.0; t2[i][j][h] = 0.0; t3[i][j][h] = 0.0; }

  // slab kt lives in stage kt % STAGES; its full / empty phase number is kt / STAGES
  const uint32_t bar_full = smem_base + STAGES * STAGE_BYTES, bar_empty = bar_full + STAGES * 8;
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) { mbar_init(bar_full + 8 * s, NT3); mbar_init(bar_empty + 8 * s, NT3 / 32); }
  }
  __syncthreads();
#pragma unroll
  for (int s = 0; s < STAGES - 1; ++s)
    if (s < nkt) { load_stage(s, s); cp_async_arrive(bar_full + 8 * s); }

  const int frow = lane >> 2, fk = lane & 3;
  const uint32_t a_off = A_KMAJOR ? (uint32_t)((wm * 32 + frow) * KROW + fk * 16)
                                  : (uint32_t)(fk * MROW + (wm * 32 + frow) * 16);
  const uint32_t b_off = (uint32_t)(A_BYTES + (wn * 16 + frow) * KROW + fk * 16);

  for (int kt = 0; kt < nkt; ++kt) {
    mbar_wait(bar_full + 8 * (kt % STAGES), (uint32_t)(kt / STAGES) & 1u);
    const uint32_t st = smem_base + (kt % STAGES) * STAGE_BYTES;
#pragma unroll
    for (int k4 = 0; k4 < BK / 4; ++k4) {
      double2 b[2];
      double sb[2];
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        b[j] = lds128(st + b_off + (uint32_t)(j * 8 * KROW + k4 * 64));
        sb[j] = b[j].x + b[j].y;
      }
      if (k4 == 0) {
        // refill the stage consumed in the previous iteration (issued after this iteration's first fragment loads
        // so that the LDGSTS burst does not sit in front of them in the LSU queue)
        const int nk = kt + STAGES - 1;
        if (nk < nkt) {
          if (kt >= 1) mbar_wait(bar_empty + 8 * (nk % STAGES), (uint32_t)((kt - 1) / STAGES) & 1u);
          load_stage(nk % STAGES, nk);
          cp_async_arrive(bar_full + 8 * (nk % STAGES));
        }
      }
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const uint32_t ao = A_KMAJOR ? (uint32_t)(i * 8 * KROW + k4 * 64) : (uint32_t)(k4 * 4 * MROW + i * 8 * 16);
        const double2 a = lds128(st + a_off + ao);
        const double sa = A_KMAJOR ? a.x - a.y : a.x + a.y;
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          dmma(t1[i][j][0], t1[i][j][1], a.x, b[j].x);
          dmma(t2[i][j][0], t2[i][j][1], a.y, b[j].y);
          dmma(t3[i][j][0], t3[i][j][1], sa, sb[j]);
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(bar_empty + 8 * (kt % STAGES));
  }
  cp_async_wait<0>();

  c128* Cout = C;
  if (EPI == EPI_PARTIAL) Cout += (int64_t)split * ldc * N;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int m = m0 + wm * 32 + i * 8 + frow;
    if (m >= M) continue;
#pragma unroll
    for (int j = 0; j < 2; ++j) {
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int n = n0 + wn * 16 + j * 8 + 2 * fk + h;
        if (n >= N) continue;
        // conj(a).b : re = T1 + T2, im = T3 - T1 + T2 ;   a.b : re = T1 - T2, im = T3 - T1 - T2
        const double re = A_KMAJOR ? t1[i][j][h] + t2[i][j][h] : t1[i][j][h] - t2[i][j][h];
        const double im = A_KMAJOR ? (t3[i][j][h] - t1[i][j][h]) + t2[i][j][h] : (t3[i][j][h] - t1[i][j][h]) - t2[i][j][h];
        c128* p = Cout + (int64_t)n * ldc + m;
        if (EPI == EPI_PARTIAL) {
          *p = cmake(re, im);
        } else if (EPI == EPI_STORE) {
          *p = cmake(alpha * re, alpha * im);
        } else {
          c128 t = *p;
          t.x = fma(alpha, re, t.x);
          t.y = fma(alpha, im, t.y);
          *p = t;
        }
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// TMA-fed 3M kernel (the default when the driver exports cuTensorMapEncodeTiled): same warp tiling, 3M arithmetic,
// mbarrier hand-over and epilogue as k_zgemm3m, but the operand slabs are brought in by the TMA engine
// (cp.async.bulk.tensor, 128-byte swizzle) instead of 512 threads x 3-6 LDGSTS with their address arithmetic:
// the instruction stream of the 16 warps is then only wait / LDS / DADD / DMMA, which is what the register-level
// probe of this loop shows to run at 92 % of the DMMA peak.
//   * matrices are described to the TMA as FP64 tensors with the (re, im) pair innermost: 8 complex = 128 bytes;
//   * K-major operands (A of CN, B): box = 8 k x rows, dense rows of 128 B in shared memory, chunk c of row r stored
//     at chunk c ^ (r & 7); the fragment of k-slot fk at step k4 is physical k = 2 fk + (k4 & 1), which makes the 2 rows
//     x 4 k of a quarter-warp hit 8 different chunks (any assignment of k to the 4 slots of m8n8k4 is valid as long
//     as A and B agree);
//   * M-major A of NN: one box of 8 m x BK k per group of 8 rows, stored [m group][k][8 m], chunk m stored at
//     m ^ (k & 7): with the same k assignment the quarter-warp (2 m x 4 k) again hits 8 different chunks;
//   * rows / k beyond the matrix are zero-filled by the TMA, so there are no predicates in the loop.
// One warp (rotating with the slab number) waits for the stage to be drained, posts the byte count on full[s] and
// issues the boxes; nobody else ever waits on empty[s].
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.expect_tx.shared.b64 st, [%0], %1;\n}\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n" ::"r"(dst),
      "l"(tm), "r"(c0), "r"(c1), "r"(bar)
      : "memory");
}

// JT: 8-column MMA tiles per warp along n -- 2: 16 warps of 32 x 16 (the shape measured throughout); 4: 8 warps of 32 x 32
// (fewer fragment loads and operand sums per DMMA, 192 accumulator registers)
template <bool A_KMAJOR, int EPI, int BK_, int STAGES_, int JT = 2>
__global__ void __launch_bounds__(NT3 * 2 / JT, 1)
k_zgemm3m_tma(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, int M, int N, int64_t K,
              int tiles_m, int64_t k_per_split, c128* __restrict__ C, int64_t ldc, double alpha, int herm) {
  constexpr int BK = BK_, STAGES = STAGES_, SS = BK / 8;        // SS sub-slabs of 8 k per stage
  constexpr int A_SUB = BM * 128, B_SUB = BN * 128;             // bytes of one 8-k sub-slab of A and of B
  constexpr int A_BYTES = SS * A_SUB, STAGE_BYTES = SS * (A_SUB + B_SUB);
  extern __shared__ __align__(1024) unsigned char smem[];
  const uint32_t smem_base = ((uint32_t)__cvta_generic_to_shared(smem) + 1023u) & ~1023u;
  constexpr int NW = 16 * 2 / JT;                                // warps of the CTA
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp % W3_M, wn = warp / W3_M;
  int tm, tn;
  if (A_KMAJOR) {
    if (herm) herm_tile((int)blockIdx.x, tm, tn);
    else { tm = blockIdx.x % tiles_m; tn = blockIdx.x / tiles_m; }
  } else { const int tiles_n = (N + BN - 1) / BN; tn = blockIdx.x % tiles_n; tm = blockIdx.x / tiles_n; }
  const int m0 = tm * BM, n0 = tn * BN;
  const int split = blockIdx.y;
  const int64_t kbeg = (int64_t)split * k_per_split;
  const int64_t kend = (kbeg + k_per_split < K) ? kbeg + k_per_split : K;
  const int nkt = (int)((kend - kbeg + BK - 1) / BK);

  const uint32_t bar_full = smem_base + STAGES * STAGE_BYTES, bar_empty = bar_full + STAGES * 8;
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) { mbar_init(bar_full + 8 * s, 1); mbar_init(bar_empty + 8 * s, NW); }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();

  // whole warp: post the byte count of slab kt on full[stage] and issue its boxes
  auto issue_slab = [&](int stage, int kt) {
    const uint32_t sa = smem_base + stage * STAGE_BYTES, sb = sa + A_BYTES, bar = bar_full + 8 * stage;
    const int k0 = (int)(kbeg + (int64_t)kt * BK);
    if (lane == 0) mbar_expect_tx(bar, STAGE_BYTES);
    __syncwarp();
    if (A_KMAJOR) {
      if (lane < SS) tma_load_2d(sa + lane * A_SUB, &tmA, 2 * (k0 + 8 * lane), m0, bar);
    } else {
      // box = 8 m (inner) x BK k; m group g goes to sa + g * (BK * 128)
      if (lane < BM / 8) tma_load_2d(sa + lane * (BK * 128), &tmA, 2 * (m0 + 8 * lane), k0, bar);
    }
    if (lane >= 16 && lane < 16 + SS) tma_load_2d(sb + (lane - 16) * B_SUB, &tmB, 2 * (k0 + 8 * (lane - 16)), n0, bar);
  };

  if (warp == 0) {
#pragma unroll 1
    for (int s = 0; s < STAGES - 1; ++s)
      if (s < nkt) issue_slab(s, s);
  }

  double t1[4][JT][2], t2[4][JT][2], t3[4][JT][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < JT; ++j)
#pragma unroll
      for (int h = 0; h < 2; ++h) { t1[i][j][h] = 0.0; t2[i][j][h] = 0.0; t3[i][j][h] = 0.0; }

  const int frow = lane >> 2, fk = lane & 3;
  // byte offsets of this thread's fragments for the even k4 steps of a sub-slab (physical k = 2 fk); the odd steps
  // (k = 2 fk + 1) are one chunk (and, for the M-major A, one k row) further: offset ^ 16 (^ 128), the stage base being
  // 1024-byte aligned
  const uint32_t a_off0 = A_KMAJOR ? (uint32_t)((wm * 32 + frow) * 128 + (((2 * fk) ^ frow) * 16))
                                   : (uint32_t)((wm * 4) * (BK * 128) + (2 * fk) * 128 + ((frow ^ (2 * fk)) * 16));
  const uint32_t b_off0 = (uint32_t)(A_BYTES + (wn * (8 * JT) + frow) * 128 + (((2 * fk) ^ frow) * 16));
  constexpr uint32_t A_ODD = A_KMAJOR ? 16u : (16u | 128u), B_ODD = 16u;

  for (int kt = 0; kt < nkt; ++kt) {
    const int stage = kt % STAGES;
    mbar_wait(bar_full + 8 * stage, (uint32_t)(kt / STAGES) & 1u);
    const uint32_t st = smem_base + stage * STAGE_BYTES;
#pragma unroll
    for (int k4 = 0; k4 < BK / 4; ++k4) {
      const int ss = k4 >> 1, par = k4 & 1;
      double2 b[JT];
      double sb[JT];
#pragma unroll
      for (int j = 0; j < JT; ++j) {
        b[j] = lds128(((st + b_off0) ^ (par ? B_ODD : 0u)) + (uint32_t)(ss * B_SUB + j * 8 * 128));
        sb[j] = b[j].x + b[j].y;
      }
      if (k4 == 0) {
        const int nk = kt + STAGES - 1;
        if (nk < nkt && warp == (kt & (NW - 1))) {
          if (kt >= 1) mbar_wait(bar_empty + 8 * (nk % STAGES), (uint32_t)((kt - 1) / STAGES) & 1u);
          issue_slab(nk % STAGES, nk);
        }
      }
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        // K-major A: sub-slab ss, row block i -> + i*8 rows;  M-major A: m group wm*4 + i, k within the box = 8 ss + ...
        const uint32_t ao = A_KMAJOR ? (uint32_t)(ss * A_SUB + i * 8 * 128) : (uint32_t)(i * (BK * 128) + ss * 8 * 128);
        const double2 a = lds128(((st + a_off0) ^ (par ? A_ODD : 0u)) + ao);
        const double sa = A_KMAJOR ? a.x - a.y : a.x + a.y;
#pragma unroll
        for (int j = 0; j < JT; ++j) {
          dmma(t1[i][j][0], t1[i][j][1], a.x, b[j].x);
          dmma(t2[i][j][0], t2[i][j][1], a.y, b[j].y);
          dmma(t3[i][j][0], t3[i][j][1], sa, sb[j]);
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(bar_empty + 8 * stage);
  }

  c128* Cout = C;
  if (EPI == EPI_PARTIAL) Cout += (int64_t)split * ldc * N;
  if (EPI == EPI_ACC) {
    // accumulate onto C: the 2 JT entries of one row block are loaded together before any of them is stored (a load behind a
    // store through the same pointer cannot be hoisted by the compiler: one round trip per row block instead of one per entry)
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int m = m0 + wm * 32 + i * 8 + frow;
      if (m >= M) continue;
      c128 old[JT][2];
#pragma unroll
      for (int j = 0; j < JT; ++j)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int n = n0 + wn * (8 * JT) + j * 8 + 2 * fk + h;
          old[j][h] = n < N ? C[(int64_t)n * ldc + m] : cmake(0.0, 0.0);
        }
#pragma unroll
      for (int j = 0; j < JT; ++j)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int n = n0 + wn * (8 * JT) + j * 8 + 2 * fk + h;
          if (n >= N) continue;
          const double re = A_KMAJOR ? t1[i][j][h] + t2[i][j][h] : t1[i][j][h] - t2[i][j][h];
          const double im = A_KMAJOR ? (t3[i][j][h] - t1[i][j][h]) + t2[i][j][h] : (t3[i][j][h] - t1[i][j][h]) - t2[i][j][h];
          C[(int64_t)n * ldc + m] = cmake(fma(alpha, re, old[j][h].x), fma(alpha, im, old[j][h].y));
        }
    }
    return;
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int m = m0 + wm * 32 + i * 8 + frow;
    if (m >= M) continue;
#pragma unroll
    for (int j = 0; j < JT; ++j) {
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int n = n0 + wn * (8 * JT) + j * 8 + 2 * fk + h;
        if (n >= N) continue;
        const double re = A_KMAJOR ? t1[i][j][h] + t2[i][j][h] : t1[i][j][h] - t2[i][j][h];
        const double im = A_KMAJOR ? (t3[i][j][h] - t1[i][j][h]) + t2[i][j][h] : (t3[i][j][h] - t1[i][j][h]) - t2[i][j][h];
        c128* p = Cout + (int64_t)n * ldc + m;
        if (EPI == EPI_PARTIAL) {
          *p = cmake(re, im);
        } else if (EPI == EPI_STORE) {
          *p = cmake(alpha * re, alpha * im);
        } else {
          c128 t = *p;
          t.x = fma(alpha, re, t.x);
          t.y = fma(alpha, im, t.y);
          *p = t;
        }
      }
    }
  }
}

// C[m + n*ldc] = scale[m] * sum_s part[s][m + n*M]   (fixed summation order => deterministic).  herm: the partial sums
// exist for floor(m/128) <= floor(n/128) only; the other entries are the conjugates of their mirror images.
// swapped: the partial sums hold the N x M matrix B^H A = (A^H B)^H (operands exchanged by launch_zgemm_cn), so every entry is
// the conjugate of its transposed image.
__global__ void __launch_bounds__(256) k_splitk_reduce(int M, int N, int nsplit, const c128* __restrict__ part,
                                                       const double* __restrict__ scale, c128* __restrict__ C,
                                                       int64_t ldc, int herm, int swapped) {
  const int64_t total = (int64_t)M * N;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int m = (int)(i % M);
    const int64_t n = i / M;
    const bool mirror = swapped || (herm && (m / BM) > (int)(n / BM));
    const int64_t src = swapped ? (int64_t)m * N + n : (mirror ? (int64_t)m * M + n : i);
    double sx = 0.0, sy = 0.0;
    for (int s = 0; s < nsplit; ++s) {
      const c128 v = part[(int64_t)s * total + src];
      sx += v.x;
      sy += v.y;
    }
    if (mirror) sy = -sy;
    const double f = scale ? scale[m] : 1.0;
    C[n * ldc + m] = cmake(f * sx, f * sy);
  }
}

// Register-resident DMMA loop: the attainable FP64 tensor-pipe rate on this GPU at its current clocks (the
// denominator of the ZGEMM roofline fraction).  32 independent accumulator pairs per warp, no memory traffic.
__global__ void __launch_bounds__(256) k_dmma_probe(int iters, double* __restrict__ sink) {
  double c[32][2];
#pragma unroll
  for (int i = 0; i < 32; ++i) { c[i][0] = 0.0; c[i][1] = 0.0; }
  double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 32; ++i) dmma(c[i][0], c[i][1], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 32; ++i) s += c[i][0] + c[i][1];
  if (s == 12345.678) sink[0] = s;
}

// 3M kernels: CN streams K = npw in slabs of 8 through 4 stages, NN (K = nproj) in slabs of 16 through 3 stages
// (measured on B200, cfg 3/4: CN 41.3 vs 40.7 TFLOP/s and NN 35.7 vs 38.2 for slabs of 8 vs 16)
constexpr int CN3_BK = 8, CN3_STAGES = 4, NN3_BK = 16, NN3_STAGES = 3;
// TMA-fed kernels: CN 8-k slabs x 6 stages (24 KB each), NN 16-k slabs x 4 stages (48 KB each); + 1 KB alignment slack
constexpr int CNT_BK = 8, CNT_STAGES = 6, NNT_BK = 16, NNT_STAGES = 4;
constexpr int smem_tma(int bk, int stages) { return stages * (bk / 8) * (BM + BN) * 128 + 2 * stages * 8 + 1024; }
constexpr int smem_cn3() { return CN3_STAGES * (Tile3<CN3_BK>::A_K + Tile3<CN3_BK>::B_) + 2 * CN3_STAGES * 8; }
constexpr int smem_nn3() { return NN3_STAGES * (Tile3<NN3_BK>::A_M + Tile3<NN3_BK>::B_) + 2 * NN3_STAGES * 8; }
constexpr int NUM_SMS = 148;
// warp-tile shapes of the TMA kernels (measured, profiles/r02j): 8 warps of 32 x 32 for CN (-3.3 % at cfg 5: fewer fragment
// loads and operand sums per DMMA), 16 warps of 32 x 16 for NN (the 32 x 32 shape is 1-5 % slower there: its accumulating epilogue
// and M-major A fragments want the extra warps)
constexpr int ZJT_CN = 4, ZJT_NN = 2;

}  // namespace

// cuTensorMapEncodeTiled through the runtime's driver entry point (libcuda is not linked)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static std::atomic<bool> g_no_tma{false};
void zgemm_set_no_tma(bool off) { g_no_tma.store(off, std::memory_order_relaxed); }

static EncodeTiledFn encode_fn() {
  if (g_no_tma.load(std::memory_order_relaxed)) return nullptr;
  static const EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      p = nullptr;
    return (EncodeTiledFn)p;
  }();
  return fn;
}

// column-major complex matrix `inner` x `outer` (leading dimension ld) as an FP64 tensor {2 inner, outer};
// box = 8 complex (128 B, swizzled) x box_outer
static bool make_map(CUtensorMap* tm, const c128* base, int64_t inner, int64_t outer, int64_t ld, int box_outer) {
  EncodeTiledFn fn = encode_fn();
  if (!fn || ((uintptr_t)base & 15) || inner < 1 || outer < 1) return false;
  const cuuint64_t dims[2] = {(cuuint64_t)(2 * inner), (cuuint64_t)outer};
  const cuuint64_t strides[1] = {(cuuint64_t)ld * sizeof(c128)};
  const cuuint32_t box[2] = {16u, (cuuint32_t)box_outer};
  const cuuint32_t estr[2] = {1u, 1u};
  return fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<c128*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// The projector matrix of a handle never changes: its two tensor maps (K-major operand of P^H Y, M-major operand of
// P C) are encoded once at setup.  `ok` is false when the driver has no TMA encoder or refused the operand.
void zgemm_make_proj_maps(ProjMaps& pm, const c128* P, int64_t npw, int64_t nproj, int64_t ldp) {
  static_assert(sizeof(CUtensorMap) == sizeof(pm.cn), "ProjMaps storage");
  pm.ok = nproj > 0 && make_map(reinterpret_cast<CUtensorMap*>(pm.cn), P, npw, nproj, ldp, BM) &&
          make_map(reinterpret_cast<CUtensorMap*>(pm.cnb), P, npw, nproj, ldp, BN) &&
          make_map(reinterpret_cast<CUtensorMap*>(pm.nn), P, npw, nproj, ldp, NNT_BK);
}

cudaError_t zgemm_init() {
  cudaError_t e = set_max_dyn_smem(reinterpret_cast<const void*>(&k_zgemm3m_tma<true, EPI_PARTIAL, CNT_BK, CNT_STAGES, ZJT_CN>));
  if (e != cudaSuccess) return e;
  e = set_max_dyn_smem(reinterpret_cast<const void*>(&k_zgemm3m_tma<false, EPI_ACC, NNT_BK, NNT_STAGES, ZJT_NN>));
  if (e != cudaSuccess) return e;
  e = set_max_dyn_smem(reinterpret_cast<const void*>(&k_zgemm3m_tma<false, EPI_STORE, NNT_BK, NNT_STAGES, ZJT_NN>));
  if (e != cudaSuccess) return e;
  e = set_max_dyn_smem(reinterpret_cast<const void*>(&k_zgemm3m<true, EPI_PARTIAL, CN3_BK, CN3_STAGES>));
  if (e != cudaSuccess) return e;
  e = set_max_dyn_smem(reinterpret_cast<const void*>(&k_zgemm3m<false, EPI_ACC, NN3_BK, NN3_STAGES>));
  if (e != cudaSuccess) return e;
  return set_max_dyn_smem(reinterpret_cast<const void*>(&k_zgemm3m<false, EPI_STORE, NN3_BK, NN3_STAGES>));
}

cudaError_t dmma_probe(int iters, int ctas, double* sink, cudaStream_t st, float* ms) {
  cudaEvent_t e0, e1;
  cudaError_t e;
  if ((e = cudaEventCreate(&e0)) != cudaSuccess) return e;
  if ((e = cudaEventCreate(&e1)) != cudaSuccess) return e;
  k_dmma_probe<<<ctas, 256, 0, st>>>(iters / 8 + 1, sink);  // warm-up
  cudaEventRecord(e0, st);
  k_dmma_probe<<<ctas, 256, 0, st>>>(iters, sink);
  cudaEventRecord(e1, st);
  count_launch();
  count_launch();
  e = cudaEventSynchronize(e1);
  if (e == cudaSuccess) e = cudaEventElapsedTime(ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return e;
}

// number of 128 x 64 tiles of C the CN kernel computes: all of them, or -- for a Hermitian C (herm) -- those that
// touch the block upper triangle  floor(m/128) <= floor(n/128)
// C = A^H B can equally be computed as (B^H A)^H: with the 128 x 64 tile the two orientations pad differently
// (cfg 5: 1728 projectors x 512 bands is 14 x 8 = 112 tiles one way, 4 x 27 = 108 the other); exchange the operands
// when that saves more than 2 % of the tiles.
static bool cn_swapped(int64_t M, int64_t N, bool herm) {
  if (herm) return false;
  const int64_t a = ((M + BM - 1) / BM) * ((N + BN - 1) / BN), b = ((N + BM - 1) / BM) * ((M + BN - 1) / BN);
  return b * 100 < a * 98;
}

static int64_t cn_tiles(int64_t M, int64_t N, bool herm) {
  if (cn_swapped(M, N, herm)) std::swap(M, N);
  const int64_t tiles_m = (M + BM - 1) / BM, tiles_n = (N + BN - 1) / BN;
  if (!herm) return tiles_m * tiles_n;
  int64_t t = 0;
  for (int64_t tn = 0; tn < tiles_n; ++tn) t += std::min<int64_t>(tiles_m, tn / 2 + 1);
  return t;
}

static int splits_for_tiles(int64_t tiles, int64_t K) {
  // Split K so that tiles * splits fills whole waves of the 148 SMs (one CTA per SM): among the candidates with at
  // most 16 waves and at least 8 k-slabs per split, take the fewest splits within 1 % of the best wave efficiency.
  const int64_t max_split = std::max<int64_t>(1, K / (8 * CNT_BK));   // small problems: one wave of short CTAs
  int best = 1;
  double best_eff = 0.0;
  for (int64_t s = 1; s <= max_split; ++s) {
    const int64_t ctas = tiles * s;
    const int64_t w = (ctas + NUM_SMS - 1) / NUM_SMS;
    if (w > 16 && s > 1) break;
    const double eff = (double)ctas / (double)(w * NUM_SMS);
    if (eff > best_eff + 0.01) { best_eff = eff; best = (int)s; }
  }
  return best;
}

int zgemm_cn_splits(int64_t M, int64_t N, int64_t K, bool herm) { return splits_for_tiles(cn_tiles(M, N, herm), K); }

size_t zgemm_cn_workspace(int64_t M, int64_t N, int64_t K, bool herm) {
  return sizeof(c128) * (size_t)zgemm_cn_splits(M, N, K, herm) * (size_t)M * (size_t)N;
}

// max over n <= N of zgemm_cn_workspace(M, n, K): the split count is not monotone in the number of tiles, so a
// workspace sized for N bands must be sized for the worst narrower block as well
size_t zgemm_cn_workspace_upto(int64_t M, int64_t N, int64_t K) {
  size_t best = 0;
  for (int64_t tn = 1; tn <= (N + BN - 1) / BN; ++tn) {
    const int64_t n = std::min<int64_t>(tn * BN, N);
    best = std::max(best, zgemm_cn_workspace(M, n, K, false));
  }
  return best;
}

void launch_zgemm_cn(int64_t M, int64_t N, int64_t K, const c128* A, int64_t lda, const c128* B, int64_t ldb,
                     const double* scale, c128* C, int64_t ldc, void* ws, cudaStream_t st, const ProjMaps* pmA, bool herm) {
  if (M <= 0 || N <= 0) return;
  if (M != N) herm = false;
  const int nsplit = zgemm_cn_splits(M, N, K, herm);
  const bool swapped = cn_swapped(M, N, herm);
  // the product the kernel computes: Mk x Nk = Ak^H Bk (the operands exchanged when `swapped`)
  const int64_t Mk = swapped ? N : M, Nk = swapped ? M : N;
  const c128 *Ak = swapped ? B : A, *Bk = swapped ? A : B;
  const int64_t ldak = swapped ? ldb : lda, ldbk = swapped ? lda : ldb;
  const int tiles_m = (int)((Mk + BM - 1) / BM);
  int64_t kps = (K + nsplit - 1) / nsplit;
  kps = (kps + CNT_BK - 1) / CNT_BK * CNT_BK;
  dim3 grid((unsigned)cn_tiles(M, N, herm), nsplit);
  c128* part = reinterpret_cast<c128*>(ws);
  {
    ScopedLaunch sl(ST_ZGEMM_CN, st);
    CUtensorMap tmA, tmB;
    const bool cached = pmA && pmA->ok && !g_no_tma.load(std::memory_order_relaxed);
    bool tma;
    if (!swapped) {
      if (cached) { memcpy(&tmA, pmA->cn, sizeof(tmA)); tma = true; }
      else tma = make_map(&tmA, Ak, K, Mk, ldak, BM);
      tma = tma && make_map(&tmB, Bk, K, Nk, ldbk, BN);
    } else {
      tma = make_map(&tmA, Ak, K, Mk, ldak, BM);
      if (tma && cached) memcpy(&tmB, pmA->cnb, sizeof(tmB));
      else tma = tma && make_map(&tmB, Bk, K, Nk, ldbk, BN);
    }
    if (tma)
      k_zgemm3m_tma<true, EPI_PARTIAL, CNT_BK, CNT_STAGES, ZJT_CN><<<grid, NT3 * 2 / ZJT_CN, smem_tma(CNT_BK, CNT_STAGES), st>>>(
          tmA, tmB, (int)Mk, (int)Nk, K, tiles_m, kps, part, Mk, 0.0, herm ? 1 : 0);
    else
      k_zgemm3m<true, EPI_PARTIAL, CN3_BK, CN3_STAGES><<<grid, NT3, smem_cn3(), st>>>(
          (int)Mk, (int)Nk, K, tiles_m, kps, Ak, ldak, Bk, ldbk, part, Mk, 0.0, herm ? 1 : 0);
  }
  const int64_t total = M * N;
  int blocks = (int)((total + 255) / 256);
  if (blocks > NUM_SMS * 8) blocks = NUM_SMS * 8;
  ScopedLaunch sl(ST_SPLITK, st);
  k_splitk_reduce<<<blocks, 256, 0, st>>>((int)M, (int)N, nsplit, part, scale, C, ldc, herm ? 1 : 0, swapped ? 1 : 0);
}

// C = alpha * A B (+ C when accumulate)
void launch_zgemm_nn(int64_t M, int64_t N, int64_t K, double alpha, const c128* A, int64_t lda, const c128* B,
                     int64_t ldb, c128* C, int64_t ldc, bool accumulate, cudaStream_t st, const ProjMaps* pmA) {
  if (M <= 0 || N <= 0 || K <= 0) return;
  const int tiles_m = (int)((M + BM - 1) / BM), tiles_n = (int)((N + BN - 1) / BN);
  dim3 grid(tiles_m * tiles_n, 1);
  ScopedLaunch sl(ST_ZGEMM_NN, st);
  CUtensorMap tmA, tmB;
  bool tma = false;
  if (pmA && pmA->ok && !g_no_tma.load(std::memory_order_relaxed)) { memcpy(&tmA, pmA->nn, sizeof(tmA)); tma = true; }
  else tma = make_map(&tmA, A, M, K, lda, NNT_BK);
  tma = tma && make_map(&tmB, B, K, N, ldb, BN);
  if (tma && accumulate)
    k_zgemm3m_tma<false, EPI_ACC, NNT_BK, NNT_STAGES, ZJT_NN><<<grid, NT3 * 2 / ZJT_NN, smem_tma(NNT_BK, NNT_STAGES), st>>>(
        tmA, tmB, (int)M, (int)N, K, tiles_m, K, C, ldc, alpha, 0);
  else if (tma)
    k_zgemm3m_tma<false, EPI_STORE, NNT_BK, NNT_STAGES, ZJT_NN><<<grid, NT3 * 2 / ZJT_NN, smem_tma(NNT_BK, NNT_STAGES), st>>>(
        tmA, tmB, (int)M, (int)N, K, tiles_m, K, C, ldc, alpha, 0);
  else if (accumulate)
    k_zgemm3m<false, EPI_ACC, NN3_BK, NN3_STAGES><<<grid, NT3, smem_nn3(), st>>>(
        (int)M, (int)N, K, tiles_m, K, A, lda, B, ldb, C, ldc, alpha, 0);
  else
    k_zgemm3m<false, EPI_STORE, NN3_BK, NN3_STAGES><<<grid, NT3, smem_nn3(), st>>>(
        (int)M, (int)N, K, tiles_m, K, A, lda, B, ldb, C, ldc, alpha, 0);
}

}  // namespace pwh

// ---------------------------------------------------------------------------------------------------------------
// pwh_gram_static -- the Gram product for callers that may not allocate (include/pwham.h): the split-K partial sums that
// pwh_gram keeps in a caller-provided workspace live in a file-scope device array of fixed size instead.  The array exists
// once per GPU that loads the library and is shared by every call: calls that overlap on the GPU race on it.  Nothing in it
// has to start at zero -- the CN kernel writes every partial entry of every split before the reduction reads it.
// ---------------------------------------------------------------------------------------------------------------
#include <mutex>

#include "../../include/pwham.h"

static_assert(PWH_GRAM_STATIC_MAX_ENTRIES == 1048576, "keep include/pwham.h and the scratch array in step");
constexpr size_t GRAM_STATIC_BYTES = (size_t)PWH_GRAM_STATIC_MAX_ENTRIES * sizeof(pwh::c128);     // 16 MiB
static __device__ __align__(256) unsigned char g_gram_static_scratch[GRAM_STATIC_BYTES];

// device address of the array on the current device: its name is only a host-side stand-in here, so the address is asked
// for once per device, with that device current
static cudaError_t gram_static_scratch(void** out) {
  constexpr int MAXDEV = 64;
  static std::mutex mu;
  static void* addr[MAXDEV] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= MAXDEV) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(mu);
  if (!addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_gram_static_scratch);
    if (e != cudaSuccess) return e;
    addr[dev] = p;
  }
  *out = addr[dev];
  return cudaSuccess;
}

extern "C" int pwh_gram_static(int64_t npw, int64_t nx, const pwh_c128* X, int64_t ldx, int64_t ny, const pwh_c128* Y,
                               int64_t ldy, pwh_c128* G, int64_t ldg, void* stream) {
  using namespace pwh;
  if (npw < 1 || nx < 0 || ny < 0) return api_fail(PWH_EINVAL, "bad sizes");
  if (nx == 0 || ny == 0) return PWH_OK;
  if (!X || !Y || !G) return api_fail(PWH_EINVAL, "null argument");
  if (ldx < npw || ldy < npw || ldg < nx) return api_fail(PWH_EINVAL, "leading dimension too small");
  if (nx > PWH_GRAM_STATIC_MAX_ENTRIES || ny > PWH_GRAM_STATIC_MAX_ENTRIES || nx * ny > (int64_t)PWH_GRAM_STATIC_MAX_ENTRIES)
    return api_fail(PWH_EINVAL, "pwh_gram_static: nx * ny = %lld exceeds the static scratch of %lld entries (use pwh_gram)",
                    (long long)(nx * ny), (long long)PWH_GRAM_STATIC_MAX_ENTRIES);
  cudaError_t e = zgemm_init();
  if (e != cudaSuccess) return api_fail(PWH_ECUDA, "zgemm_init: %s", cudaGetErrorString(e));
  void* scratch = nullptr;
  e = gram_static_scratch(&scratch);
  if (e != cudaSuccess) return api_fail(PWH_ECUDA, "cudaGetSymbolAddress: %s", cudaGetErrorString(e));
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t M = nx, N = ny, K = npw;
  // as many K splits as pwh_gram would take, capped so that the partial sums fit the array (at least one always does)
  int nsplit = zgemm_cn_splits(M, N, K, false);
  const int64_t cap = (int64_t)PWH_GRAM_STATIC_MAX_ENTRIES / (M * N);
  if (nsplit > cap) nsplit = (int)cap;
  const int tiles_m = (int)((M + BM - 1) / BM), tiles_n = (int)((N + BN - 1) / BN);
  int64_t kps = (K + nsplit - 1) / nsplit;
  kps = (kps + CNT_BK - 1) / CNT_BK * CNT_BK;
  dim3 grid((unsigned)(tiles_m * tiles_n), (unsigned)nsplit);
  c128* part = reinterpret_cast<c128*>(scratch);
  const c128 *A = reinterpret_cast<const c128*>(X), *B = reinterpret_cast<const c128*>(Y);
  CUtensorMap tmA, tmB;
  count_launch();
  if (make_map(&tmA, A, K, M, ldx, BM) && make_map(&tmB, B, K, N, ldy, BN))
    k_zgemm3m_tma<true, EPI_PARTIAL, CNT_BK, CNT_STAGES, ZJT_CN><<<grid, NT3 * 2 / ZJT_CN, smem_tma(CNT_BK, CNT_STAGES), st>>>(
        tmA, tmB, (int)M, (int)N, K, tiles_m, kps, part, M, 0.0, 0);
  else
    k_zgemm3m<true, EPI_PARTIAL, CN3_BK, CN3_STAGES><<<grid, NT3, smem_cn3(), st>>>((int)M, (int)N, K, tiles_m, kps, A, ldx, B, ldy,
                                                                                   part, M, 0.0, 0);
  const int64_t total = M * N;
  int blocks = (int)((total + 255) / 256);
  if (blocks > NUM_SMS * 8) blocks = NUM_SMS * 8;
  count_launch();
  k_splitk_reduce<<<blocks, 256, 0, st>>>((int)M, (int)N, nsplit, part, nullptr, reinterpret_cast<c128*>(G), ldg, 0, 0);
  e = cudaGetLastError();
  if (e != cudaSuccess) return api_fail(PWH_ECUDA, "pwh_gram_static launch: %s", cudaGetErrorString(e));
  return PWH_OK;
}

