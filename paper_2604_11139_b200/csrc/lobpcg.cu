// lobpcg.cu -- one LOBPCG block solve on the same H application (Algorithm 11 with
// S = I, outline PAPER.md:169-197 Algorithm 6; S-Deflate / S-Ortho / RR = Algorithms 8-10; the diagonal
// preconditioner K of PAPER.md:504).  The N x M work runs on the kernels that already exist (pwh_apply_h, the DMMA ZGEMMs
// behind Gram products and rotations, the dense M x M solvers of rr.cu); this file adds the one fused column kernel of
// lines 11-13 (residual, its norm, the band's kinetic energy, the preconditioner) and the launch sequence of the algorithm.
//
// Basis layout.  The search directions of a block live in one column-major N x 3m buffer [Psi_i | W_i | P_i] (m = M / b) with
// H applied in a second buffer of the same shape, so that S-Ortho and RR of the 2m or 3m vectors (lines 21-25) act on one
// contiguous block; the Ritz rotation writes the new [Psi_i | . | P_i] into a second pair of buffers (a GEMM cannot run in
// place) and the pairs swap roles every line minimisation.  Line 26 needs no extra pass: with the basis B orthonormal and
// C the lowest m Ritz vectors, the new Psi_i = B C and P_i = B[:, m:] C[m:, :] (the part outside span(Psi_i)).
#include "../../include/pwham.h"

#include <algorithm>
#include <cstdint>
#include <vector>

#include "launch.h"

using namespace pwh;

#define LB_TRY(expr)                                                                                      \
  do {                                                                                                    \
    cudaError_t e__ = (expr);                                                                             \
    if (e__ != cudaSuccess) return api_fail(PWH_ECUDA, "%s: %s", #expr, cudaGetErrorString(e__));        \
  } while (0)
#define LB_RC(expr)                \
  do {                             \
    const int rc__ = (expr);       \
    if (rc__ != PWH_OK) return rc__; \
  } while (0)

namespace {

constexpr int LT = 256;

__device__ __forceinline__ double lb_block_sum(double v, double* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  double s = 0.0;
  for (int i = 0; i < LT / 32; ++i) s += red[i];
  return s;
}

// Lines 11-13 for one band per CTA: W = K (H psi - lambda S psi), norms = ||H psi - lambda S psi||_2 (before K; S psi = psi
// when spsi is null),
// K(G) = t / (t + 16 x^4), t = 27 + 18 x + 12 x^2 + 8 x^3, x = kin(G) / <T>, <T> = sum kin |psi|^2 / sum |psi|^2
// (Teter-Payne-Allan; reading R16).  The second pass re-reads the two columns from L2.
__global__ void __launch_bounds__(LT) k_residual_precond(int64_t npw, const double* __restrict__ kin,
                                                         const c128* __restrict__ psi, int64_t ld,
                                                         const c128* __restrict__ hpsi, int64_t ldh,
                                                         const c128* __restrict__ spsi, int64_t lds,
                                                         const double* __restrict__ lambda, c128* __restrict__ W, int64_t ldw,
                                                         double* __restrict__ norms) {
  __shared__ double red[LT / 32];
  const c128* x = psi + (int64_t)blockIdx.x * ld;
  const c128* y = hpsi + (int64_t)blockIdx.x * ldh;
  const c128* z = spsi ? spsi + (int64_t)blockIdx.x * lds : x;     // S psi (the generalised problem) or psi itself
  c128* w = W + (int64_t)blockIdx.x * ldw;
  const double lam = lambda[blockIdx.x];
  double tk = 0.0, nn = 0.0, rr = 0.0;
  for (int64_t g = threadIdx.x; g < npw; g += LT) {
    const c128 a = x[g], b = y[g], c = z[g];
    const double a2 = fma(a.x, a.x, a.y * a.y);
    tk = fma(kin[g], a2, tk);
    nn += a2;
    const double rx = fma(-lam, c.x, b.x), ry = fma(-lam, c.y, b.y);
    rr = fma(rx, rx, fma(ry, ry, rr));
  }
  tk = lb_block_sum(tk, red);
  nn = lb_block_sum(nn, red);
  rr = lb_block_sum(rr, red);
  if (threadIdx.x == 0) norms[blockIdx.x] = sqrt(rr);
  const double ekin = tk / nn;
  for (int64_t g = threadIdx.x; g < npw; g += LT) {
    const c128 a = z[g], b = y[g];
    const double xx = kin[g] / ekin;
    const double t = 27.0 + xx * (18.0 + xx * (12.0 + 8.0 * xx));
    const double x2 = xx * xx;
    const double k = t / (t + 16.0 * x2 * x2);
    w[g] = cmake(k * fma(-lam, a.x, b.x), k * fma(-lam, a.y, b.y));
  }
}

// status of the dense solvers folded into one word: dst < 0 once anything failed, else the largest Jacobi sweep count.
// potrf-style sources report 0 / j+1 (failure), hegv-style sources > 0 sweeps / < 0 failure.
__global__ void k_info_fold(const int* __restrict__ src, int potrf_style, int* __restrict__ dst) {
  const int s = *src, d = *dst;
  if (d < 0) return;
  if (potrf_style) { if (s > 0) *dst = -s; }
  else if (s < 0) *dst = s;
  else if (s > d) *dst = s;
}

struct LbWs {
  size_t b[2], hb[2], sb[2], coef, hs, ss, c, theta, norms, info, shared, shared_bytes, total;
};

size_t up256(size_t v) { return (v + 255) / 256 * 256; }

LbWs lb_layout(const pwh_ham* ham, int64_t npw, int64_t nband, int64_t m, bool gen) {
  LbWs L;
  const size_t blk = up256((size_t)npw * 3 * m * sizeof(c128));
  const size_t mat = up256((size_t)9 * m * m * sizeof(c128));
  size_t off = 0;
  for (int i = 0; i < 2; ++i) { L.b[i] = off; off += blk; L.hb[i] = off; off += blk; L.sb[i] = off; off += gen ? blk : 0; }
  L.coef = off; off += up256((size_t)std::max<int64_t>(nband - m, 1) * m * sizeof(c128));
  L.hs = off; off += mat;
  L.ss = off; off += mat;
  L.c = off; off += mat;
  L.theta = off; off += up256((size_t)3 * m * sizeof(double));
  L.norms = off; off += up256((size_t)m * sizeof(double));
  L.info = off; off += 256;
  L.shared = off;
  // the region shared by the calls that never overlap in time; sized call by call (the split-K workspaces are not monotone)
  size_t sh = pwh_workspace_bytes(ham, m);
  for (int64_t nb : {m, 2 * m, 3 * m, nband}) sh = std::max(sh, pwh_rr_workspace_bytes(npw, nb));
  for (int64_t nb : {2 * m, 3 * m}) {
    sh = std::max(sh, pwh_dense_workspace_bytes(nb));
    sh = std::max(sh, pwh_gram_workspace_bytes(npw, nb, nb));
  }
  for (int64_t nlo = m; nlo < nband; nlo += m) sh = std::max(sh, pwh_gram_workspace_bytes(npw, nlo, m));
  L.shared_bytes = up256(sh);
  L.total = off + L.shared_bytes;
  return L;
}

}  // namespace

extern "C" size_t pwh_lobpcg_workspace_bytes(const pwh_ham* ham, int64_t nband, int64_t nblocks) {
  int64_t hi[8];
  if (!ham || nband < 1 || nblocks < 1 || nband % nblocks != 0 || pwh_ham_info(ham, hi) != PWH_OK) return 0;
  return lb_layout(ham, hi[0], nband, nband / nblocks, false).total;
}

extern "C" size_t pwh_lobpcg_gen_workspace_bytes(const pwh_ham* ham, int64_t nband, int64_t nblocks) {
  int64_t hi[8];
  if (!ham || nband < 1 || nblocks < 1 || nband % nblocks != 0 || pwh_ham_info(ham, hi) != PWH_OK) return 0;
  return lb_layout(ham, hi[0], nband, nband / nblocks, true).total;
}

// spsi == nullptr: S = I (Algorithm 11 of the norm-conserving case); otherwise the handle carries PAW blocks and every inner
// product is <., S .>: HX_SX from one set of projections, S-Deflate, S-Ortho, generalised RR, residual (H - lambda S) Psi.
static int lobpcg_impl(pwh_ham* ham, int64_t nband, int64_t nblocks, int nline, double tol, pwh_c128* psi, int64_t ld,
                       pwh_c128* hpsi, int64_t ldh, pwh_c128* spsi, int64_t lds, double* lambda, double* resid,
                       double* history, int32_t* info, void* ws, size_t ws_bytes, void* stream) {
  const bool gen = spsi != nullptr;
  int64_t hi[8];
  if (!ham || pwh_ham_info(ham, hi) != PWH_OK) return api_fail(PWH_EINVAL, "handle is null");
  const int64_t npw = hi[0];
  if (nband < 1 || nblocks < 1 || nband % nblocks != 0) return api_fail(PWH_EINVAL, "nband must be a positive multiple of nblocks");
  if (nline < 0) return api_fail(PWH_EINVAL, "nline < 0");
  if (!(tol >= 0.0)) return api_fail(PWH_EINVAL, "tol < 0");
  if (!psi || !hpsi || ld < npw || ldh < npw) return api_fail(PWH_EINVAL, "psi / hpsi null or leading dimension < npw");
  if (!lambda || !resid || !info) return api_fail(PWH_EINVAL, "lambda / resid / info null");
  const int64_t m = nband / nblocks;
  if (3 * m > npw) return api_fail(PWH_EINVAL, "3 nband / nblocks exceeds npw: the search space would be rank deficient");
  const LbWs L = lb_layout(ham, npw, nband, m, gen);
  if (!ws || (uintptr_t)ws % 256 != 0) return api_fail(PWH_EINVAL, "workspace null or not 256-byte aligned");
  if (ws_bytes < L.total) return api_fail(PWH_EINVAL, "workspace too small: %zu < %zu bytes", ws_bytes, L.total);
  cudaStream_t st = (cudaStream_t)stream;
  unsigned char* wsb = (unsigned char*)ws;
  c128* B[2] = {(c128*)(wsb + L.b[0]), (c128*)(wsb + L.b[1])};
  c128* HB[2] = {(c128*)(wsb + L.hb[0]), (c128*)(wsb + L.hb[1])};
  c128* SB[2] = {gen ? (c128*)(wsb + L.sb[0]) : nullptr, gen ? (c128*)(wsb + L.sb[1]) : nullptr};
  c128* spsi_ = reinterpret_cast<c128*>(spsi);
  c128* coef = (c128*)(wsb + L.coef);
  c128* Hs = (c128*)(wsb + L.hs);
  c128* Ss = (c128*)(wsb + L.ss);
  c128* C = (c128*)(wsb + L.c);
  double* theta = (double*)(wsb + L.theta);
  double* norms = (double*)(wsb + L.norms);
  int* sinfo = (int*)(wsb + L.info);
  void* sh = wsb + L.shared;
  const size_t shb = L.shared_bytes;
  const int64_t ldb = npw;
  const double* kin = ham_kin(ham);
  const size_t colb = (size_t)npw * sizeof(c128);
  LB_TRY(zgemm_init());
  LB_TRY(rr_kernels_init());
  LB_TRY(cudaMemsetAsync(info, 0, sizeof(int32_t), st));
  auto fold = [&](int potrf_style) {
    count_launch();
    k_info_fold<<<1, 1, 0, st>>>(sinfo, potrf_style, info);
  };
  // Algorithm 8 (S-Deflate): X <- X - Psi_0 ((S Psi_0)^H X) against the nlo bands already solved (they sit in psi / spsi)
  auto deflate = [&](c128* X, int64_t nlo) -> int {
    if (nlo == 0) return PWH_OK;
    LB_RC(pwh_gram(npw, nlo, gen ? spsi : psi, gen ? lds : ld, m, (const pwh_c128*)X, ldb, (pwh_c128*)coef, nlo, sh, shb,
                   stream));
    launch_zgemm_nn(npw, m, nlo, -1.0, (const c128*)psi, ld, coef, nlo, X, ldb, true, st);
    return PWH_OK;
  };
  auto chol = [&](int64_t n_, int64_t nb, c128* X_, c128* HX_, c128* SX_, int64_t ld_) -> int {
    if (gen)
      return pwh_chol_ortho_gen(n_, nb, (pwh_c128*)X_, ld_, (pwh_c128*)HX_, ld_, (pwh_c128*)SX_, ld_, nullptr, 0, sinfo, sh, shb,
                                stream);
    return pwh_chol_ortho(n_, nb, (pwh_c128*)X_, ld_, (pwh_c128*)HX_, ld_, nullptr, 0, sinfo, sh, shb, stream);
  };
  std::vector<double> hnorms((size_t)m);
  for (int64_t i = 0; i < nblocks; ++i) {
    const int64_t lo = i * m;
    int cur = 0;
    c128 *X = B[cur], *HX = HB[cur], *SX = SB[cur];
    // H Y (and S Y from the same projections) for m bands
    auto apply = [&](const c128* Y, c128* HY, c128* SY) -> int {
      if (gen) return pwh_apply_hs(ham, m, (const pwh_c128*)Y, ldb, (pwh_c128*)HY, ldb, (pwh_c128*)SY, ldb, sh, shb, stream);
      return pwh_apply_h(ham, m, (const pwh_c128*)Y, ldb, (pwh_c128*)HY, ldb, sh, shb, stream);
    };
    // Algorithm 9 on the first nb columns of the current basis
    auto ortho = [&](int64_t nb) -> int {
      return chol(npw, nb, X, HX, SX, ldb);
    };
    LB_TRY(cudaMemcpy2DAsync(X, colb, psi + lo * ld, (size_t)ld * sizeof(c128), colb, (size_t)m, cudaMemcpyDeviceToDevice, st));
    LB_RC(deflate(X, lo));                                                                                     // line 3
    LB_RC(apply(X, HX, SX));                                                                                   // line 6
    LB_RC(ortho(m));                                                                                           // line 8
    fold(1);
    LB_RC(pwh_rayleigh_ritz(npw, m, (pwh_c128*)X, ldb, (pwh_c128*)HX, ldb, (pwh_c128*)SX, ldb, theta, sinfo, sh, shb, stream));  // line 9
    fold(0);
    bool have_p = false;
    for (int n = 1; n <= nline; ++n) {                                                                         // line 10
      c128 *W = X + m * ldb, *HW = HX + m * ldb, *SW = gen ? SX + m * ldb : nullptr;
      {                                                                                                        // lines 11-13
        ScopedLaunch sl(ST_COLSTATS, st);
        k_residual_precond<<<(unsigned)m, LT, 0, st>>>(npw, kin, X, ldb, HX, ldb, SX, ldb, theta, W, ldb, norms);
      }
      if (history)
        LB_TRY(cudaMemcpyAsync(history + ((size_t)i * nline + (n - 1)) * m, norms, (size_t)m * sizeof(double),
                               cudaMemcpyDeviceToDevice, st));
      if (tol > 0.0) {                                                                                         // line 12
        LB_TRY(cudaMemcpyAsync(hnorms.data(), norms, (size_t)m * sizeof(double), cudaMemcpyDeviceToHost, st));
        LB_TRY(cudaStreamSynchronize(st));
        if (*std::max_element(hnorms.begin(), hnorms.end()) <= tol) break;
      }
      LB_RC(deflate(W, lo));                                                                                   // line 15
      LB_RC(apply(W, HW, SW));                                                                                 // line 18
      const int64_t nb = have_p ? 3 * m : 2 * m;
      LB_RC(ortho(nb));                                                                                        // lines 21 / 24
      fold(1);
      LB_RC(pwh_gram_herm(npw, nb, (const pwh_c128*)X, ldb, (const pwh_c128*)HX, ldb, (pwh_c128*)Hs, nb, sh, shb, stream));
      LB_RC(pwh_gram_herm(npw, nb, (const pwh_c128*)X, ldb, (const pwh_c128*)(gen ? SX : X), ldb, (pwh_c128*)Ss, nb, sh, shb,
                          stream));
      launch_hermitise((int)nb, Hs, nb, st);
      launch_hermitise((int)nb, Ss, nb, st);
      LB_RC(pwh_hegv(nb, (pwh_c128*)Hs, nb, (pwh_c128*)Ss, nb, theta, (pwh_c128*)C, nb, sinfo, sh, shb, stream));   // lines 22 / 25
      fold(0);
      // the lowest m Ritz pairs: new Psi_i = B C[:, :m]; P_i = B[:, m:] C[m:, :m]  (line 26 in the rotated basis)
      c128 *Xn = B[cur ^ 1], *HXn = HB[cur ^ 1], *SXn = SB[cur ^ 1];
      launch_zgemm_nn(npw, m, nb, 1.0, X, ldb, C, nb, Xn, ldb, false, st);
      launch_zgemm_nn(npw, m, nb, 1.0, HX, ldb, C, nb, HXn, ldb, false, st);
      launch_zgemm_nn(npw, m, nb - m, 1.0, X + m * ldb, ldb, C + m, nb, Xn + 2 * m * ldb, ldb, false, st);
      launch_zgemm_nn(npw, m, nb - m, 1.0, HX + m * ldb, ldb, C + m, nb, HXn + 2 * m * ldb, ldb, false, st);
      if (gen) {
        launch_zgemm_nn(npw, m, nb, 1.0, SX, ldb, C, nb, SXn, ldb, false, st);
        launch_zgemm_nn(npw, m, nb - m, 1.0, SX + m * ldb, ldb, C + m, nb, SXn + 2 * m * ldb, ldb, false, st);
      }
      cur ^= 1;
      X = Xn; HX = HXn; SX = SXn;
      have_p = true;
    }
    LB_TRY(cudaMemcpy2DAsync(psi + lo * ld, (size_t)ld * sizeof(c128), X, colb, colb, (size_t)m, cudaMemcpyDeviceToDevice, st));
    LB_TRY(cudaMemcpy2DAsync(hpsi + lo * ldh, (size_t)ldh * sizeof(c128), HX, colb, colb, (size_t)m, cudaMemcpyDeviceToDevice, st));
    if (gen)
      LB_TRY(cudaMemcpy2DAsync(spsi_ + lo * lds, (size_t)lds * sizeof(c128), SX, colb, colb, (size_t)m, cudaMemcpyDeviceToDevice,
                               st));
    LB_TRY(cudaMemcpyAsync(lambda + lo, theta, (size_t)m * sizeof(double), cudaMemcpyDeviceToDevice, st));
  }
  if (nblocks > 1) {                                                                                           // lines 31-34
    if (gen) LB_RC(pwh_chol_ortho_gen(npw, nband, psi, ld, hpsi, ldh, spsi, lds, nullptr, 0, sinfo, sh, shb, stream));
    else LB_RC(pwh_chol_ortho(npw, nband, psi, ld, hpsi, ldh, nullptr, 0, sinfo, sh, shb, stream));
    fold(1);
    LB_RC(pwh_rayleigh_ritz(npw, nband, psi, ld, hpsi, ldh, spsi, lds, lambda, sinfo, sh, shb, stream));
    fold(0);
  }
  launch_residual(npw, nband, gen ? (const c128*)spsi : (const c128*)psi, gen ? lds : ld, (const c128*)hpsi, ldh, lambda, nullptr,
                  0, resid, st);                                                                               // line 29
  LB_TRY(cudaGetLastError());
  return PWH_OK;
}

extern "C" int pwh_lobpcg(pwh_ham* ham, int64_t nband, int64_t nblocks, int nline, double tol, pwh_c128* psi, int64_t ld,
                          pwh_c128* hpsi, int64_t ldh, double* lambda, double* resid, double* history, int32_t* info,
                          void* ws, size_t ws_bytes, void* stream) {
  return lobpcg_impl(ham, nband, nblocks, nline, tol, psi, ld, hpsi, ldh, nullptr, 0, lambda, resid, history, info, ws, ws_bytes,
                     stream);
}

extern "C" int pwh_lobpcg_gen(pwh_ham* ham, int64_t nband, int64_t nblocks, int nline, double tol, pwh_c128* psi, int64_t ld,
                              pwh_c128* hpsi, int64_t ldh, pwh_c128* spsi, int64_t lds, double* lambda, double* resid,
                              double* history, int32_t* info, void* ws, size_t ws_bytes, void* stream) {
  int64_t hi[8];
  if (!ham || pwh_ham_info(ham, hi) != PWH_OK) return api_fail(PWH_EINVAL, "handle is null");
  if (!spsi || lds < hi[0]) return api_fail(PWH_EINVAL, "spsi null or leading dimension < npw");
  return lobpcg_impl(ham, nband, nblocks, nline, tol, psi, ld, hpsi, ldh, spsi, lds, lambda, resid, history, info, ws, ws_bytes,
                     stream);
}
