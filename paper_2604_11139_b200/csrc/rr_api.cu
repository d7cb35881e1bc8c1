// rr_api.cu -- C ABI of the Rayleigh-Ritz companion steps (include/pwham.h, second half): argument checks, workspace
// carving and launch sequences.  The N x M work runs on the ZGEMM kernels of zgemm.cu, the M x M work and the column
// statistics on the kernels of rr.cu.  Written on top of the public entry points of pwham.cu; no CPU fallback.
#include "../../include/pwham.h"

#include <algorithm>
#include <cstdint>

#include "launch.h"

using namespace pwh;

#define RR_TRY(expr)                                                                                      \
  do {                                                                                                    \
    cudaError_t e__ = (expr);                                                                             \
    if (e__ != cudaSuccess) return api_fail(PWH_ECUDA, "%s: %s", #expr, cudaGetErrorString(e__));        \
  } while (0)

static size_t up256(size_t v) { return (v + 255) / 256 * 256; }

// rows of an N x m block rotated at a time by rotate_inplace: a panel of at most 256 MB, a multiple of the ZGEMM tile
static int64_t panel_rows(int64_t npw, int64_t m) {
  int64_t rp = (int64_t)((256u << 20) / (16 * std::max<int64_t>(m, 1)));
  rp = std::max<int64_t>(128, rp / 128 * 128);
  return std::min(rp, (npw + 127) / 128 * 128);
}

// X <- X Q for an npw x m block X and an m x m matrix Q, through a row panel (a GEMM cannot run in place)
static int rotate_inplace(int64_t npw, int64_t m, c128* X, int64_t ldx, const c128* Q, int64_t ldq, c128* panel,
                          cudaStream_t st) {
  const int64_t rp = panel_rows(npw, m);
  for (int64_t r0 = 0; r0 < npw; r0 += rp) {
    const int64_t nr = std::min(rp, npw - r0);
    launch_zgemm_nn(nr, m, m, 1.0, X + r0, ldx, Q, ldq, panel, rp, false, st);
    RR_TRY(cudaMemcpy2DAsync(X + r0, (size_t)ldx * sizeof(c128), panel, (size_t)rp * sizeof(c128), (size_t)nr * sizeof(c128),
                             (size_t)m, cudaMemcpyDeviceToDevice, st));
  }
  RR_TRY(cudaGetLastError());
  return PWH_OK;
}

static int check_block(const void* p, int64_t ld, int64_t npw, const char* name) {
  if (!p) return api_fail(PWH_EINVAL, "%s is null", name);
  if (ld < npw) return api_fail(PWH_EINVAL, "%s: leading dimension smaller than npw", name);
  return PWH_OK;
}

static int check_ws(const void* ws, size_t have, size_t need) {
  if (!ws || (uintptr_t)ws % 256 != 0) return api_fail(PWH_EINVAL, "workspace null or not 256-byte aligned");
  if (have < need) return api_fail(PWH_EINVAL, "workspace too small: %zu < %zu bytes", have, need);
  return PWH_OK;
}

extern "C" int pwh_rayleigh_quotients(int64_t npw, int64_t nband, const pwh_c128* psi, int64_t ld, const pwh_c128* hpsi,
                                      int64_t ldh, const pwh_c128* spsi, int64_t lds, double* lambda, double* minmax,
                                      void* stream) {
  if (npw < 1 || nband < 0) return api_fail(PWH_EINVAL, "bad sizes");
  if (nband == 0) return PWH_OK;
  int rc;
  if ((rc = check_block(psi, ld, npw, "psi")) || (rc = check_block(hpsi, ldh, npw, "hpsi"))) return rc;
  if (spsi && lds < npw) return api_fail(PWH_EINVAL, "spsi: leading dimension smaller than npw");
  if (!lambda) return api_fail(PWH_EINVAL, "lambda is null");
  launch_rayleigh(npw, nband, (const c128*)psi, ld, (const c128*)hpsi, ldh, (const c128*)spsi, lds, lambda, nullptr, minmax,
                  (cudaStream_t)stream);
  RR_TRY(cudaGetLastError());
  return PWH_OK;
}

extern "C" int pwh_residual_norms(int64_t npw, int64_t nband, const pwh_c128* psi, int64_t ld, const pwh_c128* hpsi,
                                  int64_t ldh, const pwh_c128* spsi, int64_t lds, const double* lambda, pwh_c128* W,
                                  int64_t ldw, double* norms, void* stream) {
  if (npw < 1 || nband < 0) return api_fail(PWH_EINVAL, "bad sizes");
  if (nband == 0) return PWH_OK;
  int rc;
  if ((rc = check_block(psi, ld, npw, "psi")) || (rc = check_block(hpsi, ldh, npw, "hpsi"))) return rc;
  if (spsi && lds < npw) return api_fail(PWH_EINVAL, "spsi: leading dimension smaller than npw");
  if (W && ldw < npw) return api_fail(PWH_EINVAL, "W: leading dimension smaller than npw");
  if (!lambda || !norms) return api_fail(PWH_EINVAL, "lambda / norms null");
  // W = H psi - lambda S psi: the kernel's "psi" operand is S psi for the generalised problem
  launch_residual(npw, nband, spsi ? (const c128*)spsi : (const c128*)psi, spsi ? lds : ld, (const c128*)hpsi, ldh, lambda,
                  (c128*)W, ldw, norms, (cudaStream_t)stream);
  RR_TRY(cudaGetLastError());
  return PWH_OK;
}

extern "C" int pwh_rotate(int64_t npw, int64_t m, const pwh_c128* X, int64_t ldx, int64_t n, const pwh_c128* Q, int64_t ldq,
                          pwh_c128* Y, int64_t ldy, void* stream) {
  if (npw < 1 || m < 1 || n < 0) return api_fail(PWH_EINVAL, "bad sizes");
  if (n == 0) return PWH_OK;
  int rc;
  if ((rc = check_block(X, ldx, npw, "X")) || (rc = check_block(Y, ldy, npw, "Y"))) return rc;
  if (!Q || ldq < m) return api_fail(PWH_EINVAL, "Q null or ldq < m");
  const uintptr_t x0 = (uintptr_t)X, x1 = x0 + ((size_t)(m - 1) * ldx + npw) * sizeof(c128);
  const uintptr_t y0 = (uintptr_t)Y, y1 = y0 + ((size_t)(n - 1) * ldy + npw) * sizeof(c128);
  if (x0 < y1 && y0 < x1) return api_fail(PWH_EINVAL, "X and Y overlap");
  RR_TRY(zgemm_init());
  launch_zgemm_nn(npw, n, m, 1.0, (const c128*)X, ldx, (const c128*)Q, ldq, (c128*)Y, ldy, false, (cudaStream_t)stream);
  RR_TRY(cudaGetLastError());
  return PWH_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// dense n x n steps
// ---------------------------------------------------------------------------------------------------------------
struct DenseWs {
  size_t w, t, c, jac, part, info, total;
};
static DenseWs dense_layout(int64_t n) {
  DenseWs d;
  const size_t mat = up256((size_t)n * n * sizeof(c128));
  size_t off = 0;
  d.w = off; off += mat;
  d.t = off; off += mat;
  d.c = off; off += mat;
  d.jac = off; off += up256(jacobi_scratch_bytes((int)n));
  d.part = off; off += up256(std::max(zgemm_cn_workspace(n, n, n, false), zgemm_cn_workspace(n, n, n, true)));
  d.info = off; off += 256;
  d.total = off;
  return d;
}

extern "C" size_t pwh_dense_workspace_bytes(int64_t n) { return n < 1 ? 256 : dense_layout(n).total; }

static int check_dense(int64_t n, const void* A, int64_t lda, const char* name) {
  if (n < 1 || n > 16384) return api_fail(PWH_EINVAL, "matrix order out of range (1..16384)");
  if (!A || lda < n) return api_fail(PWH_EINVAL, "%s null or leading dimension < n", name);
  return PWH_OK;
}

extern "C" int pwh_potrf(int64_t n, pwh_c128* A, int64_t lda, int32_t* info, void* stream) {
  int rc;
  if ((rc = check_dense(n, A, lda, "A"))) return rc;
  if (!info) return api_fail(PWH_EINVAL, "info is null");
  launch_potrf_upper((int)n, (c128*)A, lda, info, (cudaStream_t)stream);
  RR_TRY(cudaGetLastError());
  return PWH_OK;
}

static int heev_impl(int64_t n, c128* A, int64_t lda, double* w, c128* X, int64_t ldx, int32_t* info, unsigned char* ws,
                     const DenseWs& d, cudaStream_t st) {
  RR_TRY(rr_kernels_init());
  launch_hermitise((int)n, A, lda, st);
  RR_TRY(launch_heev_jacobi((int)n, A, lda, w, X, ldx, info, ws + d.jac, st));
  return PWH_OK;
}

extern "C" int pwh_heev(int64_t n, pwh_c128* A, int64_t lda, double* w, pwh_c128* X, int64_t ldx, int32_t* info, void* ws,
                        size_t ws_bytes, void* stream) {
  int rc;
  if ((rc = check_dense(n, A, lda, "A")) || (rc = check_dense(n, X, ldx, "X"))) return rc;
  if (!w || !info) return api_fail(PWH_EINVAL, "w / info null");
  const DenseWs d = dense_layout(n);
  if ((rc = check_ws(ws, ws_bytes, d.total))) return rc;
  return heev_impl(n, (c128*)A, lda, w, (c128*)X, ldx, info, (unsigned char*)ws, d, (cudaStream_t)stream);
}

// A X = B X diag(w), X^H B X = I:  B = U^H U,  W = U^-1,  C = W^H A W,  C Y = Y diag(w),  X = W Y
static int hegv_impl(int64_t n, c128* A, int64_t lda, c128* B, int64_t ldb, double* w, c128* X, int64_t ldx, int32_t* info,
                     unsigned char* ws, const DenseWs& d, cudaStream_t st) {
  RR_TRY(zgemm_init());
  RR_TRY(rr_kernels_init());
  c128* W = (c128*)(ws + d.w);
  c128* T = (c128*)(ws + d.t);
  c128* C = (c128*)(ws + d.c);
  int* pinfo = (int*)(ws + d.info);
  launch_potrf_upper((int)n, B, ldb, pinfo, st);
  launch_trinv_upper((int)n, B, ldb, W, n, st);
  launch_zgemm_nn(n, n, n, 1.0, A, lda, W, n, T, n, false, st);                       // T = A W
  launch_zgemm_cn(n, n, n, W, n, T, n, nullptr, C, n, ws + d.part, st, nullptr, true);  // C = W^H T (Hermitian)
  launch_hermitise((int)n, C, n, st);
  RR_TRY(launch_heev_jacobi((int)n, C, n, w, T, n, info, ws + d.jac, st));            // eigenvectors Y in T
  launch_zgemm_nn(n, n, n, 1.0, W, n, T, n, X, ldx, false, st);                        // X = W Y
  launch_merge_info(pinfo, info, st);
  RR_TRY(cudaGetLastError());
  return PWH_OK;
}

extern "C" int pwh_hegv(int64_t n, pwh_c128* A, int64_t lda, pwh_c128* B, int64_t ldb, double* w, pwh_c128* X, int64_t ldx,
                        int32_t* info, void* ws, size_t ws_bytes, void* stream) {
  int rc;
  if ((rc = check_dense(n, A, lda, "A")) || (rc = check_dense(n, B, ldb, "B")) || (rc = check_dense(n, X, ldx, "X"))) return rc;
  if (!w || !info) return api_fail(PWH_EINVAL, "w / info null");
  const DenseWs d = dense_layout(n);
  if ((rc = check_ws(ws, ws_bytes, d.total))) return rc;
  return hegv_impl(n, (c128*)A, lda, (c128*)B, ldb, w, (c128*)X, ldx, info, (unsigned char*)ws, d, (cudaStream_t)stream);
}

// ---------------------------------------------------------------------------------------------------------------
// N x M steps: Cholesky orthonormalisation (Algorithm 9), Rayleigh-Ritz (Algorithm 10), one ChebFi iteration (Algorithm 12)
// ---------------------------------------------------------------------------------------------------------------
struct RrWs {
  size_t hs, ss, x, panel, gram, dense, total;
  DenseWs d;
};
static RrWs rr_layout(int64_t npw, int64_t m) {
  RrWs r;
  r.d = dense_layout(m);
  const size_t mat = up256((size_t)m * m * sizeof(c128));
  size_t off = 0;
  r.hs = off; off += mat;
  r.ss = off; off += mat;
  r.x = off; off += mat;
  r.panel = off; off += up256((size_t)panel_rows(npw, m) * m * sizeof(c128));
  r.gram = off; off += up256(pwh_gram_workspace_bytes(npw, m, m));
  r.dense = off; off += r.d.total;
  r.total = off;
  return r;
}

extern "C" size_t pwh_rr_workspace_bytes(int64_t npw, int64_t nband) {
  if (npw < 1 || nband < 1) return 256;
  return rr_layout(npw, nband).total;
}

static int chol_ortho_impl(int64_t npw, int64_t nband, pwh_c128* psi, int64_t ld, pwh_c128* hpsi, int64_t ldh, pwh_c128* spsi,
                           int64_t lds, pwh_c128* U, int64_t ldu, int32_t* info, void* ws, size_t ws_bytes, void* stream) {
  if (npw < 1 || nband < 0) return api_fail(PWH_EINVAL, "bad sizes");
  if (nband == 0) return PWH_OK;
  int rc;
  if ((rc = check_block(psi, ld, npw, "psi"))) return rc;
  if (hpsi && ldh < npw) return api_fail(PWH_EINVAL, "hpsi: leading dimension smaller than npw");
  if (spsi && lds < npw) return api_fail(PWH_EINVAL, "spsi: leading dimension smaller than npw");
  if (U && ldu < nband) return api_fail(PWH_EINVAL, "ldu < nband");
  if (!info) return api_fail(PWH_EINVAL, "info is null");
  const RrWs r = rr_layout(npw, nband);
  if ((rc = check_ws(ws, ws_bytes, r.total))) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  unsigned char* wsb = (unsigned char*)ws;
  c128* S = (c128*)(wsb + r.ss);
  c128* W = (c128*)(wsb + r.x);
  RR_TRY(rr_kernels_init());
  // S_Psi = Psi^H (S Psi) (Hermitian; S = I when spsi is null), S_Psi = U^H U, W = U^-1, then Psi, H Psi, S Psi <- . W
  if ((rc = pwh_gram_herm(npw, nband, psi, ld, spsi ? spsi : psi, spsi ? lds : ld, (pwh_c128*)S, nband, wsb + r.gram,
                          r.total - r.gram, stream))) return rc;
  launch_potrf_upper((int)nband, S, nband, info, st);
  if (U) RR_TRY(cudaMemcpy2DAsync(U, (size_t)ldu * sizeof(c128), S, (size_t)nband * sizeof(c128), (size_t)nband * sizeof(c128),
                                  (size_t)nband, cudaMemcpyDeviceToDevice, st));
  launch_trinv_upper((int)nband, S, nband, W, nband, st);
  if ((rc = rotate_inplace(npw, nband, (c128*)psi, ld, W, nband, (c128*)(wsb + r.panel), st))) return rc;
  if (hpsi && (rc = rotate_inplace(npw, nband, (c128*)hpsi, ldh, W, nband, (c128*)(wsb + r.panel), st))) return rc;
  if (spsi && (rc = rotate_inplace(npw, nband, (c128*)spsi, lds, W, nband, (c128*)(wsb + r.panel), st))) return rc;
  return PWH_OK;
}

extern "C" int pwh_chol_ortho(int64_t npw, int64_t nband, pwh_c128* psi, int64_t ld, pwh_c128* hpsi, int64_t ldh,
                              pwh_c128* U, int64_t ldu, int32_t* info, void* ws, size_t ws_bytes, void* stream) {
  return chol_ortho_impl(npw, nband, psi, ld, hpsi, ldh, nullptr, 0, U, ldu, info, ws, ws_bytes, stream);
}

extern "C" int pwh_chol_ortho_gen(int64_t npw, int64_t nband, pwh_c128* psi, int64_t ld, pwh_c128* hpsi, int64_t ldh,
                                  pwh_c128* spsi, int64_t lds, pwh_c128* U, int64_t ldu, int32_t* info, void* ws,
                                  size_t ws_bytes, void* stream) {
  if (!spsi) return api_fail(PWH_EINVAL, "spsi is null");
  return chol_ortho_impl(npw, nband, psi, ld, hpsi, ldh, spsi, lds, U, ldu, info, ws, ws_bytes, stream);
}

extern "C" int pwh_rayleigh_ritz(int64_t npw, int64_t nband, pwh_c128* psi, int64_t ld, pwh_c128* hpsi, int64_t ldh,
                                 pwh_c128* spsi, int64_t lds, double* lambda, int32_t* info, void* ws, size_t ws_bytes,
                                 void* stream) {
  if (npw < 1 || nband < 0) return api_fail(PWH_EINVAL, "bad sizes");
  if (nband == 0) return PWH_OK;
  int rc;
  if ((rc = check_block(psi, ld, npw, "psi")) || (rc = check_block(hpsi, ldh, npw, "hpsi"))) return rc;
  if (spsi && lds < npw) return api_fail(PWH_EINVAL, "spsi: leading dimension smaller than npw");
  if (!lambda || !info) return api_fail(PWH_EINVAL, "lambda / info null");
  const RrWs r = rr_layout(npw, nband);
  if ((rc = check_ws(ws, ws_bytes, r.total))) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  unsigned char* wsb = (unsigned char*)ws;
  c128* Hs = (c128*)(wsb + r.hs);
  c128* Ss = (c128*)(wsb + r.ss);
  c128* X = (c128*)(wsb + r.x);
  // H_Psi = Psi^H (H Psi), S_Psi = Psi^H (S Psi)  (Algorithm 10 steps 1-2), both Hermitian
  if ((rc = pwh_gram_herm(npw, nband, psi, ld, hpsi, ldh, (pwh_c128*)Hs, nband, wsb + r.gram, r.total - r.gram, stream))) return rc;
  if ((rc = pwh_gram_herm(npw, nband, psi, ld, spsi ? spsi : psi, spsi ? lds : ld, (pwh_c128*)Ss, nband, wsb + r.gram,
                          r.total - r.gram, stream))) return rc;
  launch_hermitise((int)nband, Hs, nband, st);
  launch_hermitise((int)nband, Ss, nband, st);
  // H_Psi X = S_Psi X Lambda  (step 3)
  if ((rc = hegv_impl(nband, Hs, nband, Ss, nband, lambda, X, nband, info, wsb + r.dense, r.d, st))) return rc;
  // Psi <- Psi X, H Psi <- (H Psi) X, S Psi <- (S Psi) X  (steps 4-6)
  if ((rc = rotate_inplace(npw, nband, (c128*)psi, ld, X, nband, (c128*)(wsb + r.panel), st))) return rc;
  if ((rc = rotate_inplace(npw, nband, (c128*)hpsi, ldh, X, nband, (c128*)(wsb + r.panel), st))) return rc;
  if (spsi && (rc = rotate_inplace(npw, nband, (c128*)spsi, lds, X, nband, (c128*)(wsb + r.panel), st))) return rc;
  return PWH_OK;
}

extern "C" size_t pwh_chebfi_workspace_bytes(const pwh_ham* ham, int64_t nband, int64_t block) {
  int64_t info[8];
  if (!ham || nband < 1 || pwh_ham_info(ham, info) != PWH_OK) return 0;
  if (block <= 0 || block > nband) block = nband;
  return std::max(pwh_workspace_bytes(ham, block), pwh_rr_workspace_bytes(info[0], nband)) + 256;
}

extern "C" int pwh_chebfi_iteration(pwh_ham* ham, int64_t nband, int64_t block, pwh_c128* psi, int64_t ld, pwh_c128* hpsi,
                                    int64_t ldh, pwh_c128* spsi, int64_t lds, int degree, double b, double a0_margin,
                                    double* lambda, double* resid, double* bounds_host, int32_t* info, void* ws,
                                    size_t ws_bytes, void* stream) {
  int64_t hi[8];
  if (!ham || pwh_ham_info(ham, hi) != PWH_OK) return api_fail(PWH_EINVAL, "handle is null");
  const int64_t npw = hi[0];
  if (nband < 1) return api_fail(PWH_EINVAL, "nband < 1");
  if (degree < 1) return api_fail(PWH_EINVAL, "degree < 1");
  if (!(a0_margin >= 0.0)) return api_fail(PWH_EINVAL, "a0_margin < 0");
  int rc;
  if ((rc = check_block(psi, ld, npw, "psi")) || (rc = check_block(hpsi, ldh, npw, "hpsi"))) return rc;
  if (spsi && lds < npw) return api_fail(PWH_EINVAL, "spsi: leading dimension smaller than npw");
  if (!lambda || !resid || !info) return api_fail(PWH_EINVAL, "lambda / resid / info null");
  if (block <= 0 || block > nband) block = nband;
  const size_t need = pwh_chebfi_workspace_bytes(ham, nband, block);
  if ((rc = check_ws(ws, ws_bytes, need))) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  unsigned char* wsb = (unsigned char*)ws;
  double* d_minmax = (double*)(wsb + need - 256);
  // H Psi (and S Psi: HX_SX) in column blocks
  auto hx_sx = [&]() -> int {
    for (int64_t b0 = 0; b0 < nband; b0 += block) {
      const int64_t nb = std::min(block, nband - b0);
      const int r = spsi ? pwh_apply_hs(ham, nb, psi + b0 * ld, ld, hpsi + b0 * ldh, ldh, spsi + b0 * lds, lds, ws, need - 256, stream)
                         : pwh_apply_h(ham, nb, psi + b0 * ld, ld, hpsi + b0 * ldh, ldh, ws, need - 256, stream);
      if (r) return r;
    }
    return PWH_OK;
  };
  // lines 1-2
  if ((rc = hx_sx())) return rc;
  // line 3: Rayleigh quotients, their minimum and maximum -> the filter's interval (the one host round trip of the iteration)
  launch_rayleigh(npw, nband, (const c128*)psi, ld, (const c128*)hpsi, ldh, (const c128*)spsi, lds, lambda, nullptr, d_minmax, st);
  double mm[2];
  RR_TRY(cudaMemcpyAsync(mm, d_minmax, sizeof(mm), cudaMemcpyDeviceToHost, st));
  RR_TRY(cudaStreamSynchronize(st));
  const double a = mm[1], a0 = mm[0] - a0_margin;
  if (bounds_host) { bounds_host[0] = a0; bounds_host[1] = a; }
  if (!(b > a) || !(a0 < a))
    return api_fail(PWH_EINVAL, "Rayleigh quotients span [%g, %g]: need min - a0_margin < max < b = %g", mm[0], mm[1], b);
  // lines 4-8: the filter (of S^-1 H when the overlap is not the identity)
  for (int64_t b0 = 0; b0 < nband; b0 += block) {
    const int64_t nb = std::min(block, nband - b0);
    rc = spsi ? pwh_cheb_filter_gen(ham, nb, psi + b0 * ld, ld, degree, a, b, a0, ws, need - 256, stream)
              : pwh_cheb_filter(ham, nb, psi + b0 * ld, ld, degree, a, b, a0, ws, need - 256, stream);
    if (rc) return rc;
  }
  if ((rc = hx_sx())) return rc;
  // line 10: Rayleigh-Ritz; lines 11-12: residuals
  if ((rc = pwh_rayleigh_ritz(npw, nband, psi, ld, hpsi, ldh, spsi, lds, lambda, info, ws, need - 256, stream))) return rc;
  launch_residual(npw, nband, spsi ? (const c128*)spsi : (const c128*)psi, spsi ? lds : ld, (const c128*)hpsi, ldh, lambda,
                  nullptr, 0, resid, st);
  RR_TRY(cudaGetLastError());
  return PWH_OK;
}
