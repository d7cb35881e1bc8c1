// launch.h -- internal launcher declarations shared by the libpwham translation units.
#pragma once
#include "common.cuh"

struct pwh_ham;   // the opaque handle of include/pwham.h (defined in pwham.cu)

namespace pwh {

void count_launch();

// Stage ids reported by pwh_profile_end (same order as PWH_STAGE_* in include/pwham.h).
enum { ST_SCATTER_ZINV = 0, ST_PLANE = 1, ST_ZFWD_GATHER = 2, ST_ZGEMM_CN = 3, ST_SPLITK = 4, ST_ZGEMM_NN = 5,
       ST_COLSTATS = 6, ST_SMALL = 7, ST_JACOBI = 8, ST_AXPY = 9 };
// Counts one kernel launch and, while profiling is on, brackets it with a cudaEvent pair on `st`.
class ScopedLaunch {
 public:
  ScopedLaunch(int stage, cudaStream_t st);
  ~ScopedLaunch();
 private:
  cudaStream_t st_;
  int64_t idx_;
};

// local_kernels.cu
size_t zkernel_smem(const LocalPlan& P);
size_t plane_smem(const LocalPlan& P);
cudaError_t local_kernels_init(const LocalPlan& P);
void launch_scatter_zinv(const LocalPlan& P, const c128* psi, int64_t ldpsi, c128* colbuf, int nb, cudaStream_t st);
void launch_plane(const LocalPlan& P, c128* colbuf, int nb, cudaStream_t st);
void launch_zfwd_gather(const LocalPlan& P, const c128* colbuf, const c128* y, int64_t ldy, const c128* yprev,
                        int64_t ldprev, c128* out, int64_t ldout, double alpha, double cshift, double beta, int nb,
                        cudaStream_t st);

void launch_density_plane(const LocalPlan& P, const c128* colbuf, int nb, const double* occ, double* acc, cudaStream_t st);
void launch_density_unpermute(const LocalPlan& P, const double* acc, const int* natx, const int* naty, const int* natz,
                              double weight, double* rho, cudaStream_t st);

// local_fast.cu
size_t fast_zkernel_smem(const FastPlan& P);
size_t fast_plane_smem(const FastPlan& P);
cudaError_t fast_kernels_init(const FastPlan& P);
void launch_fast_scatter_zinv(const FastPlan& P, const c128* psi, int64_t ldpsi, c128* colbuf, int nb, cudaStream_t st);
void launch_fast_plane(const FastPlan& P, c128* colbuf, int nb, cudaStream_t st);
void launch_fast_zfwd_gather(const FastPlan& P, const c128* colbuf, const c128* y, int64_t ldy, const c128* yprev,
                             int64_t ldprev, c128* out, int64_t ldout, double alpha, double cshift, double beta, int nb,
                             cudaStream_t st);

void launch_fast_density_plane(const FastPlan& P, const c128* colbuf, int nb, const double* occ, double* acc, cudaStream_t st);
void launch_fast_density_unslot(const FastPlan& P, const double* acc, double weight, double* rho, cudaStream_t st);

// local_v2.cu
bool v2_select(V2Plan& P, int n1, int n2, int nxl, int nyl, size_t smem_max, bool no_prune = false);
cudaError_t v2_kernels_init(const V2Plan& P);
void launch_v2_perm_vloc(const V2Plan& P, int r1z, int r2z, const double* vloc, double* out, cudaStream_t st);
void launch_v2_plane(const V2Plan& P, c128* colbuf, int nb, cudaStream_t st);

// local_z.cu
size_t zw_smem(const ZPlan& P);
int zw_pruned_len(int r1);   // rows of the pruned instantiation of a radix-r1 strided-role pass
cudaError_t zw_kernels_init(const ZPlan& P);
void launch_zw_scatter_zinv(const ZPlan& P, const c128* psi, int64_t ldpsi, c128* colbuf, int nb, cudaStream_t st);
void launch_zw_zfwd_gather(const ZPlan& P, const c128* colbuf, const c128* y, int64_t ldy, const c128* yprev,
                           int64_t ldprev, c128* out, int64_t ldout, double alpha, double cshift, double beta, int nb,
                           cudaStream_t st);

// zgemm.cu
cudaError_t zgemm_init();
// tests only: PWH_ZGEMM_NO_TMA=1, sampled by pwh_ham_setup, routes every ZGEMM through the cp.async kernels
void zgemm_set_no_tma(bool off);
// the two TMA descriptors of a handle's projector matrix (opaque 128-byte CUtensorMap images), encoded once at setup
struct ProjMaps {
  alignas(64) unsigned char cn[128];    // P as the A operand of C = P^H Y (boxes of 128 projectors)
  alignas(64) unsigned char cnb[128];   // P as the B operand of the exchanged product (Y^H P)^H (boxes of 64 projectors)
  alignas(64) unsigned char nn[128];
  bool ok = false;
};
void zgemm_make_proj_maps(ProjMaps& pm, const c128* P, int64_t npw, int64_t nproj, int64_t ldp);
// runs `ctas` CTAs x 8 warps x iters x 32 DMMA.8x8x4 (512 flop each) and returns the elapsed milliseconds
cudaError_t dmma_probe(int iters, int ctas, double* sink, cudaStream_t st, float* ms);
// number of K splits chosen for C(M x N) = A^H B with K = npw (herm: only the block upper triangle is computed)
int zgemm_cn_splits(int64_t M, int64_t N, int64_t K, bool herm);
size_t zgemm_cn_workspace(int64_t M, int64_t N, int64_t K, bool herm);
size_t zgemm_cn_workspace_upto(int64_t M, int64_t N, int64_t K);   // max over n <= N (non-Hermitian)
// C[m + n*ldc] = scale[m] * sum_k conj(A[k + m*lda]) * B[k + n*ldb]      (scale may be null; pmA: cached maps of A = P;
// herm: the caller asserts C is Hermitian (M == N), half of the tiles are computed and mirrored)
void launch_zgemm_cn(int64_t M, int64_t N, int64_t K, const c128* A, int64_t lda, const c128* B, int64_t ldb,
                     const double* scale, c128* C, int64_t ldc, void* ws, cudaStream_t st, const ProjMaps* pmA = nullptr,
                     bool herm = false);
// C[m + n*ldc] = alpha * sum_k A[m + k*lda] * B[k + n*ldb]  (+ C[m + n*ldc] when accumulate)
void launch_zgemm_nn(int64_t M, int64_t N, int64_t K, double alpha, const c128* A, int64_t lda, const c128* B,
                     int64_t ldb, c128* C, int64_t ldc, bool accumulate, cudaStream_t st, const ProjMaps* pmA = nullptr);

// rr.cu -- Rayleigh-Ritz companion kernels (all pointers device)
cudaError_t rr_kernels_init();
void launch_rayleigh(int64_t npw, int64_t nband, const c128* psi, int64_t ld, const c128* hpsi, int64_t ldh,
                     const c128* spsi, int64_t lds, double* lambda, double* nrm2, double* minmax, cudaStream_t st);
void launch_residual(int64_t npw, int64_t nband, const c128* psi, int64_t ld, const c128* hpsi, int64_t ldh,
                     const double* lambda, c128* W, int64_t ldw, double* norms, cudaStream_t st);
void launch_potrf_upper(int n, c128* A, int64_t lda, int* info, cudaStream_t st);
void launch_trinv_upper(int n, const c128* U, int64_t ldu, c128* W, int64_t ldw, cudaStream_t st);
void launch_hermitise(int n, c128* A, int64_t lda, cudaStream_t st);
void launch_merge_info(const int* potrf_info, int* info, cudaStream_t st);
size_t jacobi_scratch_bytes(int n);
cudaError_t launch_heev_jacobi(int n, c128* A, int64_t lda, double* w, c128* X, int64_t ldx, int* sweeps, void* scratch,
                               cudaStream_t st);

// paw.cu -- PAW-style generalised problem: block-diagonal D / Q, helpers for K of S^-1 = I - P K P^H, filter axpy
void launch_blockdiag_apply(int64_t nproj, int64_t nband, const int* blk_of, const int* blk_lo, const int64_t* boff,
                            const c128* blocks, const c128* in, int64_t ldi, c128* out, int64_t ldo, cudaStream_t st);
void launch_blocks_to_dense(int64_t nproj, const int* blk_of, const int* blk_lo, const int64_t* boff, const c128* blocks,
                            c128* out, int64_t ldo, cudaStream_t st);
void launch_conj_transpose(int n, const c128* in, int64_t ldi, c128* out, int64_t ldo, cudaStream_t st);
// A <- alpha A + beta B + gamma I  (B may be null)
void launch_mat_axpby(int n, double alpha, c128* A, int64_t lda, double beta, const c128* B, int64_t ldb, double gamma,
                      cudaStream_t st);
// out = alpha (z - c y) - beta yprev  (yprev may be null; out may alias z or yprev)
void launch_cheb_axpy(int64_t npw, int64_t nband, const c128* z, int64_t ldz, const c128* y, int64_t ldy, const c128* yprev,
                      int64_t ldp, c128* out, int64_t ldo, double alpha, double cshift, double beta, cudaStream_t st);

// pwham.cu: the kinetic diagonal kin[npw] of a handle (device pointer)
const double* ham_kin(const ::pwh_ham* ham);

// pwham.cu: records the thread-local error message of the C ABI and returns `code`
int api_fail(int code, const char* fmt, ...);

// pwham.cu: raises the dynamic shared-memory limit of a kernel to the device's opt-in maximum.  The attribute is
// process-global per kernel, so it is set to the maximum once rather than to one handle's need.
cudaError_t set_max_dyn_smem(const void* func);

}  // namespace pwh
