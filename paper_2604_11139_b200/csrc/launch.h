// launch.h -- internal launcher declarations shared by the libpwham translation units.
#pragma once
#include "common.cuh"

namespace pwh {

void count_launch();

// Stage ids reported by pwh_profile_end (same order as PWH_STAGE_* in include/pwham.h).
enum { ST_SCATTER_ZINV = 0, ST_PLANE = 1, ST_ZFWD_GATHER = 2, ST_ZGEMM_CN = 3, ST_SPLITK = 4, ST_ZGEMM_NN = 5 };
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

// local_fast.cu
size_t fast_zkernel_smem(const FastPlan& P);
size_t fast_plane_smem(const FastPlan& P);
cudaError_t fast_kernels_init(const FastPlan& P);
void launch_fast_scatter_zinv(const FastPlan& P, const c128* psi, int64_t ldpsi, c128* colbuf, int nb, cudaStream_t st);
void launch_fast_plane(const FastPlan& P, c128* colbuf, int nb, cudaStream_t st);
void launch_fast_zfwd_gather(const FastPlan& P, const c128* colbuf, const c128* y, int64_t ldy, const c128* yprev,
                             int64_t ldprev, c128* out, int64_t ldout, double alpha, double cshift, double beta, int nb,
                             cudaStream_t st);

// local_v2.cu
bool v2_select(V2Plan& P, int n1, int n2, int nxl, size_t smem_max);
cudaError_t v2_kernels_init(const V2Plan& P);
void launch_v2_perm_vloc(const V2Plan& P, int r1z, int r2z, const double* vloc, double* out, cudaStream_t st);
void launch_v2_plane(const V2Plan& P, c128* colbuf, int nb, cudaStream_t st);

// local_z.cu
size_t zw_smem(const ZPlan& P);
cudaError_t zw_kernels_init(const ZPlan& P);
void launch_zw_scatter_zinv(const ZPlan& P, const c128* psi, int64_t ldpsi, c128* colbuf, int nb, cudaStream_t st);
void launch_zw_zfwd_gather(const ZPlan& P, const c128* colbuf, const c128* y, int64_t ldy, const c128* yprev,
                           int64_t ldprev, c128* out, int64_t ldout, double alpha, double cshift, double beta, int nb,
                           cudaStream_t st);

// zgemm.cu
cudaError_t zgemm_init();
// runs `ctas` CTAs x 8 warps x iters x 32 DMMA.8x8x4 (512 flop each) and returns the elapsed milliseconds
cudaError_t dmma_probe(int iters, int ctas, double* sink, cudaStream_t st, float* ms);
// number of K splits chosen for C(M x N) = A^H B with K = npw
int zgemm_cn_splits(int64_t M, int64_t N, int64_t K);
size_t zgemm_cn_workspace(int64_t M, int64_t N, int64_t K);
// C[m + n*ldc] = scale[m] * sum_k conj(A[k + m*lda]) * B[k + n*ldb]      (scale may be null)
void launch_zgemm_cn(int64_t M, int64_t N, int64_t K, const c128* A, int64_t lda, const c128* B, int64_t ldb,
                     const double* scale, c128* C, int64_t ldc, void* ws, cudaStream_t st);
// C[m + n*ldc] += alpha * sum_k A[m + k*lda] * B[k + n*ldb]
void launch_zgemm_nn_acc(int64_t M, int64_t N, int64_t K, double alpha, const c128* A, int64_t lda, const c128* B,
                         int64_t ldb, c128* C, int64_t ldc, cudaStream_t st);

}  // namespace pwh
