// launch.h -- internal launcher declarations shared by the libpwham translation units.
#pragma once
#include "common.cuh"

namespace pwh {

void count_launch();

// local_kernels.cu
size_t zkernel_smem(const LocalPlan& P);
size_t plane_smem(const LocalPlan& P);
cudaError_t local_kernels_init(const LocalPlan& P);
void launch_scatter_zinv(const LocalPlan& P, const c128* psi, int64_t ldpsi, c128* colbuf, int nb, cudaStream_t st);
void launch_plane(const LocalPlan& P, c128* colbuf, int nb, cudaStream_t st);
void launch_zfwd_gather(const LocalPlan& P, const c128* colbuf, const c128* y, int64_t ldy, const c128* yprev,
                        int64_t ldprev, c128* out, int64_t ldout, double alpha, double cshift, double beta, int nb,
                        cudaStream_t st);

// zgemm.cu
cudaError_t zgemm_init();
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
