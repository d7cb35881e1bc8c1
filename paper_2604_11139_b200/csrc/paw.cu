// paw.cu -- small kernels of the PAW-style generalised problem H Psi = Lambda S Psi:
//   * per-atom dense blocks applied to the projections: C' = blockdiag(D^R) C and blockdiag(Q^R) C
//     (V_nonloc = sum_{R,i,j} |p_i^R> D_ij^R <p_j^R|; the paper batches these small products with
//     gemmStridedBatched -- here one thread per output entry, the blocks are at most a few dozen wide and the whole
//     step is 1e-4 of the projector ZGEMMs that surround it);
//   * helpers for the J x J matrix K of S^-1 = I - P K P^H ("Sinv ... Woodbury");
//   * the three-term axpy of the filter on S^-1 H ("X <- aX + Y ... axpy(n, m)", Algorithm 12 line 6).
// The N x J and N x M work around them runs on the DMMA ZGEMM kernels of zgemm.cu.
#include <algorithm>

#include "launch.h"

namespace pwh {

namespace {

// out[i, b] = sum_j B^R[i - lo, j - lo] in[j, b] with R the block of projector i; blocks packed column-major at boff[R]
__global__ void __launch_bounds__(256) k_blockdiag_apply(int64_t nproj, int64_t nband, const int* __restrict__ blk_of,
                                                         const int* __restrict__ blk_lo, const int64_t* __restrict__ boff,
                                                         const c128* __restrict__ blocks, const c128* __restrict__ in,
                                                         int64_t ldi, c128* __restrict__ out, int64_t ldo) {
  const int64_t total = nproj * nband;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t i = t % nproj, b = t / nproj;
    const int r = blk_of[i];
    const int lo = blk_lo[r], n = blk_lo[r + 1] - lo;
    const c128* B = blocks + boff[r] + (i - lo);       // row i - lo of the column-major block
    const c128* c = in + b * ldi + lo;
    double sx = 0.0, sy = 0.0;
    for (int j = 0; j < n; ++j) {
      const c128 m = B[(int64_t)j * n], v = c[j];
      sx = fma(m.x, v.x, fma(-m.y, v.y, sx));
      sy = fma(m.x, v.y, fma(m.y, v.x, sy));
    }
    out[b * ldo + i] = cmake(sx, sy);
  }
}

// dense n x n matrix (zero outside the blocks) from the packed blocks
__global__ void k_blocks_to_dense(int64_t nproj, const int* __restrict__ blk_of, const int* __restrict__ blk_lo,
                                  const int64_t* __restrict__ boff, const c128* __restrict__ blocks, c128* __restrict__ out,
                                  int64_t ldo) {
  const int64_t total = nproj * nproj;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t i = t % nproj, j = t / nproj;
    const int r = blk_of[i];
    const int lo = blk_lo[r], n = blk_lo[r + 1] - lo;
    out[j * ldo + i] = (blk_of[j] == r) ? blocks[boff[r] + (i - lo) + (j - lo) * (int64_t)n] : cmake(0.0, 0.0);
  }
}

// out = in^H (n x n)
__global__ void k_conj_transpose(int n, const c128* __restrict__ in, int64_t ldi, c128* __restrict__ out, int64_t ldo) {
  __shared__ c128 tile[32][33];
  const int bx = blockIdx.x * 32, by = blockIdx.y * 32, tx = threadIdx.x, ty = threadIdx.y;
  for (int k = ty; k < 32; k += 8) {
    const int r = bx + tx, c = by + k;
    tile[k][tx] = (r < n && c < n) ? in[(int64_t)c * ldi + r] : cmake(0.0, 0.0);
  }
  __syncthreads();
  for (int k = ty; k < 32; k += 8) {
    const int r = by + tx, c = bx + k;               // out[r, c] = conj(in[c, r])
    if (r < n && c < n) { const c128 v = tile[tx][k]; out[(int64_t)c * ldo + r] = cmake(v.x, -v.y); }
  }
}

// A <- alpha A + beta B (+ gamma I), n x n
__global__ void k_mat_axpby(int n, double alpha, c128* __restrict__ A, int64_t lda, double beta, const c128* __restrict__ B,
                            int64_t ldb, double gamma) {
  const int64_t total = (int64_t)n * n;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int r = (int)(t % n), c = (int)(t / n);
    c128 a = A[(int64_t)c * lda + r];
    const c128 b = B ? B[(int64_t)c * ldb + r] : cmake(0.0, 0.0);
    a = cmake(alpha * a.x + beta * b.x, alpha * a.y + beta * b.y);
    if (r == c) a.x += gamma;
    A[(int64_t)c * lda + r] = a;
  }
}

// out = alpha (z - c y) - beta yprev over an npw x nband block; out may alias z or yprev (entry by entry, same thread)
__global__ void __launch_bounds__(256) k_cheb_axpy(int64_t npw, int64_t nband, const c128* z, int64_t ldz, const c128* y,
                                                   int64_t ldy, const c128* yprev, int64_t ldp, c128* out, int64_t ldo,
                                                   double alpha, double cshift, double beta) {
  const int64_t total = npw * nband;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t g = t % npw, b = t / npw;
    const c128 zv = z[b * ldz + g], yv = y[b * ldy + g];
    c128 r = cmake(alpha * fma(-cshift, yv.x, zv.x), alpha * fma(-cshift, yv.y, zv.y));
    if (yprev) {
      const c128 pv = yprev[b * ldp + g];
      r.x = fma(-beta, pv.x, r.x);
      r.y = fma(-beta, pv.y, r.y);
    }
    out[b * ldo + g] = r;
  }
}

int grid_for(int64_t total) {
  int64_t b = (total + 255) / 256;
  return (int)std::max<int64_t>(1, std::min<int64_t>(b, 148 * 8));
}

}  // namespace

void launch_blockdiag_apply(int64_t nproj, int64_t nband, const int* blk_of, const int* blk_lo, const int64_t* boff,
                            const c128* blocks, const c128* in, int64_t ldi, c128* out, int64_t ldo, cudaStream_t st) {
  ScopedLaunch sl(ST_SMALL, st);
  k_blockdiag_apply<<<grid_for(nproj * nband), 256, 0, st>>>(nproj, nband, blk_of, blk_lo, boff, blocks, in, ldi, out, ldo);
}

void launch_blocks_to_dense(int64_t nproj, const int* blk_of, const int* blk_lo, const int64_t* boff, const c128* blocks,
                            c128* out, int64_t ldo, cudaStream_t st) {
  ScopedLaunch sl(ST_SMALL, st);
  k_blocks_to_dense<<<grid_for(nproj * nproj), 256, 0, st>>>(nproj, blk_of, blk_lo, boff, blocks, out, ldo);
}

void launch_conj_transpose(int n, const c128* in, int64_t ldi, c128* out, int64_t ldo, cudaStream_t st) {
  ScopedLaunch sl(ST_SMALL, st);
  const int t = (n + 31) / 32;
  k_conj_transpose<<<dim3(t, t), dim3(32, 8), 0, st>>>(n, in, ldi, out, ldo);
}

void launch_mat_axpby(int n, double alpha, c128* A, int64_t lda, double beta, const c128* B, int64_t ldb, double gamma,
                      cudaStream_t st) {
  ScopedLaunch sl(ST_SMALL, st);
  k_mat_axpby<<<grid_for((int64_t)n * n), 256, 0, st>>>(n, alpha, A, lda, beta, B, ldb, gamma);
}

void launch_cheb_axpy(int64_t npw, int64_t nband, const c128* z, int64_t ldz, const c128* y, int64_t ldy, const c128* yprev,
                      int64_t ldp, c128* out, int64_t ldo, double alpha, double cshift, double beta, cudaStream_t st) {
  ScopedLaunch sl(ST_AXPY, st);
  k_cheb_axpy<<<148 * 8, 256, 0, st>>>(npw, nband, z, ldz, y, ldy, yprev, ldp, out, ldo, alpha, cshift, beta);
}

}  // namespace pwh
