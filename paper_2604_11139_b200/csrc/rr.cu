// rr.cu -- the Rayleigh-Ritz companion steps that complete one Chebyshev-filtering iteration around the hot path
// (Algorithm 12 with S = I, PAPER.md:229-238 Algorithms 9 and 10, PAPER.md:153-163
// Algorithm 5).  The N x M work (Gram products, rotations Psi <- Psi X) runs on the DMMA ZGEMM kernels of zgemm.cu; this
// file holds what is left:
//   * column statistics over the plane-wave index (Rayleigh quotients, residual norms): HBM-bound, one CTA per band,
//     warp-shuffle reductions in a fixed order (deterministic);
//   * the dense M x M steps on the device, hand-written (no cuSOLVER): blocked right-looking Cholesky factorisation
//     S = U^H U (potrf), inverse of the triangular factor, and the Hermitian eigen-solve by one-sided Jacobi.
//
// Eigen-solve.  A (Hermitian, M x M) is shifted to B = A + mu I with mu a Gershgorin bound of ||A||_2, so that B is
// positive definite; the one-sided (Hestenes) Jacobi method then rotates pairs of COLUMNS of B until they are mutually
// orthogonal: B V = Q Sigma with Q unitary.  For a Hermitian positive definite B that is its eigen-decomposition: the column
// norms are the eigenvalues of B, the normalised columns the eigenvectors -- no accumulation of V, no row updates, every
// rotation reads and writes two contiguous columns.  A sweep is M-1 rounds of M/2 disjoint pairs (round-robin
// tournament); all pairs of a round are independent, one CTA per pair with both columns staged in shared memory, and the
// rounds are separated by the grid barrier of one cooperative launch (the kernel never waits for another launch).
// The pivot rotation is the 2 x 2 symmetric Schur decomposition (Golub & Van Loan, section 8.5), applied to the Gram block
// [[|b_p|^2, b_p^H b_q], [conj, |b_q|^2]].
#include <cooperative_groups.h>

#include <algorithm>
#include <cmath>

#include "launch.h"

namespace cg = cooperative_groups;

namespace pwh {

namespace {

constexpr int RT = 256;   // threads of the reduction kernels

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
// sum of `v` over the CTA, result in every thread; `red` holds blockDim.x / 32 doubles
__device__ __forceinline__ double block_sum(double v, double* red) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  v = warp_sum(v);
  __syncthreads();
  if (lane == 0) red[warp] = v;
  __syncthreads();
  double s = 0.0;
  for (int i = 0; i < nw; ++i) s += red[i];
  return s;
}

// lambda_b = Re(psi_b^H hpsi_b) / Re(psi_b^H spsi_b), spsi = S psi (null: S = I)      (Algorithm 12 line 3)
__global__ void __launch_bounds__(RT) k_rayleigh(int64_t npw, const c128* __restrict__ psi, int64_t ld,
                                                 const c128* __restrict__ hpsi, int64_t ldh, const c128* __restrict__ spsi,
                                                 int64_t lds, double* __restrict__ lambda, double* __restrict__ nrm2) {
  __shared__ double red[RT / 32];
  const c128* x = psi + (int64_t)blockIdx.x * ld;
  const c128* y = hpsi + (int64_t)blockIdx.x * ldh;
  const c128* z = spsi ? spsi + (int64_t)blockIdx.x * lds : x;
  double num = 0.0, den = 0.0;
  for (int64_t g = threadIdx.x; g < npw; g += RT) {
    const c128 a = x[g], b = y[g], c = z[g];
    num = fma(a.x, b.x, fma(a.y, b.y, num));
    den = fma(a.x, c.x, fma(a.y, c.y, den));
  }
  num = block_sum(num, red);
  den = block_sum(den, red);
  if (threadIdx.x == 0) {
    lambda[blockIdx.x] = num / den;
    if (nrm2) nrm2[blockIdx.x] = den;
  }
}

// out[0] = min, out[1] = max of v[0..n-1]   (one CTA)
__global__ void __launch_bounds__(RT) k_minmax(int64_t n, const double* __restrict__ v, double* __restrict__ out) {
  __shared__ double rmin[RT / 32], rmax[RT / 32];
  double lo = INFINITY, hi = -INFINITY;
  for (int64_t i = threadIdx.x; i < n; i += RT) { lo = fmin(lo, v[i]); hi = fmax(hi, v[i]); }
  lo = -warp_max(-lo);
  hi = warp_max(hi);
  if ((threadIdx.x & 31) == 0) { rmin[threadIdx.x >> 5] = lo; rmax[threadIdx.x >> 5] = hi; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int i = 1; i < RT / 32; ++i) { lo = fmin(lo, rmin[i]); hi = fmax(hi, rmax[i]); }
    out[0] = lo;
    out[1] = hi;
  }
}

// W_b = hpsi_b - lambda_b spsi_b (stored when W != null), norms_b = ||W_b||_2; `psi` is S psi for the generalised problem
// (Algorithm 12 lines 11-12: W <- (H - Lambda S) Psi)
__global__ void __launch_bounds__(RT) k_residual(int64_t npw, const c128* __restrict__ psi, int64_t ld,
                                                 const c128* __restrict__ hpsi, int64_t ldh,
                                                 const double* __restrict__ lambda, c128* __restrict__ W, int64_t ldw,
                                                 double* __restrict__ norms) {
  __shared__ double red[RT / 32];
  const c128* x = psi + (int64_t)blockIdx.x * ld;
  const c128* y = hpsi + (int64_t)blockIdx.x * ldh;
  const double lam = lambda[blockIdx.x];
  double s = 0.0;
  for (int64_t g = threadIdx.x; g < npw; g += RT) {
    const c128 a = x[g], b = y[g];
    const c128 w = cmake(fma(-lam, a.x, b.x), fma(-lam, a.y, b.y));
    if (W) W[(int64_t)blockIdx.x * ldw + g] = w;
    s = fma(w.x, w.x, fma(w.y, w.y, s));
  }
  s = block_sum(s, red);
  if (threadIdx.x == 0) norms[blockIdx.x] = sqrt(s);
}

// ---------------------------------------------------------------------------------------------------------------
// Cholesky factorisation A = U^H U (upper), blocked right-looking, block size 32
// ---------------------------------------------------------------------------------------------------------------
constexpr int NB = 32;

// factor the nb x nb diagonal block at (k0, k0); *info = first non-positive pivot + 1 (kept if already set)
__global__ void __launch_bounds__(NB * NB) k_potrf_diag(c128* __restrict__ A, int64_t lda, int k0, int nb, int* info) {
  __shared__ c128 a[NB][NB + 1];
  const int tx = threadIdx.x % NB, ty = threadIdx.x / NB;   // a[ty][tx] = A[k0+ty, k0+tx]
  const bool in = tx < nb && ty < nb;
  a[ty][tx] = in ? A[(int64_t)(k0 + tx) * lda + k0 + ty] : cmake(ty == tx ? 1.0 : 0.0, 0.0);
  __syncthreads();
  for (int j = 0; j < nb; ++j) {
    if (tx == j && ty == j) {
      const double d = a[j][j].x;
      if (!(d > 0.0)) { if (*info == 0) *info = k0 + j + 1; a[j][j] = cmake(1.0, 0.0); }
      else a[j][j] = cmake(sqrt(d), 0.0);
    }
    __syncthreads();
    if (ty == j && tx > j) { const double r = 1.0 / a[j][j].x; a[j][tx] = cmake(a[j][tx].x * r, a[j][tx].y * r); }
    __syncthreads();
    if (ty > j && tx >= ty) {   // A_rc -= conj(U_jr) U_jc
      const c128 u = a[j][ty], v = a[j][tx];
      a[ty][tx] = cmake(a[ty][tx].x - (u.x * v.x + u.y * v.y), a[ty][tx].y - (u.x * v.y - u.y * v.x));
    }
    __syncthreads();
  }
  if (in) A[(int64_t)(k0 + tx) * lda + k0 + ty] = (ty <= tx) ? a[ty][tx] : cmake(0.0, 0.0);
}

// panel: U12 = U11^-H A12, one warp per column j >= k0 + nb (forward substitution, x_l broadcast by shuffle)
__global__ void __launch_bounds__(256) k_potrf_trsm(c128* __restrict__ A, int64_t lda, int n, int k0, int nb) {
  __shared__ c128 u[NB][NB + 1];
  for (int i = threadIdx.x; i < NB * NB; i += 256) {
    const int r = i % NB, c = i / NB;
    u[r][c] = (r < nb && c < nb) ? A[(int64_t)(k0 + c) * lda + k0 + r] : cmake(r == c ? 1.0 : 0.0, 0.0);
  }
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int j = k0 + nb + blockIdx.x * 8 + (threadIdx.x >> 5);
  if (j >= n) return;
  c128 a = lane < nb ? A[(int64_t)j * lda + k0 + lane] : cmake(0.0, 0.0);
  for (int l = 0; l < nb; ++l) {
    const double r = 1.0 / u[l][l].x;
    const double xr = __shfl_sync(0xffffffffu, a.x, l) * r, xi = __shfl_sync(0xffffffffu, a.y, l) * r;
    if (lane == l) a = cmake(xr, xi);
    else if (lane > l) {   // a_i -= conj(U_li) x_l
      const c128 w = u[l][lane];
      a = cmake(a.x - (w.x * xr + w.y * xi), a.y - (w.x * xi - w.y * xr));
    }
  }
  if (lane < nb) A[(int64_t)j * lda + k0 + lane] = a;
}

// trailing update: A[r, c] -= sum_l conj(U12[l, r]) U12[l, c] for k1 <= r <= c < n (32 x 32 tiles on or above the diagonal)
__global__ void __launch_bounds__(NB * NB) k_potrf_update(c128* __restrict__ A, int64_t lda, int n, int k0, int nb) {
  const int k1 = k0 + nb;
  const int tr = blockIdx.y, tc = blockIdx.x;
  if (tr > tc) return;
  __shared__ c128 ur[NB][NB + 1], uc[NB][NB + 1];   // [l][local index]
  const int tx = threadIdx.x % NB, ty = threadIdx.x / NB;
  const int r0 = k1 + tr * NB, c0 = k1 + tc * NB;
  // thread (ty = l, tx = column within the tile) loads coalesced along l? rows k0..k0+nb-1 of a column are contiguous
  ur[tx][ty] = (tx < nb && r0 + ty < n) ? A[(int64_t)(r0 + ty) * lda + k0 + tx] : cmake(0.0, 0.0);
  uc[tx][ty] = (tx < nb && c0 + ty < n) ? A[(int64_t)(c0 + ty) * lda + k0 + tx] : cmake(0.0, 0.0);
  __syncthreads();
  const int r = r0 + tx, c = c0 + ty;                // thread (tx = row in tile, ty = column in tile): coalesced in r
  if (r >= n || c >= n || r > c) return;
  double sx = 0.0, sy = 0.0;
#pragma unroll 8
  for (int l = 0; l < NB; ++l) {
    const c128 a = ur[l][tx], b = uc[l][ty];         // conj(a) * b
    sx = fma(a.x, b.x, fma(a.y, b.y, sx));
    sy = fma(a.x, b.y, fma(-a.y, b.x, sy));
  }
  c128* p = A + (int64_t)c * lda + r;
  *p = cmake(p->x - sx, p->y - sy);
}

// W = U^-1 for an upper triangular U (column j of W solves U w = e_j by back substitution in axpy form, one CTA per column)
__global__ void __launch_bounds__(256) k_trinv_upper(int n, const c128* __restrict__ U, int64_t ldu, c128* __restrict__ W,
                                                     int64_t ldw) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128* w = reinterpret_cast<c128*>(smem_raw);
  const int j = blockIdx.x, tid = threadIdx.x;
  for (int i = tid; i <= j; i += 256) w[i] = cmake(i == j ? 1.0 : 0.0, 0.0);
  __syncthreads();
  for (int k = j; k >= 0; --k) {
    const double r = 1.0 / U[(int64_t)k * ldu + k].x;
    const c128 wk = cmake(w[k].x * r, w[k].y * r);
    __syncthreads();
    if (tid == 0) w[k] = wk;
    const c128* col = U + (int64_t)k * ldu;
    for (int i = tid; i < k; i += 256) {
      const c128 u = col[i];
      w[i] = cmake(w[i].x - (u.x * wk.x - u.y * wk.y), w[i].y - (u.x * wk.y + u.y * wk.x));
    }
    __syncthreads();
  }
  for (int i = tid; i < n; i += 256) W[(int64_t)j * ldw + i] = i <= j ? w[i] : cmake(0.0, 0.0);
}

// zero the strictly lower triangle
__global__ void k_zero_lower(int n, c128* __restrict__ A, int64_t lda) {
  const int64_t total = (int64_t)n * n;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int r = (int)(i % n), c = (int)(i / n);
    if (r > c) A[(int64_t)c * lda + r] = cmake(0.0, 0.0);
  }
}

// A <- (A + A^H) / 2 with a real diagonal (removes the rounding-level anti-Hermitian part of a computed product)
__global__ void k_hermitise(int n, c128* __restrict__ A, int64_t lda) {
  const int64_t total = (int64_t)n * n;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int r = (int)(i % n), c = (int)(i / n);
    if (r > c) continue;
    const c128 a = A[(int64_t)c * lda + r], b = A[(int64_t)r * lda + c];
    const c128 m = cmake(0.5 * (a.x + b.x), r == c ? 0.0 : 0.5 * (a.y - b.y));
    A[(int64_t)c * lda + r] = m;
    A[(int64_t)r * lda + c] = cmake(m.x, -m.y);
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Hermitian eigen-solve: one-sided Jacobi on B = A + mu I
// ---------------------------------------------------------------------------------------------------------------
// mu = 1.0625 * max_j sum_i |a_ij| (Gershgorin bound of ||A||_2; 1 when A = 0), B = A + mu I in place; one CTA, fixed order
__global__ void __launch_bounds__(1024) k_jacobi_shift(int n, c128* __restrict__ A, int64_t lda, double* __restrict__ mu_out) {
  __shared__ double red[32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double best = 0.0;
  for (int j = warp; j < n; j += 32) {
    double s = 0.0;
    for (int i = lane; i < n; i += 32) { const c128 a = A[(int64_t)j * lda + i]; s += sqrt(a.x * a.x + a.y * a.y); }
    s = warp_sum(s);
    best = fmax(best, s);
  }
  if (lane == 0) red[warp] = best;
  __syncthreads();
  double mu = 0.0;
  for (int i = 0; i < 32; ++i) mu = fmax(mu, red[i]);
  mu = mu > 0.0 ? 1.0625 * mu : 1.0;
  for (int j = threadIdx.x; j < n; j += 1024) A[(int64_t)j * lda + j].x += mu;
  if (threadIdx.x == 0) *mu_out = mu;
}

struct JacobiArgs {
  int n;             // matrix order
  int np;            // n rounded up to even (a dummy player n when n is odd)
  c128* B;
  int64_t ldb;
  int max_sweeps;
  double tol;        // a pair is rotated while |b_p^H b_q| > tol |b_p| |b_q|
  double* offmax;    // [max_sweeps] largest |b_p^H b_q| / (|b_p| |b_q|) met in each sweep (zeroed by the host)
  int* sweeps;       // out: sweeps performed
  int stage_cols;    // 1: both columns of a pair staged in shared memory
};

__global__ void __launch_bounds__(256) k_jacobi(const JacobiArgs P) {
  cg::grid_group grid = cg::this_grid();
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128* sp = reinterpret_cast<c128*>(smem_raw);
  c128* sq = sp + P.n;
  __shared__ double red[8];
  const int tid = threadIdx.x, n = P.n, np = P.np, m1 = np - 1;
  int sweep = 0;
  for (; sweep < P.max_sweeps; ++sweep) {
    for (int r = 0; r < m1; ++r) {
      for (int i = blockIdx.x; i < np / 2; i += gridDim.x) {
        int p, q;
        if (i == 0) { p = m1; q = r; }
        else { p = (r + i) % m1; q = (r - i + m1) % m1; }
        if (p >= n || q >= n) continue;   // the dummy player of an odd n
        c128* bp = P.B + (int64_t)p * P.ldb;
        c128* bq = P.B + (int64_t)q * P.ldb;
        double al = 0.0, be = 0.0, gx = 0.0, gy = 0.0;
        // columns are rewritten by other CTAs between rounds: read them through L2 (ld.global.cg), never through this SM's L1
        for (int k = tid; k < n; k += 256) {
          const c128 x = __ldcg(bp + k), y = __ldcg(bq + k);
          if (P.stage_cols) { sp[k] = x; sq[k] = y; }
          al = fma(x.x, x.x, fma(x.y, x.y, al));
          be = fma(y.x, y.x, fma(y.y, y.y, be));
          gx = fma(x.x, y.x, fma(x.y, y.y, gx));     // conj(x) * y
          gy = fma(x.x, y.y, fma(-x.y, y.x, gy));
        }
        al = block_sum(al, red);
        be = block_sum(be, red);
        gx = block_sum(gx, red);
        gy = block_sum(gy, red);
        const double g = sqrt(gx * gx + gy * gy), sc = sqrt(al * be);
        if (tid == 0 && sc > 0.0)
          atomicMax(reinterpret_cast<unsigned long long*>(P.offmax + sweep), (unsigned long long)__double_as_longlong(g / sc));
        if (!(g > P.tol * sc)) continue;             // uniform over the CTA
        const double zeta = (be - al) / (2.0 * g);
        const double t = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
        const double c = 1.0 / sqrt(1.0 + t * t), s = c * t;
        const double phx = gx / g, phy = gy / g;     // e^{i phi}; the rotation uses e^{-i phi} = (phx, -phy)
        for (int k = tid; k < n; k += 256) {
          const c128 x = P.stage_cols ? sp[k] : __ldcg(bp + k), y = P.stage_cols ? sq[k] : __ldcg(bq + k);
          const c128 yr = cmake(y.x * phx + y.y * phy, y.y * phx - y.x * phy);   // e^{-i phi} y
          bp[k] = cmake(c * x.x - s * yr.x, c * x.y - s * yr.y);
          bq[k] = cmake(s * x.x + c * yr.x, s * x.y + c * yr.y);
        }
      }
      grid.sync();
    }
    // the same value in every thread after the grid barrier (read through L2: other CTAs updated it with atomics)
    if (__ldcg(P.offmax + sweep) <= P.tol) { ++sweep; break; }
  }
  if (blockIdx.x == 0 && tid == 0) *P.sweeps = sweep;
}

// sig_j = |b_j|;  w_j = sig_j - mu  (one CTA per column)
__global__ void __launch_bounds__(RT) k_jacobi_norms(int n, const c128* __restrict__ B, int64_t ldb,
                                                     const double* __restrict__ mu, double* __restrict__ sig,
                                                     double* __restrict__ wraw) {
  __shared__ double red[RT / 32];
  const c128* b = B + (int64_t)blockIdx.x * ldb;
  double s = 0.0;
  for (int k = threadIdx.x; k < n; k += RT) { const c128 x = b[k]; s = fma(x.x, x.x, fma(x.y, x.y, s)); }
  s = block_sum(s, red);
  if (threadIdx.x == 0) { const double r = sqrt(s); sig[blockIdx.x] = r; wraw[blockIdx.x] = r - *mu; }
}

// ascending order: rank_j = #{i : w_i < w_j or (w_i == w_j and i < j)};  X[:, rank_j] = b_j / sig_j,  w[rank_j] = w_j
__global__ void __launch_bounds__(RT) k_jacobi_sort(int n, const c128* __restrict__ B, int64_t ldb,
                                                    const double* __restrict__ sig, const double* __restrict__ wraw,
                                                    double* __restrict__ w, c128* __restrict__ X, int64_t ldx) {
  __shared__ double red[RT / 32];
  const int j = blockIdx.x;
  const double wj = wraw[j];
  double cnt = 0.0;
  for (int i = threadIdx.x; i < n; i += RT) { const double wi = wraw[i]; cnt += (wi < wj || (wi == wj && i < j)) ? 1.0 : 0.0; }
  const int rank = (int)(block_sum(cnt, red) + 0.5);
  const double r = 1.0 / sig[j];
  const c128* b = B + (int64_t)j * ldb;
  c128* x = X + (int64_t)rank * ldx;
  for (int k = threadIdx.x; k < n; k += RT) x[k] = cmake(b[k].x * r, b[k].y * r);
  if (threadIdx.x == 0) w[rank] = wj;
}

// info convention of the dense solvers: > 0 = Jacobi sweeps used, < 0 = -(index + 1) of the non-positive Cholesky pivot
__global__ void k_merge_info(const int* __restrict__ potrf_info, int* __restrict__ info) {
  if (*potrf_info != 0) *info = -*potrf_info;
}

}  // namespace

void launch_merge_info(const int* potrf_info, int* info, cudaStream_t st) {
  ScopedLaunch sl(ST_SMALL, st);
  k_merge_info<<<1, 1, 0, st>>>(potrf_info, info);
}

// ---------------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------------
void launch_rayleigh(int64_t npw, int64_t nband, const c128* psi, int64_t ld, const c128* hpsi, int64_t ldh,
                     const c128* spsi, int64_t lds, double* lambda, double* nrm2, double* minmax, cudaStream_t st) {
  {
    ScopedLaunch sl(ST_COLSTATS, st);
    k_rayleigh<<<(unsigned)nband, RT, 0, st>>>(npw, psi, ld, hpsi, ldh, spsi, lds, lambda, nrm2);
  }
  if (minmax) {
    ScopedLaunch sl(ST_SMALL, st);
    k_minmax<<<1, RT, 0, st>>>(nband, lambda, minmax);
  }
}

void launch_residual(int64_t npw, int64_t nband, const c128* psi, int64_t ld, const c128* hpsi, int64_t ldh,
                     const double* lambda, c128* W, int64_t ldw, double* norms, cudaStream_t st) {
  ScopedLaunch sl(ST_COLSTATS, st);
  k_residual<<<(unsigned)nband, RT, 0, st>>>(npw, psi, ld, hpsi, ldh, lambda, W, ldw, norms);
}

// A (upper triangle read) -> U in place, strictly lower triangle zeroed; *info (device, zeroed here) = failing pivot + 1
void launch_potrf_upper(int n, c128* A, int64_t lda, int* info, cudaStream_t st) {
  cudaMemsetAsync(info, 0, sizeof(int), st);
  for (int k0 = 0; k0 < n; k0 += NB) {
    const int nb = std::min(NB, n - k0), rest = n - k0 - nb;
    { ScopedLaunch sl(ST_SMALL, st); k_potrf_diag<<<1, NB * NB, 0, st>>>(A, lda, k0, nb, info); }
    if (rest <= 0) break;
    { ScopedLaunch sl(ST_SMALL, st); k_potrf_trsm<<<(rest + 7) / 8, 256, 0, st>>>(A, lda, n, k0, nb); }
    const int t = (rest + NB - 1) / NB;
    { ScopedLaunch sl(ST_SMALL, st); k_potrf_update<<<dim3(t, t), NB * NB, 0, st>>>(A, lda, n, k0, nb); }
  }
  // the strictly lower triangle below the diagonal blocks (the diagonal blocks were cleaned by k_potrf_diag)
  ScopedLaunch sl(ST_SMALL, st);
  k_zero_lower<<<148 * 2, 256, 0, st>>>(n, A, lda);
}

cudaError_t rr_kernels_init() {
  cudaError_t e = set_max_dyn_smem(reinterpret_cast<const void*>(&k_trinv_upper));
  if (e != cudaSuccess) return e;
  return set_max_dyn_smem(reinterpret_cast<const void*>(&k_jacobi));
}

void launch_trinv_upper(int n, const c128* U, int64_t ldu, c128* W, int64_t ldw, cudaStream_t st) {
  ScopedLaunch sl(ST_SMALL, st);
  k_trinv_upper<<<n, 256, (size_t)n * sizeof(c128), st>>>(n, U, ldu, W, ldw);
}

void launch_hermitise(int n, c128* A, int64_t lda, cudaStream_t st) {
  ScopedLaunch sl(ST_SMALL, st);
  k_hermitise<<<148 * 2, 256, 0, st>>>(n, A, lda);
}

size_t jacobi_scratch_bytes(int n) { return sizeof(double) * (size_t)(2 * n + 64 + 8); }

// Eigen-decomposition of the Hermitian A (n x n, destroyed): w ascending, X = eigenvectors.  scratch: jacobi_scratch_bytes(n)
// device bytes.  *sweeps (device int) = sweeps used.  Cooperative launch: the grid is sized to be co-resident.
cudaError_t launch_heev_jacobi(int n, c128* A, int64_t lda, double* w, c128* X, int64_t ldx, int* sweeps, void* scratch,
                               cudaStream_t st) {
  constexpr int MAX_SWEEPS = 40;
  double* d = reinterpret_cast<double*>(scratch);
  double* mu = d;            // [1] (+7 padding)
  double* offmax = d + 8;    // [64]
  double* sig = d + 72;      // [n]
  double* wraw = sig + n;    // [n]
  cudaError_t e = cudaMemsetAsync(offmax, 0, 64 * sizeof(double), st);
  if (e != cudaSuccess) return e;
  { ScopedLaunch sl(ST_SMALL, st); k_jacobi_shift<<<1, 1024, 0, st>>>(n, A, lda, mu); }
  if (n > 1) {
    int dev = 0, sms = 0, smem_max = 0, per_sm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    JacobiArgs P;
    // a pair counts as orthogonal once its cosine is below the rounding level of a length-n dot product
    P.n = n; P.np = (n + 1) & ~1; P.B = A; P.ldb = lda; P.max_sweeps = MAX_SWEEPS;
    P.tol = std::max(1e-15, 4.5e-16 * std::sqrt((double)n));
    P.offmax = offmax; P.sweeps = sweeps;
    size_t smem = 2 * (size_t)n * sizeof(c128);
    P.stage_cols = smem + 1024 <= (size_t)smem_max ? 1 : 0;
    if (!P.stage_cols) smem = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_jacobi, 256, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    const int grid = std::max(1, std::min(P.np / 2, sms * std::min(per_sm, 4)));
    void* args[] = {(void*)&P};
    ScopedLaunch sl(ST_JACOBI, st);
    e = cudaLaunchCooperativeKernel((const void*)k_jacobi, dim3(grid), dim3(256), args, smem, st);
    if (e != cudaSuccess) return e;
  } else {
    cudaMemsetAsync(sweeps, 0, sizeof(int), st);
  }
  { ScopedLaunch sl(ST_SMALL, st); k_jacobi_norms<<<n, RT, 0, st>>>(n, A, lda, mu, sig, wraw); }
  { ScopedLaunch sl(ST_SMALL, st); k_jacobi_sort<<<n, RT, 0, st>>>(n, A, lda, sig, wraw, w, X, ldx); }
  return cudaGetLastError();
}

}  // namespace pwh
