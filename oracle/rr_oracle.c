/*
 * rr_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain CPU oracle for the steps that complete one Chebyshev-filtering iteration around the hot path of
 * arxiv/paper_2604_11139, written from the definitions / textbook algorithms in FP64 with
 * long-double accumulations, no blocking, no fusion:
 *
 *   orc_rayleigh          lambda_i = (H psi_i)^H psi_i / (psi_i^H psi_i)          PAPER.md:244; Algorithm 12 line 3
 *   orc_rotate            Y = X Q  (Psi <- Psi X, H Psi <- (H Psi) X)              Algorithm 5 steps 4-5 / Algorithm 10
 *   orc_residual          W = H Psi - Psi Lambda (S = I), column norms            Algorithm 12 lines 11-12
 *   orc_potrf_upper       S = U^H U, U upper triangular with positive diagonal    Algorithm 9 step 2 "potrf"
 *   orc_trsm_right_upper  X <- X U^-1                                             Algorithm 9 steps 3-5 "trsm"
 *   orc_heev_jacobi       A = V diag(w) V^H, cyclic two-sided Jacobi              Algorithm 5/10 step 3 "hegvd" with S_Psi = I
 *   orc_hegv              A X = B X diag(w), X^H B X = I                          Algorithm 5/10 step 3 "hegvd"
 *
 * The eigen-decomposition has no closed form; the oracle follows the classical cyclic Jacobi method for Hermitian
 * matrices (Golub & Van Loan, "Matrix Computations", section 8.5: symmetric Schur decomposition of the 2 x 2 pivot block,
 * with the complex phase of the pivot removed first), and the generalised problem is reduced to it through the Cholesky
 * factor of B exactly as LAPACK's hegvd does (B = U^H U, C = U^-H A U^-1, C Y = Y Lambda, X = U^-1 Y).  Eigenvalues are
 * returned in ascending order.  Eigenvectors are unique only up to a phase (and up to a unitary mixing inside a
 * degenerate eigenspace), so tests compare eigenvalues, residuals, orthonormality and spectral projectors, never vectors.
 *
 * Pins (tests/test_rr_oracle_pins.py): closed forms (2 x 2, diagonal, rank-one, circulant = DFT of the first row), numpy /
 * scipy library routines as special cases, Rayleigh quotients of plane waves in constant V0, exact eigenvectors of the dense
 * H give zero residuals, permutation and Givens rotations, U against numpy's Cholesky factor.  Nothing is unpinned.
 *
 * It shares no code with the CUDA path.  Layout: column-major, complex128 = (re, im) pairs, leading dimensions in elements.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double _Complex cplx;

/* lambda_i = Re(psi_i^H (H psi)_i) / (psi_i^H psi_i);  nrm2_i = psi_i^H psi_i  (may be NULL) */
void orc_rayleigh(int64_t npw, int64_t nband, const cplx *psi, int64_t ld, const cplx *hpsi, int64_t ldh, double *lambda,
                  double *nrm2) {
  for (int64_t b = 0; b < nband; ++b) {
    const cplx *x = psi + b * ld, *y = hpsi + b * ldh;
    long double num = 0.0L, den = 0.0L;
    for (int64_t g = 0; g < npw; ++g) {
      num += (long double)creal(x[g]) * creal(y[g]) + (long double)cimag(x[g]) * cimag(y[g]);
      den += (long double)creal(x[g]) * creal(x[g]) + (long double)cimag(x[g]) * cimag(x[g]);
    }
    lambda[b] = (double)(num / den);
    if (nrm2) nrm2[b] = (double)den;
  }
}

/* Y[g, j] = sum_i X[g, i] Q[i, j];  X npw x m, Q m x n, Y npw x n.  Y must not overlap X. */
void orc_rotate(int64_t npw, int64_t m, const cplx *X, int64_t ldx, int64_t n, const cplx *Q, int64_t ldq, cplx *Y,
                int64_t ldy) {
#pragma omp parallel for schedule(static)
  for (int64_t j = 0; j < n; ++j)
    for (int64_t g = 0; g < npw; ++g) {
      long double sr = 0.0L, si = 0.0L;
      for (int64_t i = 0; i < m; ++i) {
        cplx x = X[g + i * ldx], q = Q[i + j * ldq];
        sr += (long double)creal(x) * creal(q) - (long double)cimag(x) * cimag(q);
        si += (long double)creal(x) * cimag(q) + (long double)cimag(x) * creal(q);
      }
      Y[g + j * ldy] = (double)sr + I * (double)si;
    }
}

/* W_i = (H psi)_i - lambda_i psi_i, norms_i = ||W_i||_2.  W may be NULL (norms only). */
void orc_residual(int64_t npw, int64_t nband, const cplx *psi, int64_t ld, const cplx *hpsi, int64_t ldh,
                  const double *lambda, cplx *W, int64_t ldw, double *norms) {
  for (int64_t b = 0; b < nband; ++b) {
    long double s = 0.0L;
    for (int64_t g = 0; g < npw; ++g) {
      cplx w = hpsi[b * ldh + g] - lambda[b] * psi[b * ld + g];
      if (W) W[b * ldw + g] = w;
      s += (long double)creal(w) * creal(w) + (long double)cimag(w) * cimag(w);
    }
    norms[b] = (double)sqrtl(s);
  }
}

/* In place: the upper triangle of the Hermitian positive-definite A (only its upper triangle is read) becomes U with
 * A = U^H U and U_jj > 0; the strictly lower triangle is set to zero.  Returns 0, or j+1 if the j-th pivot is not positive. */
int orc_potrf_upper(int64_t n, cplx *A, int64_t lda) {
  for (int64_t j = 0; j < n; ++j) {
    long double d = creal(A[j + j * lda]);
    for (int64_t k = 0; k < j; ++k) {
      cplx u = A[k + j * lda];
      d -= (long double)creal(u) * creal(u) + (long double)cimag(u) * cimag(u);
    }
    if (!(d > 0.0L)) return (int)(j + 1);
    double ujj = (double)sqrtl(d);
    A[j + j * lda] = ujj;
    for (int64_t i = j + 1; i < n; ++i) { /* U_ji = (A_ji - sum_k conj(U_kj) U_ki) / U_jj */
      long double sr = creal(A[j + i * lda]), si = cimag(A[j + i * lda]);
      for (int64_t k = 0; k < j; ++k) {
        cplx a = A[k + j * lda], b = A[k + i * lda]; /* conj(a) * b */
        sr -= (long double)creal(a) * creal(b) + (long double)cimag(a) * cimag(b);
        si -= (long double)creal(a) * cimag(b) - (long double)cimag(a) * creal(b);
      }
      A[j + i * lda] = ((double)sr + I * (double)si) / ujj;
    }
  }
  for (int64_t j = 0; j < n; ++j)
    for (int64_t i = j + 1; i < n; ++i) A[i + j * lda] = 0.0;
  return 0;
}

/* X <- X U^-1 for an npw x n block X and an upper triangular U (solve Y U = X column by column). */
void orc_trsm_right_upper(int64_t npw, int64_t n, cplx *X, int64_t ldx, const cplx *U, int64_t ldu) {
  for (int64_t j = 0; j < n; ++j) {
    cplx ujj = U[j + j * ldu];
#pragma omp parallel for schedule(static)
    for (int64_t g = 0; g < npw; ++g) {
      long double sr = creal(X[g + j * ldx]), si = cimag(X[g + j * ldx]);
      for (int64_t k = 0; k < j; ++k) {
        cplx y = X[g + k * ldx], u = U[k + j * ldu];
        sr -= (long double)creal(y) * creal(u) - (long double)cimag(y) * cimag(u);
        si -= (long double)creal(y) * cimag(u) + (long double)cimag(y) * creal(u);
      }
      X[g + j * ldx] = ((double)sr + I * (double)si) / ujj;
    }
  }
}

/* X <- U^-1 X for an n x m block X (back substitution, column by column of X). */
static void trsm_left_upper(int64_t n, int64_t m, const cplx *U, int64_t ldu, cplx *X, int64_t ldx) {
  for (int64_t c = 0; c < m; ++c)
    for (int64_t i = n - 1; i >= 0; --i) {
      long double sr = creal(X[i + c * ldx]), si = cimag(X[i + c * ldx]);
      for (int64_t k = i + 1; k < n; ++k) {
        cplx u = U[i + k * ldu], x = X[k + c * ldx];
        sr -= (long double)creal(u) * creal(x) - (long double)cimag(u) * cimag(x);
        si -= (long double)creal(u) * cimag(x) + (long double)cimag(u) * creal(x);
      }
      X[i + c * ldx] = ((double)sr + I * (double)si) / U[i + i * ldu];
    }
}

/* X <- U^-H X for an n x m block X (forward substitution with the lower triangular U^H). */
static void trsm_left_upper_conjtrans(int64_t n, int64_t m, const cplx *U, int64_t ldu, cplx *X, int64_t ldx) {
  for (int64_t c = 0; c < m; ++c)
    for (int64_t i = 0; i < n; ++i) {
      long double sr = creal(X[i + c * ldx]), si = cimag(X[i + c * ldx]);
      for (int64_t k = 0; k < i; ++k) {
        cplx u = conj(U[k + i * ldu]), x = X[k + c * ldx]; /* (U^H)_ik = conj(U_ki) */
        sr -= (long double)creal(u) * creal(x) - (long double)cimag(u) * cimag(x);
        si -= (long double)creal(u) * cimag(x) + (long double)cimag(u) * creal(x);
      }
      X[i + c * ldx] = ((double)sr + I * (double)si) / conj(U[i + i * ldu]);
    }
}

/* Cyclic two-sided Jacobi for a Hermitian A (full matrix given; destroyed).  On return w[0..n-1] ascending and the
 * columns of V the matching orthonormal eigenvectors: A V = V diag(w).  Returns the number of sweeps used.
 * Pivot (p,q), a_pq = |a_pq| e^{i phi}:  J = [[c, s], [-s e^{-i phi}, c e^{-i phi}]] with t = tan(theta) the smaller root
 * of t^2 + 2 zeta t - 1 = 0, zeta = (a_qq - a_pp) / (2 |a_pq|);  A <- J^H A J annihilates a_pq;  V <- V J. */
int orc_heev_jacobi(int64_t n, cplx *A, int64_t lda, double *w, cplx *V, int64_t ldv) {
  for (int64_t j = 0; j < n; ++j)
    for (int64_t i = 0; i < n; ++i) V[i + j * ldv] = (i == j) ? 1.0 : 0.0;
  long double fro2 = 0.0L;
  for (int64_t j = 0; j < n; ++j)
    for (int64_t i = 0; i < n; ++i) fro2 += (long double)creal(A[i + j * lda]) * creal(A[i + j * lda]) +
                                            (long double)cimag(A[i + j * lda]) * cimag(A[i + j * lda]);
  int sweep = 0;
  for (; sweep < 60; ++sweep) {
    long double off2 = 0.0L;
    for (int64_t j = 0; j < n; ++j)
      for (int64_t i = 0; i < j; ++i) off2 += 2.0L * ((long double)creal(A[i + j * lda]) * creal(A[i + j * lda]) +
                                                     (long double)cimag(A[i + j * lda]) * cimag(A[i + j * lda]));
    if (off2 <= 1e-30L * fro2) break;
    for (int64_t p = 0; p < n - 1; ++p)
      for (int64_t q = p + 1; q < n; ++q) {
        cplx apq = A[p + q * lda];
        double g = cabs(apq);
        if (g == 0.0) continue;
        double app = creal(A[p + p * lda]), aqq = creal(A[q + q * lda]);
        double zeta = (aqq - app) / (2.0 * g);
        double t = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
        double c = 1.0 / sqrt(1.0 + t * t), s = c * t;
        cplx ph = apq / g;        /* e^{i phi} */
        cplx phc = conj(ph);      /* e^{-i phi} */
        /* columns: A <- A J, V <- V J :  col_p' = c col_p - s e^{-i phi} col_q ;  col_q' = s col_p + c e^{-i phi} col_q */
        for (int64_t i = 0; i < n; ++i) {
          cplx xp = A[i + p * lda], xq = A[i + q * lda];
          A[i + p * lda] = c * xp - s * phc * xq;
          A[i + q * lda] = s * xp + c * phc * xq;
          cplx vp = V[i + p * ldv], vq = V[i + q * ldv];
          V[i + p * ldv] = c * vp - s * phc * vq;
          V[i + q * ldv] = s * vp + c * phc * vq;
        }
        /* rows: A <- J^H A :  row_p' = c row_p - s e^{i phi} row_q ;  row_q' = s row_p + c e^{i phi} row_q */
        for (int64_t j = 0; j < n; ++j) {
          cplx xp = A[p + j * lda], xq = A[q + j * lda];
          A[p + j * lda] = c * xp - s * ph * xq;
          A[q + j * lda] = s * xp + c * ph * xq;
        }
        A[p + q * lda] = 0.0;
        A[q + p * lda] = 0.0;
        A[p + p * lda] = creal(A[p + p * lda]);
        A[q + q * lda] = creal(A[q + q * lda]);
      }
  }
  /* ascending order (selection sort on the eigenvalues, columns of V swapped along) */
  for (int64_t i = 0; i < n; ++i) w[i] = creal(A[i + i * lda]);
  for (int64_t i = 0; i < n - 1; ++i) {
    int64_t k = i;
    for (int64_t j = i + 1; j < n; ++j)
      if (w[j] < w[k]) k = j;
    if (k != i) {
      double tw = w[i]; w[i] = w[k]; w[k] = tw;
      for (int64_t r = 0; r < n; ++r) { cplx tv = V[r + i * ldv]; V[r + i * ldv] = V[r + k * ldv]; V[r + k * ldv] = tv; }
    }
  }
  return sweep;
}

/* Generalised Hermitian-definite problem A X = B X diag(w), X^H B X = I (A, B full Hermitian matrices; both destroyed).
 * Returns 0, or j+1 if B is not positive definite at pivot j. */
int orc_hegv(int64_t n, cplx *A, int64_t lda, cplx *B, int64_t ldb, double *w, cplx *X, int64_t ldx) {
  int rc = orc_potrf_upper(n, B, ldb);            /* B = U^H U */
  if (rc) return rc;
  trsm_left_upper_conjtrans(n, n, B, ldb, A, lda); /* A <- U^-H A */
  /* A <- A U^-1 : rows of A are the "bands" here, so apply the right-solve to the n x n block */
  orc_trsm_right_upper(n, n, A, lda, B, ldb);
  for (int64_t j = 0; j < n; ++j) /* symmetrise the rounding noise: C = (C + C^H)/2 */
    for (int64_t i = 0; i <= j; ++i) {
      cplx m = 0.5 * (A[i + j * lda] + conj(A[j + i * lda]));
      A[i + j * lda] = m;
      A[j + i * lda] = conj(m);
    }
  orc_heev_jacobi(n, A, lda, w, X, ldx);          /* C Y = Y Lambda */
  trsm_left_upper(n, n, B, ldb, X, ldx);          /* X = U^-1 Y */
  return 0;
}
