/*
 * pw_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU oracle for the hot path of arxiv/paper_2604_11139
 * ("GPU acceleration of plane-wave DFT calculations in ABINIT"): the matrix-free application of the
 * plane-wave Hamiltonian H = 1/2|k+G|^2 + V_loc + sum_i |p_i> D_i <p_i| to a block of bands
 * ("HX(N,m)", 327-335 section 4.2, 397), the scaled Chebyshev filter built on it
 * (Algorithm 7, 246 section 3.3, 576-593 Algorithm 12 with S = I; recurrence from
 * BASELINE.json north_star and the paper's reference [61]), and the Rayleigh-Ritz Gram
 * product Psi^H (H Psi) (Algorithm 5 step 1, 227).
 *
 * It is written from the definitions, in FP64 (dot products accumulated in long double), with no blocking,
 * fusion or reordering: scatter the G-sphere into the full FFT box, full unpruned 3-D transforms
 * (direct O(n^2)-per-axis DFT when every box side is <= 16, otherwise a simple recursive mixed-radix
 * Cooley-Tukey written only for this file), pointwise multiply, transform back, gather; projector sums as
 * plain loops.  It shares no code, header, table or constant with the CUDA path under
 * paper_2604_11139_b200/csrc and is never linked into, imported by or called from it.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * Pins (tests/test_oracle_pins.py): plane-wave eigenvalue in constant V0, shift theorem, oracle FFT vs direct
 * DFT vs numpy.fft, Hermiticity, dense H built from the convolution theorem with numpy, Chebyshev closed form
 * on exact eigenvectors, degree edge cases, Gram identities, band independence, translation covariance.
 * Nothing here is "parity unpinned".
 *
 * Layout: a block is column-major npw x nband (band b at psi + b*ld, plane-wave index contiguous),
 * complex128 = (re, im) pairs.  Projectors column-major npw x nproj.  V_loc index i1 + n1*(i2 + n2*i3).
 * FFT convention (reading R6): G->r is exp(+2 pi i m.r/n) unnormalised, r->G is exp(-...) with 1/F.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double _Complex cplx;

#define ORC_TERM_KIN 1
#define ORC_TERM_LOC 2
#define ORC_TERM_NL 4

static const long double ORC_PI = 3.14159265358979323846264338327950288L;

/* ---------------------------------------------------------------------------------------------------
 * 1-D transforms.  out[k] = sum_n in[n] exp(sign * 2 pi i n k / N), no normalisation.
 * ------------------------------------------------------------------------------------------------- */

/* w[j] = exp(sign 2 pi i j / n), j = 0..n-1, argument reduced exactly to an octant-free integer ratio. */
static void root_table(int n, int sign, cplx *w) {
  for (int j = 0; j < n; ++j) {
    long double ang = 2.0L * ORC_PI * (long double)j / (long double)n;
    w[j] = (double)cosl(ang) + I * (double)(sign * sinl(ang));
  }
}

/* direct O(n^2) DFT (the definition) */
void orc_dft1d(int n, int sign, const cplx *in, cplx *out) {
  cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)n);
  root_table(n, sign, w);
  for (int k = 0; k < n; ++k) {
    long double sr = 0.0L, si = 0.0L;
    for (int j = 0; j < n; ++j) {
      cplx t = w[(int)(((long)j * k) % n)];
      sr += (long double)creal(in[j]) * creal(t) - (long double)cimag(in[j]) * cimag(t);
      si += (long double)creal(in[j]) * cimag(t) + (long double)cimag(in[j]) * creal(t);
    }
    out[k] = (double)sr + I * (double)si;
  }
  free(w);
}

static int smallest_factor(int n) {
  if (n % 2 == 0) return 2;
  for (int p = 3; p * p <= n; p += 2)
    if (n % p == 0) return p;
  return n;
}

/* Recursive decimation-in-time Cooley-Tukey, n = p*m with p the smallest prime factor:
 *   X[k + m j] = sum_{r<p} w_n^{r(k + m j)} Y_r[k],   Y_r = DFT_m of the samples in[r], in[r+p], ...
 * `w` is the root table of the top-level length n0; w_n^t = w[t * (n0/n) mod n0]. */
static void fft_rec(int n, const cplx *in, int stride, cplx *out, const cplx *w, int n0) {
  if (n == 1) {
    out[0] = in[0];
    return;
  }
  int p = smallest_factor(n), m = n / p, step = n0 / n;
  for (int r = 0; r < p; ++r) fft_rec(m, in + (size_t)r * stride, stride * p, out + (size_t)r * m, w, n0);
  cplx t[p], x[p];
  for (int k = 0; k < m; ++k) {
    for (int r = 0; r < p; ++r) t[r] = out[r * m + k];
    for (int j = 0; j < p; ++j) {
      cplx s = 0.0;
      int kk = k + m * j;
      for (int r = 0; r < p; ++r) s += t[r] * w[(int)((((long)r * kk) % n) * step)];
      x[j] = s;
    }
    for (int j = 0; j < p; ++j) out[k + m * j] = x[j];
  }
}

/* simple FFT for any n (prime factors handled generically; intended for 2,3,5-smooth n) */
void orc_fft1d(int n, int sign, const cplx *in, cplx *out) {
  cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)n);
  root_table(n, sign, w);
  fft_rec(n, in, 1, out, w, n);
  free(w);
}

/* ---------------------------------------------------------------------------------------------------
 * 3-D transform of a full box, box[i1 + n1*(i2 + n2*i3)], axis by axis, line by line.
 * use_fft = 0 : direct DFT on every line;  1 : orc_fft1d;  -1 : direct iff all sides <= 16.
 * ------------------------------------------------------------------------------------------------- */
void orc_dft3d(const int dims[3], int sign, cplx *box, int use_fft) {
  int n1 = dims[0], n2 = dims[1], n3 = dims[2];
  if (use_fft < 0) use_fft = !(n1 <= 16 && n2 <= 16 && n3 <= 16);
  int nmax = n1 > n2 ? n1 : n2;
  if (n3 > nmax) nmax = n3;
  cplx *lin = (cplx *)malloc(sizeof(cplx) * (size_t)nmax);
  cplx *lout = (cplx *)malloc(sizeof(cplx) * (size_t)nmax);
  int n[3] = {n1, n2, n3};
  size_t str[3] = {1, (size_t)n1, (size_t)n1 * n2};
  for (int ax = 0; ax < 3; ++ax) {
    int a1 = (ax + 1) % 3, a2 = (ax + 2) % 3;
    for (int j = 0; j < n[a2]; ++j)
      for (int i = 0; i < n[a1]; ++i) {
        cplx *base = box + i * str[a1] + j * str[a2];
        for (int t = 0; t < n[ax]; ++t) lin[t] = base[t * str[ax]];
        if (use_fft)
          orc_fft1d(n[ax], sign, lin, lout);
        else
          orc_dft1d(n[ax], sign, lin, lout);
        for (int t = 0; t < n[ax]; ++t) base[t * str[ax]] = lout[t];
      }
  }
  free(lin);
  free(lout);
}

/* ---------------------------------------------------------------------------------------------------
 * Hamiltonian pieces (one band).  SURVEY.md section 8c items 1-4.
 * ------------------------------------------------------------------------------------------------- */

/* kin(G) = 1/2 |B (k + n_G)|^2, B = 2 pi (A^-1)^T, lattice rows a_i. */
void orc_kinetic(const double lattice[9], const double kpt[3], int64_t npw, const int32_t *gvec, double *kin) {
  const double *a = lattice;
  double det = a[0] * (a[4] * a[8] - a[5] * a[7]) - a[1] * (a[3] * a[8] - a[5] * a[6]) +
               a[2] * (a[3] * a[7] - a[4] * a[6]);
  /* rows of B: b_i = 2 pi (a_j x a_k) / det */
  double B[9];
  double twopi = (double)(2.0L * ORC_PI);
  B[0] = twopi * (a[4] * a[8] - a[5] * a[7]) / det;
  B[1] = twopi * (a[5] * a[6] - a[3] * a[8]) / det;
  B[2] = twopi * (a[3] * a[7] - a[4] * a[6]) / det;
  B[3] = twopi * (a[7] * a[2] - a[8] * a[1]) / det;
  B[4] = twopi * (a[8] * a[0] - a[6] * a[2]) / det;
  B[5] = twopi * (a[6] * a[1] - a[7] * a[0]) / det;
  B[6] = twopi * (a[1] * a[5] - a[2] * a[4]) / det;
  B[7] = twopi * (a[2] * a[3] - a[0] * a[5]) / det;
  B[8] = twopi * (a[0] * a[4] - a[1] * a[3]) / det;
  for (int64_t g = 0; g < npw; ++g) {
    double c0 = kpt[0] + gvec[3 * g + 0], c1 = kpt[1] + gvec[3 * g + 1], c2 = kpt[2] + gvec[3 * g + 2];
    double qx = c0 * B[0] + c1 * B[3] + c2 * B[6];
    double qy = c0 * B[1] + c1 * B[4] + c2 * B[7];
    double qz = c0 * B[2] + c1 * B[5] + c2 * B[8];
    kin[g] = 0.5 * (qx * qx + qy * qy + qz * qz);
  }
}

static inline int wrap(int n, int nbox) {
  int r = n % nbox;
  return r < 0 ? r + nbox : r;
}

/* w_loc = gather( (1/F) DFT^-( V_loc . DFT^+( scatter(psi) ) ) ).   `box` is caller scratch of F entries. */
static void local_one(const int dims[3], int64_t npw, const int32_t *gvec, const double *vloc, const cplx *psi,
                      cplx *out, cplx *box, int use_fft) {
  size_t n1 = dims[0], n2 = dims[1], n3 = dims[2], F = n1 * n2 * n3;
  memset(box, 0, sizeof(cplx) * F);
  for (int64_t g = 0; g < npw; ++g) {
    size_t i1 = wrap(gvec[3 * g], dims[0]), i2 = wrap(gvec[3 * g + 1], dims[1]), i3 = wrap(gvec[3 * g + 2], dims[2]);
    box[i1 + n1 * (i2 + n2 * i3)] = psi[g];
  }
  orc_dft3d(dims, +1, box, use_fft);
  for (size_t r = 0; r < F; ++r) box[r] *= vloc[r];
  orc_dft3d(dims, -1, box, use_fft);
  double inv = 1.0 / (double)F;
  for (int64_t g = 0; g < npw; ++g) {
    size_t i1 = wrap(gvec[3 * g], dims[0]), i2 = wrap(gvec[3 * g + 1], dims[1]), i3 = wrap(gvec[3 * g + 2], dims[2]);
    out[g] = box[i1 + n1 * (i2 + n2 * i3)] * inv;
  }
}

/* w_nl(G) = sum_i P[G,i] D_i c_i,  c_i = sum_G conj(P[G,i]) psi(G)   (PAPER.md:333 with diagonal D). */
static void nonlocal_one(int64_t npw, int64_t nproj, const cplx *proj, int64_t ldp, const double *dij,
                         const cplx *psi, cplx *out) {
  for (int64_t g = 0; g < npw; ++g) out[g] = 0.0;
  for (int64_t i = 0; i < nproj; ++i) {
    const cplx *p = proj + i * ldp;
    long double cr = 0.0L, ci = 0.0L;
    for (int64_t g = 0; g < npw; ++g) { /* conj(p) * psi */
      cr += (long double)creal(p[g]) * creal(psi[g]) + (long double)cimag(p[g]) * cimag(psi[g]);
      ci += (long double)creal(p[g]) * cimag(psi[g]) - (long double)cimag(p[g]) * creal(psi[g]);
    }
    cplx dc = dij[i] * ((double)cr + I * (double)ci);
    for (int64_t g = 0; g < npw; ++g) out[g] += p[g] * dc;
  }
}

/* H psi for a block; `terms` selects kinetic / local / nonlocal (all = 7).  Bands are independent
 * (PAPER.md:224, 329), so the loop over bands is the only parallelism used. */
int orc_apply_h(const double lattice[9], const double kpt[3], const int32_t dims[3], int64_t npw,
                const int32_t *gvec, const double *vloc, int64_t nproj, const cplx *proj, int64_t ldp,
                const double *dij, int64_t nband, const cplx *psi, int64_t ldpsi, cplx *hpsi, int64_t ldh,
                int terms, int use_fft) {
  size_t F = (size_t)dims[0] * dims[1] * dims[2];
  double *kin = (double *)malloc(sizeof(double) * (size_t)npw);
  if (!kin) return -1;
  orc_kinetic(lattice, kpt, npw, gvec, kin);
  int fail = 0;
#pragma omp parallel
  {
    cplx *box = (cplx *)malloc(sizeof(cplx) * F);
    cplx *tmp = (cplx *)malloc(sizeof(cplx) * (size_t)npw);
    if (!box || !tmp) {
#pragma omp atomic write
      fail = 1;
    } else {
#pragma omp for schedule(dynamic, 1)
      for (int64_t b = 0; b < nband; ++b) {
        const cplx *x = psi + b * ldpsi;
        cplx *y = hpsi + b * ldh;
        for (int64_t g = 0; g < npw; ++g) y[g] = (terms & ORC_TERM_KIN) ? kin[g] * x[g] : 0.0;
        if (terms & ORC_TERM_LOC) {
          local_one(dims, npw, gvec, vloc, x, tmp, box, use_fft);
          for (int64_t g = 0; g < npw; ++g) y[g] += tmp[g];
        }
        if ((terms & ORC_TERM_NL) && nproj > 0) {
          nonlocal_one(npw, nproj, proj, ldp, dij, x, tmp);
          for (int64_t g = 0; g < npw; ++g) y[g] += tmp[g];
        }
      }
    }
    free(box);
    free(tmp);
  }
  free(kin);
  return fail ? -1 : 0;
}

/* Scaled Chebyshev filter, in place (north_star; [61] PAPER.md:662):
 *   e = (b-a)/2, c = (b+a)/2, sigma_1 = e/(a0-c), Y_0 = Psi, Y_1 = (sigma_1/e)(H - c) Y_0,
 *   sigma_{j+1} = 1/(2/sigma_1 - sigma_j),  Y_{j+1} = (2 sigma_{j+1}/e)(H - c) Y_j - sigma_j sigma_{j+1} Y_{j-1}.
 * Returns Y_degree in psi.  degree == 0 is the identity. */
int orc_cheb_filter(const double lattice[9], const double kpt[3], const int32_t dims[3], int64_t npw,
                    const int32_t *gvec, const double *vloc, int64_t nproj, const cplx *proj, int64_t ldp,
                    const double *dij, int64_t nband, cplx *psi, int64_t ld, int degree, double a, double b,
                    double a0, int use_fft) {
  if (degree < 0 || !(b > a) || !(a0 < a)) return -2;
  if (degree == 0) return 0;
  size_t blk = (size_t)npw * (size_t)nband;
  cplx *yprev = (cplx *)malloc(sizeof(cplx) * blk);
  cplx *ycur = (cplx *)malloc(sizeof(cplx) * blk);
  cplx *hy = (cplx *)malloc(sizeof(cplx) * blk);
  if (!yprev || !ycur || !hy) return -1;
  double e = 0.5 * (b - a), c = 0.5 * (b + a), sigma1 = e / (a0 - c), sigma = sigma1;
  for (int64_t bb = 0; bb < nband; ++bb)
    for (int64_t g = 0; g < npw; ++g) yprev[bb * npw + g] = psi[bb * ld + g];
  int rc = orc_apply_h(lattice, kpt, dims, npw, gvec, vloc, nproj, proj, ldp, dij, nband, yprev, npw, hy, npw, 7,
                       use_fft);
  for (size_t i = 0; i < blk; ++i) ycur[i] = (sigma1 / e) * (hy[i] - c * yprev[i]);
  for (int j = 1; j < degree && rc == 0; ++j) {
    double sigma_new = 1.0 / (2.0 / sigma1 - sigma);
    rc = orc_apply_h(lattice, kpt, dims, npw, gvec, vloc, nproj, proj, ldp, dij, nband, ycur, npw, hy, npw, 7,
                     use_fft);
    for (size_t i = 0; i < blk; ++i) {
      cplx ynew = (2.0 * sigma_new / e) * (hy[i] - c * ycur[i]) - (sigma * sigma_new) * yprev[i];
      yprev[i] = ycur[i];
      ycur[i] = ynew;
    }
    sigma = sigma_new;
  }
  for (int64_t bb = 0; bb < nband; ++bb)
    for (int64_t g = 0; g < npw; ++g) psi[bb * ld + g] = ycur[bb * npw + g];
  free(yprev);
  free(ycur);
  free(hy);
  return rc;
}

/* G[i,j] = sum_g conj(X[g,i]) Y[g,j], G column-major nx x ny with leading dimension ldg.
 * The paper writes X^T Y; for complex Psi and a Hermitian H_Psi that is X^H Y. */
void orc_gram(int64_t npw, int64_t nx, const cplx *X, int64_t ldx, int64_t ny, const cplx *Y, int64_t ldy, cplx *G,
              int64_t ldg) {
#pragma omp parallel for collapse(2) schedule(static)
  for (int64_t j = 0; j < ny; ++j)
    for (int64_t i = 0; i < nx; ++i) {
      const cplx *x = X + i * ldx, *y = Y + j * ldy;
      long double sr = 0.0L, si = 0.0L;
      for (int64_t g = 0; g < npw; ++g) {
        sr += (long double)creal(x[g]) * creal(y[g]) + (long double)cimag(x[g]) * cimag(y[g]);
        si += (long double)creal(x[g]) * cimag(y[g]) - (long double)cimag(x[g]) * creal(y[g]);
      }
      G[i + j * ldg] = (double)sr + I * (double)si;
    }
}
