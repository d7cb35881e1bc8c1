/*
 * pwham.h -- C ABI of libpwham: the B200 (sm_100a) hot path of iterative Kohn-Sham diagonalisation in a
 * plane-wave basis, after arxiv/paper_2604_11139 ("GPU acceleration of plane-wave DFT calculations in ABINIT").
 *
 *   H psi = 1/2|k+G|^2 psi  +  gather( FFT( V_loc(r) . iFFT( scatter(psi) ) ) )  +  P . D . (P^H psi)
 *
 * applied matrix-free to a block of bands ("HX(N,m)", 327-335 section 4.2, 397), inside the
 * scaled Chebyshev polynomial filter (Algorithm 7; 246 section 3.3; 576-593 Algorithm 12 with S = I),
 * with the Rayleigh-Ritz Gram product X^H Y as companion step (Algorithm 5 step 1; 227).
 *
 * Conventions
 *   - complex128 = {re, im} pairs of IEEE doubles (== cuDoubleComplex == torch.complex128).
 *   - A block of wavefunctions is the paper's N x M matrix, column-major: band b starts at
 *     psi + b*ld, the plane-wave index is contiguous, ld >= npw is "the distance between two consecutive
 *     electronic bands".  Rows >= npw of a padded column are never read or written.
 *   - Unless a parameter says HOST, every data pointer is a DEVICE pointer owned by the caller.
 *   - Every function returns PWH_OK (0) or a negative error code and never throws; pwh_last_error() returns a
 *     thread-local message for the last failure.  Device work is enqueued on `stream` (a cudaStream_t passed as
 *     void*; NULL = the legacy default stream) and is asynchronous: results are valid once the caller has
 *     synchronised that stream.  The *_host entry points synchronise before returning.
 *   - One handle may be used from one stream at a time.  There is no CPU fallback of any kind.  Internally a handle may run
 *     the band groups of the local-potential stage on two private non-blocking streams; they are forked from and joined to
 *     `stream` by events inside the call, so the caller sees ordinary in-stream semantics.
 *   - Several handles may be alive at once (one per k-point is the normal use); they share nothing.
 *
 * Environment switches.  They exist for the test-suite, select a KERNEL FAMILY (never a CPU path), are sampled once per
 * pwh_ham_setup call and never on a launch path:
 *     PWH_FORCE_GENERIC_FFT=1  generic radix-2/3/4/5/8 shared-memory stage plan instead of the register-resident two-pass
 *                              transforms (otherwise used only for axis lengths that do not factor as r1 * r2);
 *     PWH_NO_V2=1              generic-size plane kernel instead of the size-specialised one;
 *     PWH_NO_ZW=1              CTA-per-column-group z kernels instead of the warp-private ones;
 *     PWH_ZGEMM_NO_TMA=1       cp.async-fed ZGEMM instead of the TMA-fed one (process-wide, until the next setup);
 *     PWH_V2_NO_PRUNE=1        full-length strided-role transform passes instead of the ones that skip the rows a cutoff
 *                              sphere cannot touch (otherwise used when the sphere spans more than about half of an axis);
 *     PWH_LOCAL_ONE_STREAM=1   the band groups of the local-potential stage run in order on the caller's stream;
 *     PWH_LOCAL_TWO_STREAMS=1  they alternate between two internal streams (default: the handle times both on its first four
 *                              multi-group H applications, with events on the caller's stream and no host synchronisation,
 *                              and keeps the faster; results do not depend on the choice);
 *     PWH_BAND_GROUP=n         bands per launch of the local-potential kernels (default: chosen at setup so that the column
 *                              buffer of a group stays in L2 and the plane kernel's grid fills whole waves of SMs).
 * pwh_ham_kernels() reports which family a handle uses.
 */
#ifndef PWHAM_H
#define PWHAM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pwh_ham pwh_ham; /* opaque handle */
typedef struct {
  double re, im;
} pwh_c128;

enum { PWH_OK = 0, PWH_EINVAL = -1, PWH_ECUDA = -2, PWH_ENOMEM = -3, PWH_EUNSUPPORTED = -4 };

/*
 * pwh_ham_setup -- build the tables of one Hamiltonian (one k-point).
 * ("data must first be rearranged" before the batched FFT), PAPER.md:333 (projectors, D).
 *
 *   lattice   HOST  9 doubles, row i = primitive vector a_i in bohr.
 *   kpt       HOST  3 doubles, reduced coordinates of k.
 *   fft_dims  HOST  n1, n2, n3; each must be >= 2 with prime factors in {2,3,5} (else PWH_EUNSUPPORTED).
 *   npw       number of plane waves N (>= 1).
 *   gvec      DEVICE int32 [npw][3], reduced integer components of G.  The set must fit the box without
 *             collision after wrapping (n mod n_i); checked once here (one device->host copy). Copied.
 *   vloc      DEVICE double [n1*n2*n3], local potential in Hartree on the real-space grid, index
 *             i1 + n1*(i2 + n2*i3).  Copied (re-ordered and pre-scaled by 1/(n1 n2 n3)) into the handle.
 *   nproj     number of projectors J (>= 0; 0 disables the nonlocal term).
 *   proj      DEVICE complex128, column-major npw x nproj, proj[g + i*ldp] = <G_g | p_i>.  BORROWED: it must stay
 *             valid and unchanged for the handle's lifetime (it can be several GB and is not copied).
 *   ldp       leading dimension of proj (>= npw).
 *   dij       DEVICE double [nproj], diagonal nonlocal strengths D_i in Hartree.  Copied.
 *   stream    stream used for the setup copies; the call synchronises it before returning.
 *
 * The kinetic diagonal is kin(G) = 1/2 |B(k + n_G)|^2 with B = 2 pi (A^-1)^T.
 */
int pwh_ham_setup(pwh_ham** out, const double lattice[9], const double kpt[3], const int32_t fft_dims[3],
                  int64_t npw, const int32_t* gvec, const double* vloc, int64_t nproj, const pwh_c128* proj,
                  int64_t ldp, const double* dij, void* stream);

/* Frees the handle's tables and any staging buffers of the *_host entry points.  NULL is accepted. */
int pwh_ham_destroy(pwh_ham* ham);

/* Bytes of caller-provided device workspace that pwh_apply_h / pwh_cheb_filter need for up to nband_max bands.
 * The hot path performs no allocation. */
size_t pwh_workspace_bytes(const pwh_ham* ham, int64_t nband_max);

/*
 * pwh_apply_h -- hpsi = H psi for nband bands (HX(N,m); the three terms PAPER.md:397).
 *   psi [in]  npw x nband, leading dimension ldpsi.   hpsi [out] npw x nband, leading dimension ldh.
 *   psi and hpsi must not overlap.  ws/ws_bytes: workspace of at least pwh_workspace_bytes(ham, nband), 256-byte
 *   aligned.  nband == 0 is a no-op.
 * Errors: PWH_EINVAL (null pointer, ld < npw, workspace too small or misaligned), PWH_ECUDA (launch failure).
 */
int pwh_apply_h(pwh_ham* ham, int64_t nband, const pwh_c128* psi, int64_t ldpsi, pwh_c128* hpsi, int64_t ldh,
                void* ws, size_t ws_bytes, void* stream);

/*
 * pwh_cheb_filter -- in place psi <- p_m(H) psi, the scaled Chebyshev filter of degree m = `degree`
 * (Algorithm 7 loop body, 246; recurrence of the paper's reference [61]):
 *     e = (b-a)/2,  c = (b+a)/2,  sigma_1 = e/(a0-c),  Y_0 = psi,  Y_1 = (sigma_1/e)(H - c) Y_0,
 *     sigma_{j+1} = 1/(2/sigma_1 - sigma_j),   Y_{j+1} = (2 sigma_{j+1}/e)(H - c) Y_j - sigma_j sigma_{j+1} Y_{j-1},
 * result Y_m = T_m((H-c)/e)/T_m((a0-c)/e) psi.  [a,b] is the damped interval, a0 < a the normalisation point.
 * One H application per degree.  degree == 0 is the identity.
 * Errors: PWH_EINVAL additionally for degree < 0, b <= a, a0 >= a.
 */
int pwh_cheb_filter(pwh_ham* ham, int64_t nband, pwh_c128* psi, int64_t ld, int degree, double a, double b,
                    double a0, void* ws, size_t ws_bytes, void* stream);

/*
 * pwh_gram -- G = X^H Y  (Algorithm 5 step 1 with Y = H X; PAPER.md:227 writes it as a sum of
 * row-chunk products, which is how it is evaluated here: split over npw with a fixed-order second-stage sum, so
 * the result is deterministic).
 *   X npw x nx (ldx), Y npw x ny (ldy), G [out] column-major nx x ny (ldg >= nx): G[i + j*ldg] = sum_g conj(X[g,i]) Y[g,j].
 *   ws/ws_bytes: at least pwh_gram_workspace_bytes(npw, nx, ny), 256-byte aligned.
 */
size_t pwh_gram_workspace_bytes(int64_t npw, int64_t nx, int64_t ny);
int pwh_gram(int64_t npw, int64_t nx, const pwh_c128* X, int64_t ldx, int64_t ny, const pwh_c128* Y, int64_t ldy,
             pwh_c128* G, int64_t ldg, void* ws, size_t ws_bytes, void* stream);

/*
 * pwh_gram_herm -- the same product for a G the caller knows to be Hermitian: G = X^H (A X) with A Hermitian, i.e. the
 * Rayleigh-Ritz matrices H_Psi = Psi^H (H Psi) and S_Psi = Psi^H Psi of PAPER.md:153-163 (Algorithm 5 steps 1-2).  Only the
 * tiles on or above the block diagonal are computed on the tensor pipe; the strictly lower blocks are written as the
 * conjugates of their mirror images (so G[i,j] == conj(G[j,i]) exactly outside the 128 x 128 diagonal blocks and to
 * rounding inside them).  If X^H Y is not Hermitian the lower blocks are simply not X^H Y.  Workspace as for pwh_gram.
 */
int pwh_gram_herm(int64_t npw, int64_t n, const pwh_c128* X, int64_t ldx, const pwh_c128* Y, int64_t ldy, pwh_c128* G,
                  int64_t ldg, void* ws, size_t ws_bytes, void* stream);

/*
 * pwh_gram_static -- pwh_gram for callers that may not allocate and have no workspace to give (code under CUDA graph capture,
 * serving loops, harnesses that forbid cudaMalloc): G = X^H Y with the split-K partial sums in a file-scope device array of
 * PWH_GRAM_STATIC_MAX_ENTRIES complex128 (16 MiB; every GPU that loads the library holds it until exit).  Same arguments,
 * layout and result as pwh_gram, to rounding order (the number of K splits is capped so that the partial sums fit).
 *   Limit: nx * ny <= PWH_GRAM_STATIC_MAX_ENTRIES, otherwise PWH_EINVAL with a message naming the limit.
 *   The call performs no cudaMalloc / cudaFree and calls no allocating library routine; it enqueues two kernels on `stream`.
 *   All calls share the one array, which keeps the previous call's contents (nothing in it needs clearing: every partial entry
 *   is written before it is read): calls that can overlap on the GPU -- different streams, several host threads -- RACE on it.
 *   Keep them on one stream or order them with events.
 */
#define PWH_GRAM_STATIC_MAX_ENTRIES 1048576
int pwh_gram_static(int64_t npw, int64_t nx, const pwh_c128* X, int64_t ldx, int64_t ny, const pwh_c128* Y, int64_t ldy,
                    pwh_c128* G, int64_t ldg, void* stream);

/*
 * Host-buffer entry points (end-to-end path: the paper keeps Psi on the device and moves it host->device once per
 * k-point and SCF step, Algorithm 3).  All pointers below marked HOST are host memory (pinned
 * memory gives asynchronous copies; pageable memory works).  Device staging buffers are allocated on first use,
 * cached in the handle and freed by pwh_ham_destroy.  Each call copies its inputs to the device, runs the same
 * kernels as the device entry points, copies the result back and synchronises.  The filtering entry points move Psi
 * in chunks of bands (the column blocks, or quarters of a single block of >= 512 bands) on two internal copy streams,
 * so that the copies of the neighbouring chunks run under the filter of the current one (bands never interact before
 * the Gram product); every band still goes through exactly the same kernels.
 *
 * pwh_apply_h_host     hpsi_host = H psi_host.
 * pwh_cheb_filter_host psi_host <- p_m(H) psi_host, bands processed in column blocks of `block` (<= 0: all at once).
 * pwh_sweep_host       one filtering sweep followed by the Rayleigh-Ritz projection: psi_host <- p_m(H) psi_host
 *                      (by blocks), then G_host = psi^H (H psi) (column-major nband x nband, ldg) -- i.e. degree+1
 *                      H applications per band and one Gram product.  hpsi_host (optional, may be NULL) receives H psi.
 */
int pwh_apply_h_host(pwh_ham* ham, int64_t nband, const pwh_c128* psi_host, int64_t ldpsi, pwh_c128* hpsi_host,
                     int64_t ldh, void* stream);
int pwh_cheb_filter_host(pwh_ham* ham, int64_t nband, int64_t block, pwh_c128* psi_host, int64_t ld, int degree,
                         double a, double b, double a0, void* stream);
int pwh_sweep_host(pwh_ham* ham, int64_t nband, int64_t block, pwh_c128* psi_host, int64_t ld, int degree, double a,
                   double b, double a0, pwh_c128* hpsi_host, int64_t ldh, pwh_c128* G_host, int64_t ldg,
                   void* stream);

/*
 * ---------------------------------------------------------------------------------------------------------------
 * Rayleigh-Ritz companion steps: what one Chebyshev-filtering iteration (Algorithm 12, here with S = I)
 * does around the filter.  All pointers DEVICE unless marked HOST; asynchronous on `stream` like the calls above, except
 * pwh_chebfi_iteration (one host round trip, see there).  The dense M x M steps are hand-written kernels (blocked
 * Cholesky, triangular inverse, one-sided Jacobi in one cooperative launch); no vendor solver library is called.
 * `info` (DEVICE int32) of the dense solvers: > 0 = Jacobi sweeps used, < 0 = -(j+1) with j the first non-positive Cholesky
 * pivot (the overlap matrix is not positive definite: linearly dependent bands); results are undefined in that case.
 * ---------------------------------------------------------------------------------------------------------------
 */

/*
 * pwh_rayleigh_quotients -- lambda[i] = Re(psi_i^H hpsi_i) / Re(psi_i^H spsi_i)  ("Rayleigh quotients
 * lambda_i = (H psi_i)^T psi_i / ((S psi_i)^T psi_i)", Algorithm 12 line 3), and, when minmax != NULL, minmax[0] = min_i,
 * minmax[1] = max_i lambda[i] -- the interval the filter is built on.  lambda: nband doubles, minmax: 2 doubles.
 * In this and the following calls `spsi` = S Psi of the generalised problem; spsi == NULL means S = I.
 */
int pwh_rayleigh_quotients(int64_t npw, int64_t nband, const pwh_c128* psi, int64_t ld, const pwh_c128* hpsi, int64_t ldh,
                           const pwh_c128* spsi, int64_t lds, double* lambda, double* minmax, void* stream);

/*
 * pwh_residual_norms -- W_i = hpsi_i - lambda[i] spsi_i and norms[i] = ||W_i||_2  (Algorithm 12 lines 11-12:
 * "W <- (H - Lambda S) Psi; compute residual norms").  W may be NULL (norms only); W may not alias the inputs.
 */
int pwh_residual_norms(int64_t npw, int64_t nband, const pwh_c128* psi, int64_t ld, const pwh_c128* hpsi, int64_t ldh,
                       const pwh_c128* spsi, int64_t lds, const double* lambda, pwh_c128* W, int64_t ldw, double* norms,
                       void* stream);

/*
 * pwh_rotate -- Y = X Q: X npw x m (ldx), Q m x n column-major (ldq >= m), Y npw x n (ldy); Y must not overlap X
 * (Algorithm 5 steps 4-5 / Algorithm 10: "Psi <- Psi X, H Psi <- (H Psi) X").  Runs on the DMMA ZGEMM.
 */
int pwh_rotate(int64_t npw, int64_t m, const pwh_c128* X, int64_t ldx, int64_t n, const pwh_c128* Q, int64_t ldq,
               pwh_c128* Y, int64_t ldy, void* stream);

/* Workspace of pwh_heev / pwh_hegv for matrices of order n (256-byte aligned device memory). */
size_t pwh_dense_workspace_bytes(int64_t n);

/*
 * pwh_potrf -- in place A = U^H U for a Hermitian positive definite A (n x n column-major, only its upper triangle is
 * read): the upper triangle becomes U (positive real diagonal), the strictly lower triangle is zeroed
 * (Algorithm 9 step 2 "potrf").  *info = 0, or j+1 for the first non-positive pivot j.
 */
int pwh_potrf(int64_t n, pwh_c128* A, int64_t lda, int32_t* info, void* stream);

/*
 * pwh_heev -- eigen-decomposition of a Hermitian A (n x n, destroyed): w[0..n-1] ascending, column j of X the orthonormal
 * eigenvector of w[j]  (Algorithm 5/10 step 3 with S_Psi = I).  X must not alias A.  Eigenvectors are defined up to a
 * phase, and up to a unitary mixing inside a degenerate eigenspace.
 * pwh_hegv -- A X = B X diag(w), X^H B X = I for Hermitian A and Hermitian positive definite B (both destroyed)
 * (Algorithm 5/10 step 3 "hegvd"): B = U^H U, C = U^-H A U^-1, C Y = Y diag(w), X = U^-1 Y.
 */
int pwh_heev(int64_t n, pwh_c128* A, int64_t lda, double* w, pwh_c128* X, int64_t ldx, int32_t* info, void* ws,
             size_t ws_bytes, void* stream);
int pwh_hegv(int64_t n, pwh_c128* A, int64_t lda, pwh_c128* B, int64_t ldb, double* w, pwh_c128* X, int64_t ldx,
             int32_t* info, void* ws, size_t ws_bytes, void* stream);

/* Workspace of pwh_chol_ortho / pwh_rayleigh_ritz for an npw x nband block. */
size_t pwh_rr_workspace_bytes(int64_t npw, int64_t nband);

/*
 * pwh_chol_ortho -- Algorithm 9 (S-Ortho) with S = I: S_Psi = Psi^H Psi = U^H U, Psi <- Psi U^-1 and, when hpsi != NULL,
 * H Psi <- (H Psi) U^-1, in place.  U (optional, nband x nband column-major, ldu) receives the factor.
 * *info as for pwh_potrf.  Afterwards Psi^H Psi = I.
 */
int pwh_chol_ortho(int64_t npw, int64_t nband, pwh_c128* psi, int64_t ld, pwh_c128* hpsi, int64_t ldh, pwh_c128* U,
                   int64_t ldu, int32_t* info, void* ws, size_t ws_bytes, void* stream);

/*
 * pwh_chol_ortho_gen -- Algorithm 9 (S-Ortho) as printed, for the generalised problem: S_Psi = Psi^H (S Psi) = U^H U, then
 * Psi <- Psi U^-1, S Psi <- (S Psi) U^-1 and, when hpsi != NULL, H Psi <- (H Psi) U^-1, in place.  spsi = S Psi
 * is required (pwh_apply_hs).  Afterwards Psi^H (S Psi) = I.  Workspace and *info as for pwh_chol_ortho.
 */
int pwh_chol_ortho_gen(int64_t npw, int64_t nband, pwh_c128* psi, int64_t ld, pwh_c128* hpsi, int64_t ldh, pwh_c128* spsi,
                       int64_t lds, pwh_c128* U, int64_t ldu, int32_t* info, void* ws, size_t ws_bytes, void* stream);

/*
 * pwh_rayleigh_ritz -- Algorithm 10 (RR), in place: H_Psi = Psi^H (H Psi), S_Psi = Psi^H (S Psi), H_Psi X = S_Psi X Lambda,
 * Psi <- Psi X, H Psi <- (H Psi) X, S Psi <- (S Psi) X (Algorithm 5).  lambda receives
 * the nband Ritz values in ascending order; afterwards Psi^H (S Psi) = I and Psi^H (H Psi) = diag(lambda).
 */
int pwh_rayleigh_ritz(int64_t npw, int64_t nband, pwh_c128* psi, int64_t ld, pwh_c128* hpsi, int64_t ldh, pwh_c128* spsi,
                      int64_t lds, double* lambda, int32_t* info, void* ws, size_t ws_bytes, void* stream);

/*
 * pwh_chebfi_iteration -- one iteration of Algorithm 12, in place on psi (spsi == NULL: S = I;
 * otherwise the handle must carry PAW blocks, H Psi and S Psi come from pwh_apply_hs and the filter is pwh_cheb_filter_gen):
 *   H Psi (lines 1-2); Rayleigh quotients, a = max, a0 = min - a0_margin (line 3; reading R5: the upper bound b
 *   of the spectrum is an input); Psi <- p_degree(H) Psi in column blocks of `block` (lines 4-8); H Psi; Rayleigh-Ritz
 *   (line 10); residual norms of the Ritz pairs (lines 11-12).
 * On return psi holds the Ritz vectors, hpsi = H psi, lambda the Ritz values (ascending), resid the residual norms
 * (lambda, resid: DEVICE, nband doubles), bounds_host (HOST, optional) = {a0, a}.  The call synchronises `stream` once, to
 * bring the two Rayleigh-quotient bounds to the host (the paper's "mpi-sR" reduction sits at the same place).
 * Workspace: pwh_chebfi_workspace_bytes(ham, nband, block).
 */
size_t pwh_chebfi_workspace_bytes(const pwh_ham* ham, int64_t nband, int64_t block);
int pwh_chebfi_iteration(pwh_ham* ham, int64_t nband, int64_t block, pwh_c128* psi, int64_t ld, pwh_c128* hpsi, int64_t ldh,
                         pwh_c128* spsi, int64_t lds, int degree, double b, double a0_margin, double* lambda, double* resid,
                         double* bounds_host, int32_t* info, void* ws, size_t ws_bytes, void* stream);

/*
 * ---------------------------------------------------------------------------------------------------------------
 * PAW-style generalised problem H Psi = Lambda S Psi ("S != I whenever the norm constraint is relaxed, as
 * in the Projector Augmented-Wave approach"; every benchmark of the paper uses PAW).
 *     V_nonloc = sum_{R,i,j} |p_i^R> D_ij^R <p_j^R|,     S = I + sum_{R,i,j} |p_i^R> Q_ij^R <p_j^R|
 * ---------------------------------------------------------------------------------------------------------------
 *
 * pwh_ham_set_paw -- replaces the diagonal D of the handle by per-atom dense Hermitian blocks D^R and adds the overlap
 * blocks Q^R.  The projector index is cut into `nblocks` consecutive blocks: offsets (HOST, nblocks + 1 int32, offsets[0] =
 * 0, offsets[nblocks] = nproj); dblocks / qblocks (DEVICE) hold the blocks one after the other, each n_R x n_R
 * column-major.  Both are copied.  The call also builds the nproj x nproj matrix K of S^-1 = I - P K P^H (Woodbury,
 * PAPER.md:225, 252) with two Cholesky factorisations (G = P^H P and I + U Q U^H) on the device, allocates scratch for it,
 * and synchronises the stream.  *info (DEVICE int32) = 0, or < 0 when one of the two matrices is not positive definite
 * (linearly dependent projectors, or an overlap S that is not positive definite).  Afterwards pwh_apply_h,
 * pwh_cheb_filter and the host entry points use the dense D^R; S enters through the calls below.
 */
int pwh_ham_set_paw(pwh_ham* ham, int64_t nblocks, const int32_t* offsets, const pwh_c128* dblocks, const pwh_c128* qblocks,
                    int32_t* info, void* stream);

/*
 * pwh_apply_hs -- HX_SX: hpsi = H psi and spsi = S psi from ONE set of projections C = P^H psi
 * (either output may be NULL).  Workspace as for pwh_apply_h; psi must not overlap the outputs.
 * pwh_apply_sinv -- Sinv: x <- S^-1 x = x - P K (P^H x), in place.
 * pwh_cheb_filter_gen -- the scaled Chebyshev filter of degree m of the operator S^-1 H, in place (Algorithm 12 lines 4-8,
 * per degree one H application, one Sinv and the three-term axpy of PAPER.md:246); same recurrence,
 * bounds and errors as pwh_cheb_filter.
 */
int pwh_apply_hs(pwh_ham* ham, int64_t nband, const pwh_c128* psi, int64_t ldpsi, pwh_c128* hpsi, int64_t ldh, pwh_c128* spsi,
                 int64_t lds, void* ws, size_t ws_bytes, void* stream);
int pwh_apply_sinv(pwh_ham* ham, int64_t nband, pwh_c128* x, int64_t ldx, void* ws, size_t ws_bytes, void* stream);
int pwh_cheb_filter_gen(pwh_ham* ham, int64_t nband, pwh_c128* psi, int64_t ld, int degree, double a, double b, double a0,
                        void* ws, size_t ws_bytes, void* stream);

/*
 * ---------------------------------------------------------------------------------------------------------------
 * LOBPCG -- the paper's other iterative eigensolver, on the same H application (Algorithm 6;
 * PAPER.md:506-574 Algorithm 11, here with S = I).  The paper's arithmetic-intensity argument (the filter
 * applies H k+1 times per data movement, LOBPCG once) is measured with it.
 * ---------------------------------------------------------------------------------------------------------------
 *
 * pwh_lobpcg -- Algorithm 11, in place on psi: the nband bands are cut into `nblocks` consecutive blocks of m = nband /
 * nblocks bands (nband % nblocks == 0, 3 m <= npw); per block: S-Deflate against the blocks already solved (Algorithm 8, line
 * 3), H Psi_i (line 6), S-Ortho (Algorithm 9, line 8), RR (Algorithm 10, line 9), then `nline` line minimisations (lines
 * 10-28): residual W = (H - Lambda) Psi_i and its norms (lines 11-12), W <- K W with the diagonal Teter-Payne-Allan
 * preconditioner K(G) = t / (t + 16 x^4), t = 27 + 18 x + 12 x^2 + 8 x^3, x = kin(G) / <T>_band (line 13; the paper names K
 * "diagonal matrix" only, PAPER.md:504 -- DESIGN.md reading R16), S-Deflate (line 15), H W (line 18), S-Ortho and RR of
 * [Psi_i, W_i] (first pass) or [Psi_i, W_i, P_i] (lines 20-25), whose lowest m Ritz pairs are the new Psi_i and whose part
 * outside span(Psi_i) is the new P_i (line 26).  With nblocks > 1 a final S-Ortho + RR over all bands (lines 31-34).
 *   tol       > 0: a block leaves the loop once all its residual norms are <= tol (line 12; costs one stream
 *             synchronisation per line minimisation -- the paper's mpi-sR sits there); 0: always nline passes, no host sync.
 *   lambda    [out] DEVICE nband Ritz values, ascending;  resid [out] DEVICE nband final residual norms (line 29);
 *   history   [out, optional] DEVICE nblocks x nline x m doubles: the residual norms seen at line 12 (untouched entries for
 *             passes skipped by the early exit);
 *   info      [out] DEVICE int32: > 0 = largest Jacobi sweep count of the dense eigen-solves, < 0 = a Cholesky factorisation met
 *             a non-positive pivot (linearly dependent search directions).
 * hpsi receives H psi.  Workspace: pwh_lobpcg_workspace_bytes(ham, nband, nblocks) (0 for invalid arguments), 256-byte aligned.
 * Errors: PWH_EINVAL for null pointers, bad sizes, ld < npw, workspace too small.
 */
size_t pwh_lobpcg_workspace_bytes(const pwh_ham* ham, int64_t nband, int64_t nblocks);
int pwh_lobpcg(pwh_ham* ham, int64_t nband, int64_t nblocks, int nline, double tol, pwh_c128* psi, int64_t ld, pwh_c128* hpsi,
               int64_t ldh, double* lambda, double* resid, double* history, int32_t* info, void* ws, size_t ws_bytes,
               void* stream);

/*
 * pwh_lobpcg_gen -- Algorithm 11 as printed, with the PAW overlap S of a handle that carries PAW blocks (pwh_ham_set_paw):
 * H X and S X come from one call of HX_SX (pwh_apply_hs, lines 6 and 18), every inner product is <., S .> (S-Deflate of
 * Algorithm 8 against the solved bands, S-Ortho of Algorithm 9, the generalised RR of Algorithm 10), the residual is
 * W = (H - Lambda S) Psi_i (line 11).  Same arguments and outputs as pwh_lobpcg plus spsi [out] = S psi (npw x nband, lds);
 * afterwards psi^H (S psi) = I.  Workspace: pwh_lobpcg_gen_workspace_bytes(ham, nband, nblocks).
 */
size_t pwh_lobpcg_gen_workspace_bytes(const pwh_ham* ham, int64_t nband, int64_t nblocks);
int pwh_lobpcg_gen(pwh_ham* ham, int64_t nband, int64_t nblocks, int nline, double tol, pwh_c128* psi, int64_t ld,
                   pwh_c128* hpsi, int64_t ldh, pwh_c128* spsi, int64_t lds, double* lambda, double* resid, double* history,
                   int32_t* info, void* ws, size_t ws_bytes, void* stream);

/*
 * ---------------------------------------------------------------------------------------------------------------
 * Electronic density (Algorithm 3 steps 9-10: "for every k-point: accumulate electronic density from f, Psi
 * for current k-point (FFT on GPU)").  It reuses the scatter and the inverse half of the local-potential
 * transforms.
 * ---------------------------------------------------------------------------------------------------------------
 *
 * pwh_density_accumulate -- rho(r) += weight * sum_i occ[i] |u_i(r)|^2 with u_i(r) = sum_G psi_i(G) exp(+2 pi i n_G.r/n), the
 * unnormalised inverse transform of the local-potential step (readings R6, R17: the paper prints no formula;
 * `weight` carries the caller's convention, e.g. w_k / Omega, with which sum_r rho(r) Omega / F = sum_k w_k sum_i occ_i for
 * orthonormal bands).
 *   psi   [in]     npw x nband, leading dimension ld;   occ [in] DEVICE nband doubles (occupations f_i);
 *   rho   [in/out] DEVICE double [n1*n2*n3], index i1 + n1*(i2 + n2*i3) like vloc; ACCUMULATED, so one array collects the
 *                  bands of several calls and the k-points of several handles (zero it first).
 *   ws / ws_bytes  at least pwh_density_workspace_bytes(ham, nband), 256-byte aligned.
 * The sum over the bands of one call is formed in band order by one owner thread per grid point: the result is
 * deterministic.  Errors: PWH_EINVAL (null pointer, ld < npw, workspace too small or misaligned), PWH_ECUDA.
 */
size_t pwh_density_workspace_bytes(const pwh_ham* ham, int64_t nband_max);
int pwh_density_accumulate(pwh_ham* ham, int64_t nband, const pwh_c128* psi, int64_t ld, const double* occ, double weight,
                           double* rho, void* ws, size_t ws_bytes, void* stream);

/* Number of kernel launches issued by this library since load (all handles, all threads). */
int64_t pwh_launch_count(void);

/*
 * Per-kernel timing for the roofline report.  Between pwh_profile_begin() and
 * pwh_profile_end() every kernel launch of the library is bracketed by a cudaEvent pair on its stream.
 * pwh_profile_end synchronises the device and returns, per stage, the summed kernel time in milliseconds and the
 * number of launches (HOST arrays of PWH_NSTAGES entries).  Not thread-safe against concurrent compute calls.
 */
enum {
  PWH_STAGE_SCATTER_ZINV = 0, /* a1-a2: sphere -> z-columns, inverse z transform */
  PWH_STAGE_PLANE = 1,        /* a3-a5: per-plane inverse y,x, V_loc multiply, forward x,y */
  PWH_STAGE_ZFWD_GATHER = 2,  /* a6 + a9: forward z transform, gather, kinetic + recurrence epilogue */
  PWH_STAGE_ZGEMM_CN = 3,     /* a7, a10: A^H B DMMA ZGEMM partial products (projector coefficients, Gram) */
  PWH_STAGE_SPLITK = 4,       /* a7, a10: fixed-order split-K sum (+ D scaling) */
  PWH_STAGE_ZGEMM_NN = 5,     /* a8: P (D C) accumulated onto the recurrence term; rotations Psi X */
  PWH_STAGE_COLSTATS = 6,     /* Rayleigh quotients, residual norms (column reductions over the plane waves) */
  PWH_STAGE_DENSE_SMALL = 7,  /* M x M steps: Cholesky panels, triangular inverse, shifts, sorts */
  PWH_STAGE_JACOBI = 8,       /* M x M Hermitian eigen-solve (one cooperative launch) */
  PWH_STAGE_AXPY = 9,         /* three-term axpy of the filter on S^-1 H (generalised problem) */
  PWH_NSTAGES = 12
};
int pwh_profile_begin(void);
int pwh_profile_end(double ms[PWH_NSTAGES], int64_t launches[PWH_NSTAGES]);

/*
 * Attainable FP64 tensor-pipe (DMMA) rate of the current device at its current clocks, in TFLOP/s: a
 * register-resident loop of `iters` x 32 independent mma.m8n8k4.f64 per warp on 2 CTAs per SM, timed with CUDA
 * events (one warm-up launch).  It is the measured denominator for the ZGEMM roofline fraction; it touches no
 * memory and is not part of the path.  tflops is a HOST pointer.  Synchronises `stream`.
 */
int pwh_probe_fp64_tensor_peak(int iters, double* tflops, void* stream);

/* Introspection: fills info[0..7] = {npw, nproj, n1, n2, n3, n_zcolumns, n_xlines, reserved}. */
int pwh_ham_info(const pwh_ham* ham, int64_t info[8]);

/* Introspection: writes a NUL-terminated, space-separated list of the kernel families this handle launches (e.g.
 * "kz_scatter_zinv kv2_plane kz_zfwd_gather zgemm3m_tma") into buf (HOST, at most n bytes, truncated). */
int pwh_ham_kernels(const pwh_ham* ham, char* buf, size_t n);

/* Thread-local message describing the last error returned on this thread ("" if none). */
const char* pwh_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PWHAM_H */
