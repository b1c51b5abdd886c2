/* bs.h — C-ABI boundary of the B200-native phononic band-structure hot path.
 *
 * Method: mixed-variational plane-wave formulation of arXiv:1310.6380 ("PAPER.md" below), 2-D plane strain
 * (eq. 13-14), plane waves alpha,beta in [-Mt,Mt] (eq. 15), matrices Phi, Psi(=paper's
 * Omega), H of PAPER.md:140-173 (eq. 17-20), eigenproblem PAPER.md:94-104 (eq. 10-11) solved as the Hermitian pencil
 * K(k) U = lambda Psi U, K(k) = H(k)^dagger Phi^{-1} H(k), lambda = omega^2.  Readings of ambiguous passages: DESIGN.md
 * section 3.
 *
 * Conventions common to every call
 *   - All matrices are column-major complex128 stored as interleaved (re,im) doubles, leading dimension = order.
 *   - N = (2Mt+1)^2 plane waves; plane wave g <-> (a1,a2), g = (a1+Mt)(2Mt+1) + (a2+Mt)  (PAPER.md:150, 0-based).
 *   - Entry (row alpha = test function, column beta = trial function) uses q = G_beta - G_alpha.
 *   - "host" / "device" is stated per pointer.  Inputs are copied at bs_create_cell (the caller keeps its arrays).
 *   - Every call returns a bs_status; bs_last_error() gives a thread-local message for the last failure.
 *   - A handle is not thread-safe; distinct handles are independent.  `stream` is a cudaStream_t passed as void*
 *     (NULL = the legacy default stream).  All kernels of a call are launched on that stream.
 *   - There is NO CPU fallback: without a CUDA device every compute call returns BS_ERR_CUDA.
 */
#ifndef BS_H_
#define BS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bs_cell bs_cell; /* opaque; owns small device buffers (geometry), borrows the big workspace */

typedef enum {
  BS_OK = 0,
  BS_ERR_ARG = -1,      /* null pointer, negative size, nbands > 2N, ... */
  BS_ERR_GEOMETRY = -2, /* polygon with non-positive signed area, or sum of areas != |det lattice| (1e-10 relative) */
  BS_ERR_NOT_PD = -3,   /* a Cholesky pivot of Phi or of R (Psi = diag(R,R)) was not positive */
  BS_ERR_STATE = -4,    /* call order violated (e.g. bs_bands before bs_assemble) */
  BS_ERR_CUDA = -5,     /* CUDA runtime error, or no device */
  BS_ERR_NOMEM = -6     /* workspace missing or too small */
} bs_status;

/* Options for bs_set_option. */
typedef enum {
  BS_OPT_PENCIL_MODE = 0, /* 0 = BS_PENCIL_POLY (default), 1 = BS_PENCIL_DIRECT; see bs_bands */
  BS_OPT_PANEL = 1,       /* two-stage: band width b in {8, 16, 32}; one-stage: panel width 4..32, multiple of 4.
                             0 (default) = automatic: 16 (measured best at every size with the register-tile chasing
                             kernel of stage 2) */
  BS_OPT_TIMING = 2       /* 1 = CUDA events around the stages (bs_get_timings); 2 = also around every kernel launch,
                             summed per kernel class (bs_get_kernel_timings).  Both add a final stream synchronise. */
} bs_option;
enum { BS_PENCIL_POLY = 0, BS_PENCIL_DIRECT = 1 };
/* BS_OPT_TRIDIAG (option 3): algorithm of S6.  0 = two-stage (dense -> band by DMMA GEMMs, band -> tridiagonal by bulge
 * chasing; default; matrices with n <= 112 are tridiagonalised inside shared memory by one CTA instead),
 * 1 = one-stage blocked Householder (matrix-vector bound; kept as a cross-check),
 * 2 = two-stage with the band of stage 2 always streamed through the shared-memory ring (the configuration large matrices
 * get anyway), also where the whole band would fit.  A tuning / test variant: the same algorithm as 0 and the SAME BITS
 * (the chasing step is compiled without multiply-add contraction, so its two inlined copies round identically; the
 * result does not depend on how many sweeps overlap either: tests/test_gpu_blocks.py). */
enum { BS_OPT_TRIDIAG = 3 };
enum { BS_TRIDIAG_TWO_STAGE = 0, BS_TRIDIAG_ONE_STAGE = 1, BS_TRIDIAG_TWO_STAGE_STREAMED = 2 };
/* BS_OPT_ASSEMBLY (option 4): quadrature of the shape integrals in S1.  0 = exact closed-form polygon integral (default),
 * 1 = the paper's centroid rule I_p(q) ~ A_p exp(i q.c_p) (PAPER.md:106 eq. 12, :213 eq. 22; c_p = area centroid), kept as the
 * paper-faithful variant: its matrices converge to the exact ones as the mesh is refined. */
enum { BS_OPT_ASSEMBLY = 4 };
enum { BS_ASSEMBLY_EXACT = 0, BS_ASSEMBLY_CENTROID = 1 };
/* BS_OPT_PHI_INVERSE (option 5): 0 = automatic (default): when every phase is isotropic plane strain, Phi has the block
 * structure [[A, B, 0], [B, A, 0], [0, 0, 2(A-B)]] and Phi^{-1} is composed from the two N x N inverses
 * (A+B)^{-1} and (A-B)^{-1}; 1 = always factor and invert the full 3N x 3N matrix (any compliance; cross-check). */
enum { BS_OPT_PHI_INVERSE = 5 };
/* BS_OPT_OUTPUT (option 6), step S8: what bs_bands / bs_bands_batch write.  0 = lambda = omega^2 (default; may be slightly
 * negative at k = 0 where the exact value is 0), 1 = omega = sqrt(max(lambda, 0)) (omega_N = sqrt(lambda_N)).
 * In a batch the lead handle (cells[0]) decides. */
enum { BS_OPT_OUTPUT = 6 };
enum { BS_OUTPUT_OMEGA2 = 0, BS_OUTPUT_OMEGA = 1 };

/* Stage indices of bs_get_timings (milliseconds, CUDA events on the call's stream). */
enum {
  BS_T_TABLE = 0,   /* S1 shape-integral table               */
  BS_T_EXPAND = 1,  /* S2 expansion to Phi, R                */
  BS_T_FACTOR = 2,  /* S3 Cholesky(Phi), Phi^{-1}, Cholesky(R), L_R^{-1} */
  BS_T_COEF = 3,    /* S4+S5 on the six k-polynomial coefficient matrices (POLY mode, inside bs_assemble) */
  BS_T_PENCIL = 4,  /* S4(+S5 in DIRECT mode): per-k formation of A(k)   */
  BS_T_TRIDIAG = 5, /* S6 Householder tridiagonalisation     */
  BS_T_BISECT = 6,  /* S7 Sturm bisection                    */
  BS_T_COUNT = 8
};

/* PAPER.md:121 (eq. 14): isotropic plane-strain compliance D_jkmn from Young's modulus E and Poisson ratio nu.
 * E, nu: host, n doubles each.  compliance_out: host, n x 6 doubles, row = [D1111 D2222 D1122 D1112 D2212 D1212]
 * (the component order of PAPER.md:167-171, eq. 20).  Pure host arithmetic.  BS_ERR_ARG on null / n<0 / E<=0 / nu>=0.5. */
bs_status bs_isotropic_plane_strain(int32_t n, const double *E, const double *nu, double *compliance_out);

/* PAPER.md:21-37 (section II: lattice vectors h^1,h^2, phases with their own compliance D and density rho).
 *   lattice     host, 4 doubles [h1x h1y h2x h2y]: rows of [A]_{jk} = h^j . e^k.
 *   nphase      number of phases P >= 1; each phase is one simple polygon.
 *   vert_offset host, P+1 int32, CSR offsets into verts (vert_offset[0] = 0, >= 3 vertices per polygon).
 *   verts       host, 2*vert_offset[P] doubles, Cartesian (x,y) pairs, counter-clockwise.  Polygons may stick out of
 *               the cell (lattice-translated pieces); together they must tile the cell area exactly.
 *   compliance  host, P x 6 doubles [D1111 D2222 D1122 D1112 D2212 D1212] per phase (eq. 20).
 *   density     host, P doubles, > 0.
 *   out         receives the handle (free with bs_destroy_cell).
 * Does S0 (reciprocal basis eq. 1, fractional coordinates, per-edge arrays) on the host and copies them to the device.
 * Errors: BS_ERR_ARG, BS_ERR_GEOMETRY, BS_ERR_CUDA. */
bs_status bs_create_cell(const double lattice[4], int32_t nphase, const int32_t *vert_offset, const double *verts,
                         const double *compliance, const double *density, bs_cell **out);

/* Optimisation-loop shape: ncells cells that share ONE geometry (lattice
 * and polygons) and differ in their material properties only.
 *   compliance  host, ncells x P x 6 doubles;  density  host, ncells x P doubles;  out  receives ncells handles.
 * The handles behave like those of bs_create_cell (each is destroyed with bs_destroy_cell; the shared geometry is freed
 * with the last of them).  When ALL cells of a bs_assemble / bs_assemble_batch call share one geometry, step S1 evaluates
 * the polygon integrals I_p(q_D) ONCE into a (P x index-difference) table that stays with the geometry, and every cell's
 * table is the small product T = W I of its weights with it (one batched DMMA GEMM) instead of re-integrating every
 * polygon per cell.  Errors: as bs_create_cell. */
bs_status bs_create_cells_shared(const double lattice[4], int32_t nphase, const int32_t *vert_offset, const double *verts,
                                 int32_t ncells, const double *compliance, const double *density, bs_cell **out);

/* New material properties for an existing handle (same geometry): compliance host P x 6, density host P.  The next
 * bs_assemble uses them; with a shared geometry the polygon integrals are not evaluated again.  The copy is ordered after
 * the work already enqueued on the handle's stream.  Errors: BS_ERR_ARG. */
bs_status bs_set_properties(bs_cell *cell, const double *compliance, const double *density);

/* Waits for the stream of the handle's last call (NOT for the whole device: other streams of the caller keep
 * running), then releases the handle.  Its small device blocks go back to a
 * process-wide cache (at most 256 MiB) that later bs_create_cell calls draw from, so create/destroy loops do not pay
 * cudaMalloc / cudaFree.  NULL is accepted. */
void bs_destroy_cell(bs_cell *cell);

bs_status bs_set_option(bs_cell *cell, int32_t option, int32_t value);

/* Device workspace the handle needs for truncation Mt and up to nk k-points per bs_bands call (depends on the
 * options set so far).  The caller allocates it (e.g. a torch uint8 tensor), 256-byte aligned, and lends it with
 * bs_set_workspace; it must stay alive and untouched until bs_destroy_cell or the next bs_set_workspace. */
bs_status bs_workspace_bytes(const bs_cell *cell, int32_t truncation, int32_t nk, size_t *bytes);
bs_status bs_set_workspace(bs_cell *cell, void *dev_ptr, size_t bytes);

/* S1+S2+S3 (+ the k-independent part of S4/S5 in POLY mode), PAPER.md:140-173:
 *   S1  T_c(D) = sum_p w_{c,p} I_p(D1 q^1 + D2 q^2) for every index difference D in [-2Mt,2Mt]^2, with the closed-form
 *       polygon integral I_p(q) = int_{Omega_p} exp(i q.x) dx (exact version of the centroid rule eq. 12/22);
 *   S2  Phi (3N x 3N, eq. 20 with its factors 1/2/4) and R (N x N, eq. 19; Psi = diag(R,R));
 *   S3  Phi = L L^dagger, Y = Phi^{-1} explicitly, R = L_R L_R^dagger, L_R^{-1}.
 * Asynchronous on `stream` except for one final synchronise that reads the Cholesky status.
 * Errors: BS_ERR_ARG (Mt < 0 or 2N > 2048), BS_ERR_NOMEM, BS_ERR_NOT_PD, BS_ERR_CUDA. */
bs_status bs_assemble(bs_cell *cell, int32_t truncation, void *stream);

/* The same for ncells handles in one set of launches (config 4: optimisation-loop batch).  All cells must have a
 * workspace set for the same truncation, the same options, live on the same device and have the SAME CELL AREA
 * |det lattice| (one V^2 scales K(k) of every cell of a launch); anything else is BS_ERR_ARG before any launch. */
bs_status bs_assemble_batch(bs_cell *const *cells, int32_t ncells, int32_t truncation, void *stream);

/* Parity access after bs_assemble: copies Phi (3N x 3N) and Psi (2N x 2N) to HOST buffers (either may be NULL). */
bs_status bs_get_matrices(bs_cell *cell, void *phi_host, void *psi_host);
/* Parity access: the table T_c(D), host, 7 x (4Mt+1) x (4Mt+1) complex128, index [c][D1+2Mt][D2+2Mt];
 * channels c = Dv11 Dv22 Dv12 Dv13 Dv23 Dv33 (Voigt weights of eq. 20) then rho. */
bs_status bs_get_table(bs_cell *cell, void *table_host);
/* Parity access: K(k) = H^dagger Phi^{-1} H (2N x 2N, HOST out) at one reduced k-point (S4 only). */
bs_status bs_get_pencil(bs_cell *cell, const double kred[2], void *K_host, void *stream);

/* S4..S8 for nk k-points:
 *   kpts        HOST, nk x 2 doubles, reduced coordinates (Q1,Q2), k = Q1 q^1 + Q2 q^2.
 *   nbands      1 <= nbands <= 2N.
 *   omega2_out  nk x nbands doubles, row-major, ascending lambda = omega^2 per k; HOST or DEVICE pointer
 *               (detected); a host pointer implies a final stream synchronise.
 * All k-points are in flight on the device at once; there is no host round-trip between k-points.
 * POLY mode: A(k) = L_Psi^{-1} K(k) L_Psi^{-dagger} is evaluated as the quadratic polynomial in (kx,ky) whose six
 * coefficient matrices bs_assemble prepared; DIRECT mode forms K(k) by the scaling kernel and reduces it per k.
 * Errors: BS_ERR_STATE, BS_ERR_ARG, BS_ERR_NOMEM (nk larger than the workspace was sized for), BS_ERR_CUDA. */
bs_status bs_bands(bs_cell *cell, int32_t nk, const double *kpts, int32_t nbands, double *omega2_out, void *stream);

/* The same k-points for ncells assembled cells in one set of launches.  omega2_out: ncells x nk x nbands.
 * Limits (BS_ERR_ARG): ncells * nk <= 65535 eigenproblems per call (split larger batches over several calls);
 * 2N <= 2048; equal cell areas, options and device across the batch (see bs_assemble_batch). */
bs_status bs_bands_batch(bs_cell *const *cells, int32_t ncells, int32_t nk, const double *kpts, int32_t nbands,
                         double *omega2_out, void *stream);

/* BS_OPT_MODES (option 7): the largest number of mode shapes per k-point bs_modes may be asked for (0 = off, default).
 * Set it BEFORE bs_workspace_bytes / bs_assemble: the workspace then also holds the reflectors of the band reduction, a
 * copy of the band and the vectors (about 2N x 2N complex more per k-point). */
enum { BS_OPT_MODES = 7 };

/* BS_OPT_REFINE (option 8; 0 = off, default; 1): bs_modes returns in omega2_out, instead of the eigenvalues of the assembled
 * pencil, the Rayleigh quotients of its modes in factored form, omega^2_j = (H u_j)^dagger Phi^-1 (H u_j) / (u_j^dagger Psi u_j).
 * The eigenvalues of K(k) = H^dagger Phi^-1 H carry an absolute error of ~eps lambda_max, which destroys the relative
 * accuracy of the acoustic branches next to Gamma (omega^2 / lambda_max ~ 1e-10 at |k| = 1e-4 of the zone: omega wrong in
 * the 7th digit); the factored quotient is accurate to ~eps kappa(Phi) relative (the accuracy of the singular-value route
 * omega = sigma(L_Phi^-1 H L_Psi^-dagger), SURVEY 8(c)-7 / DESIGN.md R8, without forming an SVD) as long as
 * omega^2 / lambda_max >~ 1e-12.  bs_bands is not affected. */
enum { BS_OPT_REFINE = 8 };

/* Mode shapes of the lowest nbands branches ("the eigenvectors U give the displacement mode shapes and
 * S = -Phi^-1 H* U the stress mode shapes").  One handle, nk k-points.
 *   omega2_out  nk x nbands doubles as bs_bands (host or device).
 *   U_out       nk blocks of 2N x nbands complex128, column-major (column j = displacement coefficients (u1 | u2) of band j
 *               on the N plane waves, Psi-orthonormal: U^dagger Psi U = I); host or device; may be NULL.
 *   S_out       nk blocks of 3N x nbands: stress coefficients (s11 | s22 | s12), S = Phi^-1 H U with H = V B(k) (the paper's
 *               H* is -H, R3), so that Phi S = H U and H^dagger S = lambda Psi U (eq. 10); may be NULL.
 * Phases and, inside a degenerate eigenvalue, the basis are arbitrary.  Method: the eigenvalues as bs_bands; eigenvectors of
 * the Hermitian band matrix of S6 stage 1 by inverse iteration (pivoted band LU, modified Gram-Schmidt inside clusters);
 * back-transformation through the block reflectors of stage 1 and L_Psi^-H.  Synchronises the stream.
 * Errors: BS_ERR_STATE (BS_OPT_MODES not set, or omega output selected), BS_ERR_ARG (nbands > BS_OPT_MODES), as bs_bands. */
bs_status bs_modes(bs_cell *cell, int32_t nk, const double *kpts, int32_t nbands, double *omega2_out, void *U_out,
                   void *S_out, void *stream);
/* The same for a batch of handles (as bs_bands_batch: equal options, truncation and cell area; ncells * nk <= 65535): omega2_out
 * ncells x nk x nbands; U_out ncells x nk blocks of 2N x nbands; S_out ncells x nk blocks of 3N x nbands, cell-major.  Every
 * matrix is treated exactly as in the single-handle call (bitwise equal results). */
bs_status bs_modes_batch(bs_cell *const *cells, int32_t ncells, int32_t nk, const double *kpts, int32_t nbands,
                         double *omega2_out, void *U_out, void *S_out, void *stream);

/* Parity access after bs_bands: the tridiagonal T(k) of the last call, HOST out: d (nk x 2N), e (nk x 2N, last unused). */
bs_status bs_get_tridiagonal(bs_cell *cell, double *d_host, double *e_host);

/* Stage timings of the last bs_assemble / bs_bands on this handle (BS_OPT_TIMING=1), HOST out, BS_T_COUNT doubles (ms).
 * For a batch call the timings are recorded on cells[0]. */
bs_status bs_get_timings(bs_cell *cell, double *ms_out);

/* Kernel classes of bs_get_kernel_timings. */
enum {
  BS_KC_TABLE = 0,        /* S1 table kernel (FP64 ALU)                         work: real flops                     */
  BS_KC_EXPAND = 1,       /* S2 expansion                                       work: bytes written                  */
  BS_KC_GEMM_FACTOR = 2,  /* DMMA zgemm launches of S3                          work: real flops                     */
  BS_KC_GEMM_REDUCE = 3,  /* DMMA zgemm launches of S5 (and of the POLY coefficient reduction)                       */
  BS_KC_GEMM_TRIDIAG = 4, /* DMMA zgemm launches of S6: Hermitian rank-2b updates  work: real flops                  */
  BS_KC_HEMV = 5,         /* S6 Hermitian matrix-vector kernel                  work: bytes of the lower triangle    */
  BS_KC_PANEL = 6,        /* S6 panel / reflector kernels                                                            */
  BS_KC_STURM = 7,        /* S7                                                                                      */
  BS_KC_PENCIL = 8,       /* S4 scaling kernel                                  work: bytes moved                    */
  BS_KC_COMBINE = 9,      /* S4 polynomial combination (POLY mode)              work: bytes moved                    */
  BS_KC_POTRF_DIAG = 10,  /* S3 diagonal-block factor kernel                                                         */
  BS_KC_OTHER = 11,
  BS_KC_BULGE = 12,       /* S6 stage 2: band -> tridiagonal bulge chasing                                           */
  BS_KC_GEMM_HEMM = 13,   /* S6 stage 1: Z = A22 V (Hermitian A22, lower triangle read), DMMA             work: real flops */
  BS_KC_GEMM_WY = 14,     /* S6 stage 1: the two small compact-WY GEMMs per panel, DMMA                    work: real flops */
  BS_KC_TRIDIAG_SMALL = 15, /* S6 for n <= 112: whole matrix in shared memory, unblocked Householder    work: real flops */
  BS_KC_COUNT = 16
};
/* Per-class totals of the last bs_assemble / bs_bands led by this handle under BS_OPT_TIMING = 2: device milliseconds
 * (CUDA events on the call's stream around every launch), ALGORITHMIC work credited at launch time (flops or bytes, see
 * the enum) and number of launches.  HOST out, BS_KC_COUNT entries each.  BS_ERR_STATE if timing mode 2 was never set. */
bs_status bs_get_kernel_timings(bs_cell *cell, double *ms_out, double *work_out, int64_t *count_out);

/* Number of kernel launches issued by the library on behalf of this handle since creation (batch: on cells[0]). */
int64_t bs_launch_count(const bs_cell *cell);

const char *bs_last_error(void); /* thread-local, valid until the next call on this thread */

/* ---- diagnostics: the dense building blocks, exposed so that tests can check them in isolation ------------------- */
/* C = alpha op(A) op(B) + beta C on DEVICE column-major complex128 arrays; op: 0 = none, 1 = conjugate transpose.
 * flags: see DESIGN.md section 5 (BS_GEMM_*).  batch >= 1 matrices with the given element strides.  The complex
 * product is the three-multiplication form (norm-wise error bound, not component-wise).  C must not overlap A or B,
 * except C == A with opA = 0, opB = 1, N <= 64, flags = 0 (in-place right multiplication by a small block). */
bs_status bs_zgemm(int32_t opA, int32_t opB, int32_t M, int32_t N, int32_t K, const double alpha[2], const void *A,
                   int32_t lda, int64_t strideA, const void *B, int32_t ldb, int64_t strideB, const double beta[2],
                   void *C, int32_t ldc, int64_t strideC, int32_t batch, int32_t flags, void *stream);
/* In-place lower Cholesky of `batch` n x n DEVICE matrices (stride in elements) and X = L^{-1} (lower, zeros above);
 * tmp: DEVICE scratch of batch*strideA elements; dinv: DEVICE scratch, batch*ceil(n/64)*64*64 elements;
 * info: DEVICE int32[batch] (0 = ok, else 1-based failing pivot). */
bs_status bs_zpotrf_trtri(int32_t n, void *A, int32_t lda, int64_t strideA, void *X, void *tmp, void *dinv,
                          int32_t *info, int32_t batch, void *stream);
/* Householder tridiagonalisation of `batch` n x n Hermitian DEVICE matrices (lower triangle read; trailing blocks are
 * overwritten), n <= 2048, Q^H A Q = T real symmetric tridiagonal (eigenvalues of the pencil).
 * d, e: DEVICE, batch x n doubles (e[.][n-1] unused).  scratch: DEVICE, batch * bs_zhetrd_scratch_elems(n, nb) complex128
 * elements.  nb: panel width (clamped to 4..32).  Synchronises the stream before returning. */
size_t bs_zhetrd_scratch_elems(int32_t n, int32_t nb);
bs_status bs_zhetrd(int32_t n, void *A, int32_t lda, int64_t strideA, double *d, double *e, void *scratch, int32_t nb,
                    int32_t algo /* BS_TRIDIAG_* ; two-stage: nb is the band width, rounded to 8/16/32 */,
                    int32_t batch, void *stream);
/* bs_zhetrd without any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, serving
 * loops, harnesses that forbid it): the same two-stage reduction (band width 16; n <= 112: the shared-memory kernel),
 * Q^H A Q = T (the eigenvalues of the pencil), with ALL of its scratch (reflector blocks, band
 * storage, progress words of the bulge chase) in one file-scope static device array of BS_ZHETRD_STATIC_BYTES that
 * every GPU which loads the library holds until the process exits.  The call issues no cudaMalloc / cudaFree and calls
 * no allocating library routine; it does not synchronise: d and e are valid once `stream` has reached the end of the
 * work enqueued here.  A, d, e: DEVICE, as for bs_zhetrd (A: batch matrices, strideA elements apart, lower triangle
 * read, overwritten; d, e: batch x n doubles).  The device of `stream` must be the current device.
 * Limit: bs_zhetrd_static_bytes(n, batch) <= BS_ZHETRD_STATIC_BYTES (one matrix up to n = 2048, six of n = 450, ten of
 * n = 242), otherwise BS_ERR_ARG with the two numbers in bs_last_error(); n > 2048 is BS_ERR_ARG as for bs_zhetrd.
 * ALL calls on a device share the array, whatever the stream or host thread: calls whose GPU work overlaps race on it
 * (order them on one stream, or with events).  The array keeps the previous call's contents; the call clears what
 * must start at zero (the progress words) on `stream` itself. */
#define BS_ZHETRD_STATIC_BYTES (8 * 1024 * 1024)
size_t bs_zhetrd_static_bytes(int32_t n, int32_t batch);
bs_status bs_zhetrd_static(int32_t n, void *A, int32_t lda, int64_t strideA, double *d, double *e, int32_t batch,
                           void *stream);
/* Lowest nev eigenvalues of `batch` real symmetric tridiagonal matrices (d, e: DEVICE, batch x n) by Sturm bisection;
 * lam: DEVICE, batch x nev, ascending. */
bs_status bs_sturm(int32_t n, const double *d, const double *e, int32_t nev, double *lam, int32_t batch, void *stream);

/* FP64 roofline denominators of the current device, measured with register-only loops on `stream` (about 30 ms):
 * DMMA (mma.sync m8n8k4 f64, the FP64 tensor pipe) and DFMA TFLOP/s.  HOST out.  Synchronises. */
bs_status bs_fp64_peak(double *dmma_tflops, double *dfma_tflops, void *stream);

enum {
  BS_GEMM_LOWER_ONLY = 1, /* compute only tiles that intersect the lower triangle of C */
  BS_GEMM_KLO_ROW = 2,    /* op(A)[m][k] = 0 for k < m   (start the k loop at the tile's first row)   */
  BS_GEMM_KHI_ROW = 4,    /* op(A)[m][k] = 0 for k > m   (stop the k loop after the tile's last row)  */
  BS_GEMM_KLO_COL = 8,    /* op(B)[k][n] = 0 for k < n */
  BS_GEMM_KHI_COL = 16,   /* op(B)[k][n] = 0 for k > n */
  BS_GEMM_A_HERM_LOWER = 32 /* A is M x M Hermitian, only its lower triangle is read (opA = opB = 0, K = M): HEMM */
};

#ifdef __cplusplus
}
#endif
#endif /* BS_H_ */
