/*
 * sparc_gpu.h -- C-ABI boundary of the B200-native CheFSI hot path (arxiv 2302.09708).
 *
 * What the library computes (citations are /root/reference/PAPER.md line numbers; "R<n>" are the
 * readings listed in DESIGN.md section 3):
 *
 *   H = -1/2 Laplacian + Veff + V_nl, applied matrix-free to a block of N_s FP64 orbitals on a uniform
 *   3-D grid of N_d = nx*ny*nz nodes (Algorithm 1, 102, 122).  The Laplacian is the
 *   central finite-difference stencil of order n0 (3*n0+1 taps), periodic or Dirichlet
 *   per axis; Veff multiplies pointwise; V_nl = sum_J S_J^T chi_J
 *   diag(gamma_J) chi_J^T S_J applies each atom's dense projector matrix to "the appropriate
 *   components" of the orbitals.  On top of H:
 *     - the Chebyshev filter  X <- p_m((H - cI)/e) X
 *     - the projection        Hs = X^T H X,  Ms = X^T X
 *     - the rotation          X <- X Q   (Q = eigenvectors supplied by the caller, or computed on the device by
 *                             sparc_gpu_eigensolve)
 *   and: the gradient stencil / projector contraction / nonlocal force, the subspace
 *   eigensolve, the complex k-point variants (*_k) and the local pieces of the multi-GPU row partition.
 *
 * Conventions
 *   - FP64 throughout; real orbitals (Gamma point) except in the *_k entry points (complex, interleaved
 *     re/im).  Grid linear index i = x + nx*(y + ny*z).
 *   - Psi, X, Y: N_d x ncols, column-major, leading dimension ld >= N_d; one column = one orbital.
 *     Hs, Ms, Q: ns x ns, column-major, ld = ns.
 *   - Pointers named *_dev are DEVICE pointers owned by the caller (e.g. PyTorch tensors); pointers in
 *     sparc_gpu_desc are HOST pointers, copied at create (the caller may free them afterwards).
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Every operator call
 *     (set_veff, hamiltonian_apply, chebyshev_filter, project, rotate, and the "next" operators below) is
 *     asynchronous on `stream`, never synchronises the device and never touches host memory.  The
 *     exceptions are support calls and say so: create / destroy (blocking uploads), sparc_gpu_probe_peak
 *     (synchronises `stream`), sparc_gpu_get_info with a "prof_ns:<k>" key (waits for the recorded events)
 *     and the *_host entry points (host buffers; they synchronise before returning).
 *   - Every call makes ctx's device current for its duration and restores the caller's current device.
 *   - `ws_dev` is caller-owned device scratch of at least sparc_gpu_workspace_bytes(...) bytes, 256-byte
 *     aligned.  The ABI carries no size with the pointer: declare it once with
 *     sparc_gpu_set_workspace_size and every operator call that needs more returns WORKSPACE_TOO_SMALL
 *     instead of overrunning the buffer.  The library allocates only its immutable tables (weights, chi,
 *     index maps, Veff copy).
 *   - Every call returns 0 on success or a negative sparc_gpu_status.  No exceptions, no exit(), no
 *     printing.  There is NO CPU fallback: without an sm_100 device create fails with UNSUPPORTED.
 */
#ifndef SPARC_GPU_H
#define SPARC_GPU_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sparc_gpu_ctx sparc_gpu_ctx;   /* opaque, owned by the library */

typedef enum {
    SPARC_GPU_SUCCESS = 0,
    SPARC_GPU_INVALID_ARG = -1,         /* NULL pointer, negative size, ld < N_d, degree < 0, bad op ...  */
    SPARC_GPU_UNSUPPORTED = -2,         /* fd_order not even in 2..12; periodic axis with n < n0+1 (R10);
                                           device is not compute capability 10.x                            */
    SPARC_GPU_BAD_BOUNDS = -3,          /* filter bounds must satisfy a0 < a < b (R5)                       */
    SPARC_GPU_BAD_DESCRIPTOR = -4,      /* support index out of range / not strictly ascending within an
                                           atom, inconsistent chi_ptr / supp_ptr, n_proj < 0 or > 16        */
    SPARC_GPU_WORKSPACE_TOO_SMALL = -5, /* the call needs more scratch than sparc_gpu_set_workspace_size declared */
    SPARC_GPU_OUT_OF_MEMORY = -6,       /* device allocation of the library's tables failed                 */
    SPARC_GPU_CUDA_ERROR = -7,          /* any other CUDA runtime / driver error                            */
    SPARC_GPU_STATIC_SCRATCH_EXCEEDED = -8  /* sparc_gpu_gram_static: m * n is more than the built-in scratch holds */
} sparc_gpu_status;

typedef enum {
    SPARC_GPU_OP_HAMILTONIAN_APPLY = 0,
    SPARC_GPU_OP_CHEBYSHEV_FILTER = 1,
    SPARC_GPU_OP_PROJECT = 2,
    SPARC_GPU_OP_ROTATE = 3,
    SPARC_GPU_OP_GRADIENT_PROJECT = 4,
    SPARC_GPU_OP_NONLOCAL_FORCE = 5,
    SPARC_GPU_OP_EIGENSOLVE = 6,
    SPARC_GPU_OP_HAMILTONIAN_APPLY_K = 7,
    SPARC_GPU_OP_CHEBYSHEV_FILTER_K = 8,
    SPARC_GPU_OP_PROJECT_K = 9,
    SPARC_GPU_OP_ROTATE_K = 10,
    SPARC_GPU_OP_GRAM = 11
} sparc_gpu_op;

/* Problem description (all pointers HOST, copied at create).  PAPER.md:118 "The matrix X, effective
 * potential, and nonlocal projectors are then transferred from the host CPU to its mapped GPU". */
typedef struct {
    int32_t n[3];             /* nx, ny, nz                                                         */
    double h[3];              /* grid spacing per axis, bohr (R17)                                  */
    int32_t bc[3];            /* 0 = periodic, 1 = Dirichlet: psi = 0 outside [0, n-1] (R9)         */
    int32_t fd_order;         /* n0: even, 2..12; stencil radius n0/2 (R1)            */
    int32_t n_atoms;          /* may be 0 (no nonlocal term)                                        */
    const int64_t *supp_ptr;  /* [n_atoms+1] offsets into supp_idx                                  */
    const int32_t *supp_idx;  /* grid linear indices, strictly ascending within an atom (R8)        */
    const int32_t *n_proj;    /* [n_atoms] number of projectors P_J of atom J (0..16)               */
    const int64_t *chi_ptr;   /* [n_atoms+1] offsets (in doubles) into chi; atom J owns n_J*P_J     */
    const double *chi;        /* per atom: n_J x P_J, column-major ("dense matrix")    */
    const double *gamma;      /* concatenated P_J Kleinman-Bylander energies per atom (R6, R7)      */
    const double *veff;       /* [N_d] or NULL (then set later with sparc_gpu_set_veff; zero until) */
    int32_t device;           /* CUDA device ordinal                                                */
} sparc_gpu_desc;

/* Create a context on desc->device: validates the descriptor, uploads it, builds the stencil
 * coefficient tables and the point -> (atom, row) inverse map used by the nonlocal pull kernel. */
int sparc_gpu_create(const sparc_gpu_desc *desc, sparc_gpu_ctx **out);
int sparc_gpu_destroy(sparc_gpu_ctx *ctx);

/* New effective potential for the next SCF iteration: copies N_d doubles from
 * veff_dev into the context's own buffer, asynchronously on `stream`. */
int sparc_gpu_set_veff(sparc_gpu_ctx *ctx, const double *veff_dev, void *stream);

/* Scratch needed by `op` on `ns` columns.  `block` is the column block (apply, filter, project) or the
 * row panel (rotate) the call will be given; <= 0 means "library chooses" (query with the same value
 * you will pass to the call). */
int sparc_gpu_workspace_bytes(const sparc_gpu_ctx *ctx, int op, int64_t ns, int64_t block,
                              int64_t *bytes);

/* Declare the size in bytes of the buffer that will be passed as `ws_dev` to the following calls on this context
 * (0 = undeclared: no check, the caller vouches for sparc_gpu_workspace_bytes).  Host-side state only. */
int sparc_gpu_set_workspace_size(sparc_gpu_ctx *ctx, int64_t bytes);

/* Y = H X on ncols columns (eq. 4, 122-126).  X and Y must not overlap.
 * ldx, ldy >= N_d.  X is not modified. */
int sparc_gpu_hamiltonian_apply(sparc_gpu_ctx *ctx, const double *X_dev, int64_t ldx, double *Y_dev,
                                int64_t ldy, int64_t ncols, void *ws_dev, void *stream);

/* In-place scaled Chebyshev filter (three-term scaled recurrence of refs [61,62], R3):
 *   e = (b-a)/2, c = (b+a)/2, sigma_1 = e/(a0-c), tau = 2/sigma_1,
 *   Y_1 = (sigma_1/e)(H X - c X);  Y_{k+1} = (2 sigma_{k+1}/e)(H Y_k - c Y_k) - sigma_k sigma_{k+1} Y_{k-1},
 *   sigma_{k+1} = 1/(tau - sigma_k);   Psi <- Y_degree  ( = T_m((H-cI)/e) Psi / T_m((a0-c)/e) ).
 * b = upper bound of the spectrum (lambda_Nd), a = filter cutoff (lambda_c), a0 = lower bound; requires
 * a0 < a < b (BAD_BOUNDS).  degree = 0 is the identity, degree < 0 INVALID_ARG (R4).  Columns are
 * processed in blocks of `col_block` (<= 0: library chooses); the result does not depend on it (R19). */
int sparc_gpu_chebyshev_filter(sparc_gpu_ctx *ctx, double *Psi_dev, int64_t ld, int64_t ns, int degree,
                               double a, double b, double a0, int64_t col_block, void *ws_dev,
                               void *stream);

/* Hs = Psi^T (H Psi), Ms = Psi^T Psi (R11: H Psi is formed internally by
 * column blocks).  Both outputs are full ns x ns matrices with both triangles filled (R12). */
int sparc_gpu_project(sparc_gpu_ctx *ctx, const double *Psi_dev, int64_t ld, int64_t ns, double *Hs_dev,
                      double *Ms_dev, int64_t col_block, void *ws_dev, void *stream);

/* Psi <- Psi Q in place, by row panels of `row_panel` rows (<= 0: library chooses) staged through the
 * workspace.  The result does not depend on row_panel (R19). */
int sparc_gpu_rotate(sparc_gpu_ctx *ctx, double *Psi_dev, int64_t ld, int64_t ns, const double *Q_dev,
                     int64_t row_panel, void *ws_dev, void *stream);

/* ---- gradient stencil and projector contraction for the nonlocal force ----------------
 * PAPER.md:110 "the application of the gradient operator on the Kohn-Sham orbitals" and "nonlocal projector
 * multiplications" are the two kernels of the nonlocal Hellmann-Feynman force. */

/* Y = D_axis X on ncols columns: central finite-difference FIRST derivative of the same order n0 as the Laplacian
 * (radius n0/2; weights w_p = (-1)^{p+1} (n!)^2 / (p (n-p)! (n+p)!), w_{-p} = -w_p, reading R21), along axis 0 (x), 1 (y)
 * or 2 (z); periodic axes wrap, neighbours outside a Dirichlet face contribute 0 (R9).  X and Y must not overlap. */
int sparc_gpu_gradient(sparc_gpu_ctx *ctx, int axis, const double *X_dev, int64_t ldx, double *Y_dev, int64_t ldy,
                       int64_t ncols, void *stream);

/* W = chi^T X: W[po_J + q, col] = sum_t chi_J[t, q] X[idx_J[t], col], po_J = sum_{I<J} P_I; no Gamma, no volume factor
 * (R6, R7).  W_dev: n_proj_total x ncols column-major, ld = n_proj_total. */
int sparc_gpu_nl_project(sparc_gpu_ctx *ctx, const double *X_dev, int64_t ldx, int64_t ncols, double *W_dev, void *stream);

/* W = chi^T (D_axis X), the gradient formed by column blocks in the workspace (op GRADIENT_PROJECT). */
int sparc_gpu_gradient_project(sparc_gpu_ctx *ctx, int axis, const double *X_dev, int64_t ldx, int64_t ncols,
                               double *W_dev, int64_t col_block, void *ws_dev, void *stream);

/* Nonlocal Hellmann-Feynman force (reading R22):
 *   F[J, a] = -2 sum_n occ[n] sum_q gamma_Jq (chi_Jq^T psi_n) (chi_Jq^T D_a psi_n),
 * occ_dev[ns] = occupation (times spin degeneracy) of each orbital; F_dev: n_atoms x 3 doubles, row-major (F[3 J + a]),
 * overwritten.  Workspace op NONLOCAL_FORCE.  Bitwise reproducible (fixed reduction order). */
int sparc_gpu_nonlocal_force(sparc_gpu_ctx *ctx, const double *Psi_dev, int64_t ld, int64_t ns, const double *occ_dev,
                             double *F_dev, int64_t col_block, void *ws_dev, void *stream);

/* ---- the subspace eigenproblem on the device ---------------------------------------------
 * Generalized symmetric-definite eigenproblem  Hs Z = Ms Z D  of the subspace step (Algorithm 1
 * "Subspace diagonalization", 148-154 eq. 9; the paper calls cusolverDnDsygvd).  Hs symmetric, Ms symmetric positive
 * definite, both n x n column-major (ld = n), read only.  Outputs: D_dev[n] ascending; Z_dev n x n column-major with
 * Z^T Ms Z = I, unique up to the sign of each column and rotations inside degenerate eigenspaces (reading R23) -- Z is the Q
 * of sparc_gpu_rotate.  Method: Cholesky Ms = L L^T, A = L^-1 Hs L^-T, one-sided Jacobi on a Cholesky factor of the shifted
 * A, Rayleigh-quotient eigenvalues, Z = L^-T V (csrc/eig.cu).  Everything is queued on `stream`; convergence is tested on the
 * device.  info_dev (2 x int32): [0] status 0 ok / 1 Ms not positive definite / 2 not converged, [1] sweeps.  The call returns
 * SUCCESS in all three cases (it never waits for the device): with status 1 or 2 Z and D are NOT usable, so pass info_dev and
 * read it after synchronising -- NULL is accepted, but then a failed solve is silent.  A fixed number of sweep launches (30) is
 * always queued; the ones after convergence return at once.
 * Workspace op EIGENSOLVE with ns = n.  n <= 12800 (a column pair must fit shared memory), else UNSUPPORTED. */
int sparc_gpu_eigensolve(sparc_gpu_ctx *ctx, int64_t n, const double *Hs_dev, const double *Ms_dev, double *Z_dev,
                         double *D_dev, int32_t *info_dev, void *ws_dev, void *stream);

/* ---- complex (k-point) variant ------------------------------------------------------------
 * PAPER.md:35 ("complex-valued ... Bloch wavevectors"), 126 / 146 / 166 (the Zgemm forms), 176 (Monkhorst-Pack grids).
 * Complex arrays are interleaved (re, im) doubles; leading dimensions and ns x ns sizes count COMPLEX elements.
 * Readings R24-R27: psi(r + L_a e_a) = exp(i theta_a) psi(r) on a periodic axis (theta_a = k_a L_a; ignored on Dirichlet axes):
 * a stencil tap wrapping through the upper (lower) face of axis a carries exp(+i theta_a) (exp(-i theta_a)); a support row
 * folded into the cell by the image shift w_a in {-1, 0, +1} per axis acts as chi~[t, q] = chi[t, q] exp(-i sum_a w_a theta_a),
 * V_nl = sum_J chi~_J Gamma_J chi~_J^H (chi real). */

/* Select the k-point of the following *_k calls.  theta: 3 doubles (HOST); supp_shift: int8 [supp_total][3] image shifts of the
 * support rows in the order of desc->supp_idx (HOST), or NULL (all zero).  Blocking (synchronises the device, uploads tables). */
int sparc_gpu_set_kpoint(sparc_gpu_ctx *ctx, const double *theta, const int8_t *supp_shift);

/* Y = H(k) X on complex columns (workspace op HAMILTONIAN_APPLY_K). */
int sparc_gpu_hamiltonian_apply_k(sparc_gpu_ctx *ctx, const double *X_dev, int64_t ldx, double *Y_dev, int64_t ldy,
                                  int64_t ncols, void *ws_dev, void *stream);
/* In-place scaled Chebyshev filter with H(k): the recurrence of sparc_gpu_chebyshev_filter on complex columns. */
int sparc_gpu_chebyshev_filter_k(sparc_gpu_ctx *ctx, double *Psi_dev, int64_t ld, int64_t ns, int degree, double a,
                                 double b, double a0, int64_t col_block, void *ws_dev, void *stream);
/* Hs = Psi^H (H(k) Psi), Ms = Psi^H Psi: complex ns x ns column-major, Hermitian up to rounding, both triangles filled
 * (PAPER.md:146 cublasZgemm with the conjugate transpose). */
int sparc_gpu_project_k(sparc_gpu_ctx *ctx, const double *Psi_dev, int64_t ld, int64_t ns, double *Hs_dev, double *Ms_dev,
                        int64_t col_block, void *ws_dev, void *stream);
/* Psi <- Psi Q in place by row panels, Q complex ns x ns (PAPER.md:166 cublasZgemm). */
int sparc_gpu_rotate_k(sparc_gpu_ctx *ctx, double *Psi_dev, int64_t ld, int64_t ns, const double *Q_dev, int64_t row_panel,
                       void *ws_dev, void *stream);

/* ---- local pieces of the row-partitioned projection and rotation -----------------------------
 * With X and Y = H X redistributed into row blocks X~^(k), Y~^(k) (eq. 5), rank k forms
 * H~^(k) = X~^(k)T Y~^(k), M~^(k) = X~^(k)T X~^(k) (eqs. 6-8; the sums over k are one all-reduce each, made by the
 * caller, paper_2302_09708_b200/dist.py) and later rotates its rows, X^(k) = X~^(k) Z~ (eqs. 10-11). */

/* C (m x n, column-major, ld = m) = A^T B, contraction over `nrows` rows; A: nrows x m (lda), B: nrows x n (ldb).
 * symmetric != 0 (needs m = n and a product that IS symmetric, e.g. A = B): upper-triangle tiles + mirror (R12).
 * Workspace op GRAM with ns = max(m, n).  nrows = 0 (a rank that owns no rows): C is zeroed; A_dev, B_dev and ws_dev are not
 * looked at and may be NULL. */
int sparc_gpu_gram(sparc_gpu_ctx *ctx, const double *A_dev, int64_t lda, const double *B_dev, int64_t ldb, int64_t nrows,
                   int64_t m, int64_t n, double *C_dev, int symmetric, void *ws_dev, void *stream);

/* X <- X Q in place on a block of `nrows` rows (ld >= nrows): sparc_gpu_rotate for a row block (workspace op ROTATE). */
int sparc_gpu_rotate_rows(sparc_gpu_ctx *ctx, double *X_dev, int64_t ld, int64_t nrows, int64_t ns, const double *Q_dev,
                          int64_t row_panel, void *ws_dev, void *stream);

/* ---- The Gram product for callers that cannot allocate device memory ------------------------------------------------------------
 * sparc_gpu_gram wants two things a caller may be unable to give at the moment it needs X^T Y: a context (sparc_gpu_create
 * uploads its tables with cudaMalloc) and a workspace for the split-K partial products.  Who is in that position:
 *   - an SCF driver that has given all free HBM to its own arena for the orbital blocks (Psi of the largest workload is 82 GB;
 *     with H Psi beside it nothing is left to lend as ws_dev), or an MPI rank under a per-process memory cap (MPS, MIG slice)
 *     where a cudaMalloc in the middle of an SCF iteration can fail;
 *   - code inside an overlapped region, such as the distributed step with copies, collectives and kernels in flight on several
 *     streams: cudaFree waits for the whole device and cudaMalloc may, so either one stalls every stream;
 *   - a plug-in inside a host application whose rules route all device memory through the host's allocator.
 * sparc_gpu_gram_static computes the same C = A^T B (layouts, `symmetric` and the fixed-order, bitwise repeatable reduction
 * as in sparc_gpu_gram) and calls no cudaMalloc, cudaFree or allocating library routine, ever.  It needs no context, only the
 * device ordinal.  Its split-K partial products go to an array of SPARC_GPU_GRAM_STATIC_MAX_ELEMS doubles (16 MiB) that is
 * compiled into the library: every GPU on which the library's code gets loaded holds those 16 MiB until the process exits.
 *   Limit: m * n <= SPARC_GPU_GRAM_STATIC_MAX_ELEMS (e.g. 1448 x 1448); beyond it the call does nothing and returns
 *          SPARC_GPU_STATIC_SCRATCH_EXCEEDED.  nrows is not limited.  Fewer partials fit than in a 2 GiB workspace, so for
 *          m * n above 32768 the row split can differ from sparc_gpu_gram's: results agree to rounding, not bit for bit.
 *   First call on a device: looks up the array's address on that GPU (cudaGetSymbolAddress) and sets kernel attributes.  Make
 *          that first call ahead of any stream capture; a call with nrows = 0 (C is zeroed) is enough.  Thread-safe.
 *   Sharing: there is ONE array per GPU, shared by every call from every thread.  Two calls whose kernels can overlap on the
 *          GPU (different streams with no dependency between them) race on it and give wrong results; calls on one stream,
 *          or ordered by events, are safe.  The array keeps whatever the last call left in it; each call overwrites every
 *          element it later reads, so nothing has to be (or is) cleared between calls.
 * Errors: INVALID_ARG (NULL / negative / lda, ldb < nrows / symmetric with m != n / device outside 0..63), UNSUPPORTED (device
 * is not compute capability 10.x), STATIC_SCRATCH_EXCEEDED, CUDA_ERROR.  nrows = 0 zeroes C. */
#define SPARC_GPU_GRAM_STATIC_MAX_ELEMS 2097152
int sparc_gpu_gram_static(int device, const double *A_dev, int64_t lda, const double *B_dev, int64_t ldb, int64_t nrows,
                          int64_t m, int64_t n, double *C_dev, int symmetric, void *stream);

/* One whole CheFSI step -- filter, project, rotate -- for a block that lives in HOST memory (what the paper's code does
 * around every step with cublasSet/GetVector: PAPER.md:118, 128, 138, 146, 158, 166), with the PCIe copies overlapped with
 * the kernels: columns are uploaded chunk by chunk while earlier chunks are filtered (columns are independent,
 * PAPER.md:120); Hs and Ms are downloaded when the projection is done; the rotation runs row panel by row panel
 * and every finished panel is downloaded while the next one is multiplied.
 *   Psi_in_host, Psi_out_host : N_d x ns column-major, ld_host >= N_d, HOST (pinned memory for full PCIe rate; they may
 *                               be the same buffer)
 *   Q_host (in), Hs_host, Ms_host (out) : ns x ns column-major HOST.  Q is the caller's eigenvector matrix; the
 *                               eigensolve stays outside this call (a caller that needs Hs, Ms first uses
 *                               sparc_gpu_eigensolve on the device or the separate operator calls)
 *   Psi_dev  : DEVICE scratch for the block, N_d x ns with ld_dev >= N_d;  mats_dev: DEVICE scratch of 3 ns^2 doubles
 *   ws_dev   : DEVICE scratch of max(workspace_bytes(CHEBYSHEV_FILTER), workspace_bytes(PROJECT), workspace_bytes(ROTATE))
 * Work is queued on `stream` and two copy streams owned by the context; the call SYNCHRONISES all three before it returns,
 * on success and on every error return alike (nothing is left in flight into the caller's buffers). */
int sparc_gpu_chefsi_step_host(sparc_gpu_ctx *ctx, const double *Psi_in_host, double *Psi_out_host, int64_t ld_host,
                               int64_t ns, int degree, double a, double b, double a0, const double *Q_host,
                               double *Hs_host, double *Ms_host, double *Psi_dev, int64_t ld_dev, double *mats_dev,
                               int64_t col_block, int64_t row_panel, void *ws_dev, void *stream);

/* The same step with the subspace eigenproblem inside it -- Algorithm 1 as the paper states it (filter,
 * project, "Subspace diagonalization", rotate): after the projection Hs Z = Ms Z D is solved on the device (sparc_gpu_eigensolve,
 * no host LAPACK in between) and the block is rotated by Z.  Differences from sparc_gpu_chefsi_step_host:
 *   D_host (out, ns doubles, ascending), info_host (out, 2 x int32: [0] status 0 ok / 1 Ms not positive definite / 2 Jacobi not
 *   converged, [1] sweeps) replace Q_host.  The host waits once mid-step for info.  Status 1: the block is NOT rotated,
 *   Psi_out_host receives the filtered block and the call still returns SUCCESS -- check info_host[0].
 *   mats_dev : 3 ns^2 + ns + 1 doubles (Hs, Ms, Z, then D and info);
 *   ws_dev   : additionally >= workspace_bytes(EIGENSOLVE, ns).  ns is bounded as in sparc_gpu_eigensolve. */
int sparc_gpu_chefsi_step_host_solve(sparc_gpu_ctx *ctx, const double *Psi_in_host, double *Psi_out_host, int64_t ld_host,
                                     int64_t ns, int degree, double a, double b, double a0, double *D_host, int32_t *info_host,
                                     double *Hs_host, double *Ms_host, double *Psi_dev, int64_t ld_dev, double *mats_dev,
                                     int64_t col_block, int64_t row_panel, void *ws_dev, void *stream);

/* ---- support entry points (not operators of the method) ------------------------------------- */

/* dst[k] = lo + (hi-lo) * u(seed, stream_id, index0 + k), k < count: the counter-based uniform generator
 * of the synthetic workloads, restated on the device so that large Psi blocks never
 * cross PCIe.  dst_dev is a device pointer. */
int sparc_gpu_fill_uniform(double *dst_dev, int64_t count, uint64_t seed, uint64_t stream_id,
                           uint64_t index0, double lo, double hi, int device, void *stream);

/* Register-resident throughput probes: the roofline denominators of the FP64-bound kernels, measured on the
 * device the library runs on.  kind 0: FP64 FMA (DFMA) TFLOP/s; kind 1: FP64 tensor
 * (DMMA m8n8k4) TFLOP/s; kind 2: device copy GB/s (read + write bytes) over scratch_dev.  value_out is a HOST
 * pointer; scratch_dev a DEVICE buffer of scratch_bytes (>= 64; kind 2 copies its first half onto its second).
 * Synchronises `stream` (best of 4 timed repetitions after a warm-up).  Not an operator of the method. */
int sparc_gpu_probe_peak(int device, int kind, double *value_out, void *scratch_dev, int64_t scratch_bytes,
                         void *stream);

/* Tuning / test knobs (host-side state of the context; unknown key or out-of-range value -> INVALID_ARG).
 *   "stencil_path"    0 auto, 1 generic kernel, 2 TMA + DFMA kernel, 3 TMA + DMMA in-plane taps; 2 and 3 make the
 *                     operator call return UNSUPPORTED when the grid does not meet their preconditions
 *   "nonlocal"        1 on, 0 off: drops V_nl (used by closed-form pins)
 *   "nonlocal_mode"   0 auto (brick-tiled DMMA kernel when supported, else 2), 1 project + pull: bitwise reproducible,
 *                     2 per-atom kernel with atomic scatter, 3 brick kernel or UNSUPPORTED
 *   "nlb_kernel"      brick kernel: 0 auto (persistent kernel when every brick's chi blocks fit its store), 1 general
 *                     kernel, 2 persistent kernel or UNSUPPORTED;  "nlb_cap" (test knob): cap on the chi blocks kept in
 *                     shared memory by the general kernel (forces load rounds);  "nlb_dbg": timing experiments only
 *   "gemm_path"       0 auto, 1 simple FMA kernel, 2 DMMA kernel
 *   "gemm_full"       0: Hs, Ms as upper-triangle tiles + mirror (R12), 1: all tiles
 *   "stencil_ay" (0 auto, 1, 2), "stencil_ty" (0 auto, else tile rows), "stencil_stages" (0 auto, 2..8 TMA ring depth),
 *   "stencil_zchunks" (0 auto), "stencil_xt" (0 auto, else 32..96 multiple of 8: x-tile width of the hybrid kernel on grids
 *   wider than 96 points): tile knobs of the stencil kernels
 *   "eig_coop"        1 (default): one cooperative launch per Jacobi sweep of sparc_gpu_eigensolve, 0: one launch per round
 *   "profile" (0 / 1), "profile_reset": per-kernel CUDA-event timing, read back through sparc_gpu_get_info */
int sparc_gpu_set_option(sparc_gpu_ctx *ctx, const char *key, int64_t value);

/* Read-only counters / facts.  key:
 *   "kernel_launches" (cumulative kernels launched by this context), "nd", "n_proj_total", "covered_points", "sm_count",
 *   "stencil_path_last" (1 generic, 2 TMA + DFMA, 3 TMA + DMMA hybrid: the kernel the last local pass used),
 *   "nl_brick" (1: the brick tables exist), "nl_brick_blocks", "nl_brick_active" (chi blocks / bricks with work),
 *   "nl_brick_max_blocks", "nl_brick_max_jobs" (most chi blocks / atoms of any one brick),
 *   "gemm_tn_mflop", "gemm_nn_mflop" (flop issued by the DMMA GEMMs since the last "profile_reset", in 1e6),
 *   "prof_count:<k>" launches and "prof_ns:<k>" summed nanoseconds of kernel kind k since the last "profile_reset"
 *   (k: 0 generic stencil, 1 TMA stencils, 2 nl project, 3 nl pull, 4 GEMM TN, 5 GEMM NN, 6 split-K reduce, 7 copies /
 *   mirror, 8 per-atom nonlocal, 9 brick nonlocal, 10 gradient stencil / force contraction, 11 eigensolver kernels, 12 k-point kernels).  "prof_ns:<k>" waits for
 *   the recorded events (cudaEventSynchronize): the one get_info key that blocks. */
int sparc_gpu_get_info(const sparc_gpu_ctx *ctx, const char *key, int64_t *value);

const char *sparc_gpu_error_string(int code);
const char *sparc_gpu_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPARC_GPU_H */
