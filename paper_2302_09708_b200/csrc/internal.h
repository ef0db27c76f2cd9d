// internal.h -- shared declarations of the sparc_gpu CUDA library (product code; not used by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/sparc_gpu.h"

#define SPARC_MAX_RADIUS 6
#define SPARC_MAX_PROJ 16

// Coefficients of one fused stencil pass.  With H_loc = -1/2 L + Veff the kernel computes
//   Out = alpha * (H_loc X + shift * X) + beta * Prev
// cx/cy/cz[p] = -1/2 * w_p / h_axis^2 (p = 1..radius), c0 = -1/2 * w_0 * sum_axis 1/h_axis^2.
struct StencilCoef {
    double cx[SPARC_MAX_RADIUS + 1];
    double cy[SPARC_MAX_RADIUS + 1];
    double cz[SPARC_MAX_RADIUS + 1];
    double c0;
};

// One entry of the point -> (atom, support row) inverse map used by the nonlocal pull kernel.
struct CoverEntry {
    int64_t chi_off;   // offset (doubles) of chi_J[t, 0]
    int32_t n_j;       // stride between projector columns of chi_J
    int32_t pofs_p;    // (offset of atom J's first projector in D) << 8 | P_J
};

// Tables of the brick-tiled nonlocal kernel (nonlocal_brick.cu): built at create, immutable.
struct NlBrick {
    int ok = 0;                // 0: grid does not meet the preconditions, per-atom kernels are used
    int pclass = 0;            // 4 or 9: projector-count class the blocks are laid out for
    int bx = 0, by = 0, bz = 0;   // brick shape, bx * by * bz = 128
    int32_t n_active = 0;      // bricks met by at least one support
    int64_t n_blocks = 0;      // chi blocks = touched (brick, atom, octet) triples
    int32_t *d_org = nullptr;      // [n_active][4]: x0, y0, z0, union octet mask
    int32_t *d_job_ptr = nullptr;  // [n_active + 1]
    void *d_jobs = nullptr;        // BrickJob[]
    int64_t max_blocks = 0;        // most chi blocks any one brick has
    int64_t max_jobs = 0;          // most atoms meeting any one brick
    double *d_blk = nullptr;       // chi sqrt|gamma| blocks, one copy serving pull and projection
};

// Tile choice of the TMA stencil kernel (stencil_tma.cu): depends only on the grid, the boundary flags and the
// "stencil_*" options, so it is computed once per context and invalidated by sparc_gpu_set_option.
struct StencilTileChoice {
    int valid = 0;             // 0: not computed yet, 1: usable, -1: no tile fits (kernel unsupported on this grid)
    int AY = 0, TY = 0, threads = 0, ctas_per_sm = 0, nstage = 0, W = 0, variant = 0;
    uint32_t psi_bytes = 0, tile_bytes = 0, stage_bytes = 0;
    size_t smem = 0;
};

struct sparc_gpu_ctx {
    int device = 0;
    int sm_count = 0;
    int32_t n[3] = {0, 0, 0};
    double h[3] = {0, 0, 0};
    int32_t bc[3] = {0, 0, 0};
    int32_t radius = 0;
    int64_t nd = 0;
    StencilCoef coef = {};     // alpha = 1 coefficients (host copy)
    double w[SPARC_MAX_RADIUS + 1] = {0};
    double w1[SPARC_MAX_RADIUS + 1] = {0};   // first-derivative weights (gradient stencil, forces)
    // nonlocal tables (device)
    int32_t n_atoms = 0;
    int32_t n_proj_total = 0;
    int32_t max_proj = 0;
    int64_t supp_total = 0;
    int64_t *d_supp_ptr = nullptr;       // [n_atoms+1]
    int32_t *d_supp_idx = nullptr;       // [supp_total]
    int32_t *d_n_proj = nullptr;         // [n_atoms]
    int32_t *d_proj_ofs = nullptr;       // [n_atoms+1] prefix sum of n_proj
    int64_t *d_chi_ptr = nullptr;        // [n_atoms+1]
    double *d_chi = nullptr;
    double *d_gamma = nullptr;           // [n_proj_total]
    // inverse (pull) map
    int64_t n_covered = 0;
    int32_t *d_cov_idx = nullptr;        // [n_covered] grid index of each covered point (ascending)
    int64_t *d_cov_ptr = nullptr;        // [n_covered+1] offsets into d_cov_ent
    CoverEntry *d_cov_ent = nullptr;     // [supp_total]
    NlBrick nlb;
    // local potential
    double *d_veff = nullptr;            // [nd]
    // options
    int opt_stencil_path = 0;      // 0 auto, 1 generic, 2 TMA (DFMA), 3 TMA + DMMA in-plane taps
    int opt_nonlocal = 1;          // 1 on
    int opt_gemm_path = 0;         // 0 auto, 1 simple, 2 DMMA
    int opt_nlb_kernel = 0;        // brick kernel: 0 auto (persistent when every brick fits its store), 1 general, 2 persistent
    int opt_nlb_cap = 0;           // test knob: cap on the chi blocks the brick kernel keeps in shared memory (0 = all that fit)
    int opt_nlb_dbg = 0;           // timing experiments (nonlocal_brick.cu)
    int opt_gemm_full = 0;         // 0: Hs, Ms computed as upper triangle + mirror (R12); 1: all tiles
    int opt_nonlocal_mode = 0;     // 0 auto (brick kernel when supported, else 2), 1 project + pull (deterministic),
                                   // 2 per-atom kernel with atomic scatter, 3 brick kernel or UNSUPPORTED
    int opt_stencil_ay = 0;        // 0 auto, 1 or 2: rows per consumer thread of the TMA stencil kernel
    int opt_stencil_ty = 0;        // 0 auto, else forced tile rows of the TMA stencil kernel
    int opt_stencil_stages = 0;    // 0 auto, else cap on the smem ring depth (2..8)
    int opt_stencil_xt = 0;        // 0 auto, else forced x-tile width of the hybrid stencil on grids wider than 96 (32..96, multiple of 8)
    int opt_eig_coop = 1;          // eigensolve: 1 = one cooperative launch per Jacobi sweep (grid barrier between rounds), 0 = one launch per round
    int opt_stencil_zchunks = 0;   // 0 auto, else forced number of z chunks
    // size of the buffer the caller passes as ws_dev (sparc_gpu_set_workspace_size); 0 = not declared, no check
    int64_t ws_bytes = 0;
    // counters
    mutable int64_t kernel_launches = 0;
    double gemm_flop[2] = {0, 0};  // flop issued by the DMMA GEMMs since the last "profile_reset": [0] TN, [1] NN
    int stencil_path_last = 0;
    mutable StencilTileChoice tma_choice;  // cache (stencil_tma.cu)
    uint64_t func_attr_done = 0;   // kernel variants whose dynamic shared-memory attribute is set (nonlocal_brick.cu)
    // driver entry point for tensor-map encoding (resolved at create; NULL if unavailable)
    void *fn_encode_tiled = nullptr;
    // k-point state (kpoint.cu): Bloch phase per axis, exp(i phi_t) per support row and per cover entry
    double k_theta[3] = {0, 0, 0};
    int k_set = 0;
    double2 *d_k_phase = nullptr;        // [supp_total]
    double2 *d_k_cov_phase = nullptr;    // [supp_total], in the order of d_cov_ent
    std::vector<int64_t> h_cov_row;      // host: global support row of each cover entry
    // copy streams of the host-buffer entry point (step_host.cu), created on first use
    cudaStream_t copy_stream[2] = {nullptr, nullptr};
    // optional per-kernel CUDA-event timing (option "profile"); NULL when off
    struct ProfState *prof = nullptr;
};

// Make ctx->device current for the duration of a C-ABI call and restore the caller's device afterwards.
struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { (void)cudaGetLastError(); prev = -1; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) { (void)cudaGetLastError(); ok = false; }
    }
    ~DeviceGuard() { if (prev >= 0) (void)cudaSetDevice(prev); }
};

// Kernel kinds for the event profiler and the launch counters.
enum KernelKind {
    KK_STENCIL_GENERIC = 0, KK_STENCIL_TMA = 1, KK_NL_PROJECT = 2, KK_NL_PULL = 3, KK_GEMM_TN = 4,
    KK_GEMM_NN = 5, KK_SPLITK_REDUCE = 6, KK_COPY2D = 7, KK_NL_FUSED = 8, KK_NL_BRICK = 9, KK_GRADIENT = 10, KK_EIG = 11, KK_KPOINT = 12, KK_COUNT = 13
};
// Bracket one kernel launch with events when profiling is on (no-ops otherwise); both bump the counters.
void prof_begin(sparc_gpu_ctx *ctx, int kind, cudaStream_t st);
void prof_end(sparc_gpu_ctx *ctx, int kind, cudaStream_t st);

#define SPARC_CUDA_TRY(expr)                                         \
    do {                                                             \
        cudaError_t _e = (expr);                                     \
        if (_e != cudaSuccess) {                                     \
            (void)cudaGetLastError();                                \
            return (_e == cudaErrorMemoryAllocation) ? SPARC_GPU_OUT_OF_MEMORY : SPARC_GPU_CUDA_ERROR; \
        }                                                            \
    } while (0)

#define SPARC_TRY(expr)                    \
    do {                                   \
        int _s = (expr);                   \
        if (_s != SPARC_GPU_SUCCESS) return _s; \
    } while (0)

static inline int64_t round_up_i64(int64_t v, int64_t m) { return (v + m - 1) / m * m; }

// Carving of the caller's workspace for one operator call (context.cu).
struct WsLayout {
    int64_t block;       // column block / row panel actually used
    int64_t ldw;         // leading dimension of the work block
    int64_t off_w, off_d, off_g;
    int64_t total;
};
int ws_layout(const sparc_gpu_ctx *c, int op, int64_t ns, int64_t block, WsLayout *L);
int ws_check(const sparc_gpu_ctx *c, const WsLayout &L);
int ws_layout_k(const sparc_gpu_ctx *c, int op, int64_t ns, int64_t block, WsLayout *L);   // k-point operators (kpoint.cu)
void kpoint_free(sparc_gpu_ctx *c);

// ---- kernel launchers (each returns a sparc_gpu_status and bumps ctx->kernel_launches) ----------

// Out = alpha * (H_loc X + shift X) + beta * Prev   (Prev may be NULL when beta == 0; Prev may alias Out)
int launch_stencil_generic(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, double *Out, int64_t ldo,
                           const double *Prev, int64_t ldp, int64_t ncols, double alpha, double shift,
                           double beta, cudaStream_t st);
// same contract; returns SPARC_GPU_UNSUPPORTED if the shape does not meet the TMA kernel's preconditions
int launch_stencil_tma(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, double *Out, int64_t ldo,
                       const double *Prev, int64_t ldp, int64_t ncols, double alpha, double shift,
                       double beta, cudaStream_t st);
// same contract; hybrid kernel: in-plane taps as DMMA, z taps as DFMA (stencil_dmma.cu)
int launch_stencil_dmma(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, double *Out, int64_t ldo,
                        const double *Prev, int64_t ldp, int64_t ncols, double alpha, double shift,
                        double beta, cudaStream_t st);
bool stencil_dmma_supported(const sparc_gpu_ctx *ctx, const double *X, int64_t ldx, const double *Out,
                            int64_t ldo, const double *Prev, int64_t ldp);
bool stencil_tma_supported(const sparc_gpu_ctx *ctx, const double *X, int64_t ldx, const double *Out,
                           int64_t ldo, const double *Prev, int64_t ldp);

// D[q, col] = scale * gamma[q] * sum_t chi[t, q] X[idx[t], col]     (D: n_proj_total x ncols, ld = n_proj_total)
int launch_nl_project(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, int64_t ncols, double scale,
                      double *D, cudaStream_t st);
// W[q, col] = sum_t chi[t, q] X[idx[t], col]   (no Gamma; W: n_proj_total x ncols, ld = n_proj_total)
int launch_nl_project_raw(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, int64_t ncols, double *W, cudaStream_t st);
// Out[i, col] += sum_{(J,t) covering i} sum_q chi_J[t, q] D[ofs_J + q, col]
int launch_nl_pull(sparc_gpu_ctx *ctx, const double *D, double *Out, int64_t ldo, int64_t ncols,
                   cudaStream_t st);

// Out[idx_J, col] += scale * chi_J diag(gamma_J) chi_J^T X[idx_J, col] for every atom J: fused gather / GEMM / atomic
// scatter (default nonlocal path; not bitwise reproducible across runs, see option "nonlocal_mode")
int launch_nl_fused(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, double *Out, int64_t ldo, int64_t ncols,
                    double scale, cudaStream_t st);

// Brick-tiled nonlocal kernel (nonlocal_brick.cu).  A C buffer holds D = scale Gamma chi^T Psi as one slab of up to 144 doubles
// per (atom, 16-column group), in the order of the pull kernel's operand fragments: nlb_c_doubles(ctx, ncols) doubles.
static inline int64_t nlb_c_cols(int64_t ncols) { return (ncols + 63) / 64 * 64; }
static inline int64_t nlb_c_doubles(const sparc_gpu_ctx *c, int64_t ncols)
{
    return (int64_t)(c->n_atoms > 0 ? c->n_atoms : 1) * 9 * nlb_c_cols(ncols);
}
//   mode 1 (project): c_out += scale Gamma chi^T X        (X read only; c_out zeroed by the caller)
//   mode 2 (pull)   : Out += chi c_in
//   mode 3 (both)   : Out += chi c_in, then c_out += scale Gamma chi^T Out   (scale: the alpha of the step that pulls c_out)
int nlb_build(sparc_gpu_ctx *ctx, const sparc_gpu_desc *d);
void nlb_free(sparc_gpu_ctx *ctx);
bool nlb_supported(const sparc_gpu_ctx *ctx, const double *X, int64_t ld);
int launch_nl_brick(sparc_gpu_ctx *ctx, int mode, double *XorOut, int64_t ld, int64_t ncols, double scale,
                    const double *c_in, double *c_out, cudaStream_t st);

// C (M x N, col-major, ldc) = A^T B, A: K x M (lda), B: K x N (ldb), contraction over K rows.
// ws: split-K partials (gemm_tn_ws_bytes).  diag >= 0: the result is (a column block, starting at global column diag,
// of) a symmetric matrix: tiles strictly below the diagonal may be skipped (launch_mirror_upper fills them in).
int64_t gemm_tn_ws_bytes(const sparc_gpu_ctx *ctx, int64_t M, int64_t N, int64_t K);
int launch_gemm_tn(sparc_gpu_ctx *ctx, const double *A, int64_t lda, const double *B, int64_t ldb,
                   double *C, int64_t ldc, int64_t M, int64_t N, int64_t K, void *ws, int64_t diag, cudaStream_t st);
// C[i, j] = C[j, i] for i > j (after a launch_gemm_tn with diag >= 0)
int launch_mirror_upper(sparc_gpu_ctx *ctx, double *C, int64_t ldc, int64_t n, cudaStream_t st);
// C (M x N, ldc) = A B, A: M x K col-major (lda), B: K x N col-major (ldb)
int launch_gemm_nn(sparc_gpu_ctx *ctx, const double *A, int64_t lda, const double *B, int64_t ldb,
                   double *C, int64_t ldc, int64_t M, int64_t N, int64_t K, cudaStream_t st);
// rotation by row panels (context.cu): panel size / stage pitch for ns columns, and one panel Psi_rows <- Psi_rows Q
int rotate_layout(const sparc_gpu_ctx *ctx, int64_t ns, int64_t row_panel, int64_t *rp, int64_t *ldw);
int rotate_panel(sparc_gpu_ctx *ctx, double *Psi_rows, int64_t ld, int64_t nr, int64_t ns, const double *Q, double *T,
                 int64_t ldw, cudaStream_t st);
// dst (rows x cols, ldd) = src (rows x cols, lds)
int launch_copy_2d(sparc_gpu_ctx *ctx, double *dst, int64_t ldd, const double *src, int64_t lds,
                   int64_t rows, int64_t cols, cudaStream_t st);
