// eig.cu -- SURVEY.md section 8(f) NEXT-1: the N_s x N_s generalized symmetric-definite eigenproblem of the subspace step
//   Hs Z = Ms Z D,  Z^T Ms Z = I,  D ascending          (Algorithm 1, 148-154 section II.C eq. 9)
// on the device, so that filter -> project -> solve -> rotate needs no host hop.  The paper calls cusolverDnDsygvd
// (PAPER.md:154); here every step is a hand-written FP64 kernel and the whole solve is queued asynchronously on one stream
// (convergence is tested on the device; the sweeps left over after convergence return at once).
//
//   E1  Ms = L L^T                     blocked right-looking Cholesky (64-wide panels: diagonal block, panel solve, trailing update)
//   E2  A  = L^-1 Hs L^-T              two blocked forward substitutions (the second on the transpose), then A <- (A + A^T)/2
//   E3  eigen-decomposition of A by the ONE-SIDED (Hestenes) Jacobi method on a Cholesky factor:
//         sigma = 1.05 max_i sum_j |A_ij| (Gershgorin: A + sigma I is positive definite with condition number <= 41),
//         A + sigma I = R R^T,  G = R^T  (so G^T G = A + sigma I);  plane rotations G <- G J, V <- V J make the columns of G
//         mutually orthogonal: then V^T (A + sigma I) V = diag(|g_j|^2), i.e. V = eigenvectors, |g_j|^2 - sigma = eigenvalues.
//         V is not accumulated during the sweeps: G_final = R^T V, so V = R^-T G_final (one back substitution).
//       Pairs follow the round-robin (tournament) ordering: n/2 disjoint column pairs per round, n - 1 rounds per sweep, one
//       CTA per pair.  Only whole columns are touched, so every access is a contiguous run (a two-sided Jacobi would also
//       rotate rows).  Jacobi on the Cholesky factor converges in few sweeps (Veselic-Hari).
//   E4  eigenvalues refined as Rayleigh quotients mu_j = v_j^T A v_j, sorted ascending (stable rank sort), Z = L^-T V
//       (blocked back substitution).
// info[0] = status: 0 ok, 1 Ms not positive definite, 2 Jacobi not converged in the sweep budget; info[1] = sweeps used.
#include <cooperative_groups.h>

#include <algorithm>

#include "internal.h"

namespace {

constexpr int NB = 64;            // panel width of the blocked factorisation / substitutions
constexpr int MAX_SWEEPS = 30;

struct EigScalars {               // device-side control block (in the workspace)
    double sigma;                 // Gershgorin shift
    double rowsum_max;            // max_i sum_j |A_ij| (bit pattern ordered as an unsigned integer: values are >= 0)
    unsigned long long off_max;   // largest |g_p . g_q| / (|g_p| |g_q|) seen in the current sweep (bits of a double >= 0)
    int done;                     // 1: converged (or failed): remaining kernels return at once
    int status;
    int sweeps;
    int pad;
};

// ---- C (m x n) -= op(A) op(B), op(A): m x k, op(B): k x n; 64 x 64 tile, 256 threads, 4 x 4 per thread -----------------
template <bool TA, bool TB>
__global__ void __launch_bounds__(256)
gemm_sub_kernel(int m, int n, int k, const double *__restrict__ A, int64_t lda, const double *__restrict__ B, int64_t ldb,
                double *C, int64_t ldc, const EigScalars *sc)
{
    if (sc && sc->status) return;
    __shared__ double As[16][64 + 1];
    __shared__ double Bs[16][64 + 1];
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    const int m0 = blockIdx.x * 64, n0 = blockIdx.y * 64;
    double acc[4][4] = {{0.0}};
    for (int k0 = 0; k0 < k; k0 += 16) {
        for (int e = threadIdx.x; e < 16 * 64; e += 256) {
            // A tile: (kk, i); B tile: (kk, j) -- the fastest index of e follows the contiguous global direction
            int kk, i;
            if (TA) { kk = e & 15; i = e >> 4; } else { i = e & 63; kk = e >> 6; }
            double v = 0.0;
            if (m0 + i < m && k0 + kk < k) v = TA ? A[(k0 + kk) + (int64_t)(m0 + i) * lda] : A[(m0 + i) + (int64_t)(k0 + kk) * lda];
            As[kk][i] = v;
            int j;
            if (TB) { j = e & 63; kk = e >> 6; } else { kk = e & 15; j = e >> 4; }
            v = 0.0;
            if (n0 + j < n && k0 + kk < k) v = TB ? B[(n0 + j) + (int64_t)(k0 + kk) * ldb] : B[(k0 + kk) + (int64_t)(n0 + j) * ldb];
            Bs[kk][j] = v;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < 16; ++kk) {
            double a[4], b[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) { a[r] = As[kk][tx + 16 * r]; b[r] = Bs[kk][ty + 16 * r]; }
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[r][c] = fma(a[r], b[c], acc[r][c]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int i = m0 + tx + 16 * r, j = n0 + ty + 16 * c;
            if (i < m && j < n) C[i + (int64_t)j * ldc] -= acc[r][c];
        }
}

// ---- Cholesky of the nb x nb diagonal block at A (lower triangle), one CTA; non-positive pivot -> status 1 ---------------
__global__ void __launch_bounds__(NB)
potrf_diag_kernel(int nb, double *A, int64_t lda, EigScalars *sc)
{
    if (sc->status) return;
    __shared__ double S[NB][NB + 1];
    const int t = threadIdx.x;
    for (int j = 0; j < nb; ++j)
        if (t < nb) S[t][j] = A[t + (int64_t)j * lda];
    __syncthreads();
    for (int j = 0; j < nb; ++j) {
        const double d = S[j][j];
        if (!(d > 0.0)) { if (t == 0) { sc->status = 1; sc->done = 1; } return; }
        const double r = sqrt(d);
        __syncthreads();
        if (t == j) S[j][j] = r;
        else if (t > j && t < nb) S[t][j] /= r;
        __syncthreads();
        // trailing update of row t: S[t][c] -= S[t][j] S[c][j], j < c <= t
        if (t > j && t < nb)
            for (int c = j + 1; c <= t; ++c) S[t][c] -= S[t][j] * S[c][j];
        __syncthreads();
    }
    for (int j = 0; j < nb; ++j)
        if (t < nb) A[t + (int64_t)j * lda] = (t >= j) ? S[t][j] : 0.0;
}

// ---- rows below the diagonal block: X L_kk^T = P, one thread per row (forward substitution along the row) -------------------
__global__ void __launch_bounds__(128)
trsm_panel_kernel(int m, int nb, const double *__restrict__ Lkk, int64_t ldl, double *P, int64_t ldp, const EigScalars *sc)
{
    if (sc->status) return;
    __shared__ double S[NB][NB + 1];
    for (int e = threadIdx.x; e < nb * nb; e += blockDim.x) S[e % nb][e / nb] = Lkk[(e % nb) + (int64_t)(e / nb) * ldl];
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    double x[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) {
        if (j < nb) {
            double s = P[i + (int64_t)j * ldp];
#pragma unroll
            for (int c = 0; c < NB; ++c)
                if (c < j) s -= x[c] * S[j][c];
            x[j] = s / S[j][j];
            P[i + (int64_t)j * ldp] = x[j];
        }
    }
}

// ---- diagonal block of a left solve: L_kk X = B (FWD) or L_kk^T X = B (backward), one thread per right-hand side ------------
template <bool FWD>
__global__ void __launch_bounds__(128)
trsm_diag_left_kernel(int nb, int nrhs, const double *__restrict__ Lkk, int64_t ldl, double *B, int64_t ldb, const EigScalars *sc)
{
    if (sc->status) return;
    __shared__ double S[NB][NB + 1];
    for (int e = threadIdx.x; e < nb * nb; e += blockDim.x) S[e % nb][e / nb] = Lkk[(e % nb) + (int64_t)(e / nb) * ldl];
    __syncthreads();
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= nrhs) return;
    double *b = B + (int64_t)j * ldb;
    double x[NB];
    if (FWD) {
#pragma unroll
        for (int i = 0; i < NB; ++i) {
            if (i < nb) {
                double s = b[i];
#pragma unroll
                for (int c = 0; c < NB; ++c)
                    if (c < i) s -= S[i][c] * x[c];
                x[i] = s / S[i][i];
            }
        }
    } else {
#pragma unroll
        for (int ii = 0; ii < NB; ++ii) {
            const int i = NB - 1 - ii;
            if (i < nb) {
                double s = b[i];
#pragma unroll
                for (int c = 0; c < NB; ++c)
                    if (c > i && c < nb) s -= S[c][i] * x[c];
                x[i] = s / S[i][i];
            }
        }
    }
#pragma unroll
    for (int i = 0; i < NB; ++i)
        if (i < nb) b[i] = x[i];
}

// dst (n x n, ldd) = src^T (lds); UPPER: keep only i <= j of dst (the rest zero)
template <bool UPPER>
__global__ void __launch_bounds__(256)
transpose_kernel(int n, const double *__restrict__ src, int64_t lds, double *dst, int64_t ldd)
{
    __shared__ double T[32][33];
    const int bx = blockIdx.x * 32, by = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int r = ty; r < 32; r += 8)
        if (bx + tx < n && by + r < n) T[r][tx] = src[(bx + tx) + (int64_t)(by + r) * lds];
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        const int i = by + tx, j = bx + r;            // dst(i, j) = src(j, i)
        if (i < n && j < n) dst[i + (int64_t)j * ldd] = (!UPPER || i <= j) ? T[tx][r] : 0.0;
    }
}

// dst = (src + src^T) / 2 and rowsum_max = max_i sum_j |dst_ij|  (one CTA per column = row, by symmetry)
__global__ void __launch_bounds__(256)
symmetrize_kernel(int n, const double *__restrict__ src, int64_t lds, double *dst, int64_t ldd, EigScalars *sc)
{
    if (sc->status) return;
    __shared__ double red[256];
    const int j = blockIdx.x;
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const double v = 0.5 * (src[i + (int64_t)j * lds] + src[j + (int64_t)i * lds]);
        dst[i + (int64_t)j * ldd] = v;
        s += fabs(v);
    }
    red[threadIdx.x] = s;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0)
        atomicMax(reinterpret_cast<unsigned long long *>(&sc->rowsum_max), (unsigned long long)__double_as_longlong(red[0]));
}

__global__ void set_shift_kernel(int n, double *A, int64_t lda, EigScalars *sc)
{
    if (sc->status) return;
    double sg = 1.05 * sc->rowsum_max;
    if (!(sg > 0.0)) sg = 1.0;                         // A = 0: any positive shift
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) A[i + (int64_t)i * lda] += sg;
    if (i == 0) sc->sigma = sg;
}

__global__ void init_scalars_kernel(EigScalars *sc)
{
    sc->sigma = 0.0; sc->rowsum_max = 0.0; sc->off_max = 0ull; sc->done = 0; sc->status = 0; sc->sweeps = 0; sc->pad = 0;
}

__device__ __forceinline__ double block_sum(double v, double *red)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5;
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[w] = v;
    __syncthreads();
    double s = 0.0;
    for (int k = 0; k < (int)(blockDim.x >> 5); ++k) s += red[k];     // fixed order: every thread gets the same bits
    return s;
}

// One pair of one tournament round: the CTA rotates the columns (p, q) of G (and of V, if accumulated) so that g_p . g_q = 0.
// Every thread of the CTA takes the same path (the barriers inside block_sum are uniform).
__device__ __forceinline__ void jacobi_pair(int n, int npad, int round, int k, double *G, int64_t ldg, double *V, int64_t ldv,
                                            double tol, EigScalars *sc, double *cols, double *red)
{
    const int m = npad - 1;
    int p, q;
    if (k == 0) { p = round % m; q = npad - 1; }
    else { p = (round + k) % m; q = (round - k + m) % m; }
    if (p > q) { const int t = p; p = q; q = t; }
    if (q >= n) return;                                // the bye of an odd n
    double *gp = G + (int64_t)p * ldg, *gq = G + (int64_t)q * ldg;
    double *sp = cols, *sq = cols + n;
    double a = 0.0, b = 0.0, c = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const double x = gp[i], y = gq[i];
        sp[i] = x; sq[i] = y;
        a = fma(x, x, a); b = fma(y, y, b); c = fma(x, y, c);
    }
    a = block_sum(a, red); b = block_sum(b, red); c = block_sum(c, red);
    const double denom = sqrt(a) * sqrt(b);
    const double off = denom > 0.0 ? fabs(c) / denom : 0.0;
    if (threadIdx.x == 0) atomicMax(&sc->off_max, (unsigned long long)__double_as_longlong(off));
    if (!(off > tol)) return;                          // already orthogonal to working precision
    const double zeta = (b - a) / (2.0 * c);
    const double t = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
    const double cs = 1.0 / sqrt(1.0 + t * t), sn = cs * t;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const double x = sp[i], y = sq[i];
        gp[i] = cs * x - sn * y;
        gq[i] = sn * x + cs * y;
    }
    if (!V) return;                                    // the rotations are recovered from G afterwards (V = G_0^-1 G)
    double *vp = V + (int64_t)p * ldv, *vq = V + (int64_t)q * ldv;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const double x = vp[i], y = vq[i];
        vp[i] = cs * x - sn * y;
        vq[i] = sn * x + cs * y;
    }
}

// One round per launch: CTA k takes pair k (the fallback when a cooperative launch is not possible).
__global__ void __launch_bounds__(256)
jacobi_round_kernel(int n, int npad, int round, double *G, int64_t ldg, double *V, int64_t ldv, double tol, EigScalars *sc)
{
    if (sc->done) return;
    extern __shared__ double cols[];                   // g_p, g_q
    __shared__ double red[8];
    jacobi_pair(n, npad, round, blockIdx.x, G, ldg, V, ldv, tol, sc, cols, red);
}

__device__ __forceinline__ void sweep_end(double tol, int last, EigScalars *sc)
{
    sc->sweeps += 1;
    const double off = __longlong_as_double((long long)sc->off_max);
    if (off <= tol) sc->done = 1;
    else if (last) { sc->done = 1; sc->status = 2; }
    sc->off_max = 0ull;
}

// A whole sweep (n - 1 rounds) in ONE cooperative launch: the co-resident CTAs share the pairs of a round and meet at a
// grid-wide barrier between rounds, which costs a fraction of a kernel launch -- for N_s <= 2048 the factor sits in L2 and the
// per-round launches were the bottleneck.  `done` is read once at the start (it only changes after the last barrier).
__global__ void __launch_bounds__(256)
jacobi_sweep_coop_kernel(int n, int npad, double *G, int64_t ldg, double tol, int last, EigScalars *sc)
{
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    extern __shared__ double cols[];
    __shared__ double red[8];
    if (sc->done) return;
    for (int r = 0; r < npad - 1; ++r) {
        for (int k = blockIdx.x; k < npad / 2; k += gridDim.x) {
            jacobi_pair(n, npad, r, k, G, ldg, nullptr, 0, tol, sc, cols, red);
            __syncthreads();                           // the staged pair is rewritten by the CTA's next pair
        }
        grid.sync();
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) sweep_end(tol, last, sc);
}

__global__ void sweep_end_kernel(double tol, int last, EigScalars *sc)
{
    if (sc->done) return;
    sweep_end(tol, last, sc);
}

// mu[j] = sign * v_j . w_j (Rayleigh quotient v_j^T A v_j with W = sign * A V precomputed), one CTA per column
__global__ void __launch_bounds__(256)
rayleigh_kernel(int n, const double *__restrict__ V, int64_t ldv, const double *__restrict__ AV, int64_t lda, double sign,
                double *mu)
{
    __shared__ double red[8];
    const int j = blockIdx.x;
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) s = fma(V[i + (int64_t)j * ldv], AV[i + (int64_t)j * lda], s);
    s = block_sum(s, red);
    if (threadIdx.x == 0) mu[j] = sign * s;
}

// stable ascending rank of mu[j]; D[rank] = mu[j]; column j of V goes to column rank of Vs
__global__ void __launch_bounds__(256)
rank_kernel(int n, const double *__restrict__ mu, int *rank, double *D)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const double v = mu[j];
    int r = 0;
    for (int i = 0; i < n; ++i) { const double u = mu[i]; r += (u < v || (u == v && i < j)) ? 1 : 0; }
    rank[j] = r;
    D[r] = v;
}

__global__ void __launch_bounds__(256)
permute_cols_kernel(int n, const double *__restrict__ V, int64_t ldv, const int *__restrict__ rank, double *Vs, int64_t lds)
{
    const int j = blockIdx.y;
    double *d = Vs + (int64_t)rank[j] * lds;
    const double *s = V + (int64_t)j * ldv;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) d[i] = s[i];
}

#define EIG_LAUNCH(kind, ...)                 \
    do {                                      \
        prof_begin(ctx, KK_EIG, st);          \
        __VA_ARGS__;                          \
        prof_end(ctx, KK_EIG, st);            \
        SPARC_CUDA_TRY(cudaGetLastError());   \
    } while (0)

int potrf_lower(sparc_gpu_ctx *ctx, int n, double *A, int64_t lda, EigScalars *sc, cudaStream_t st)
{
    for (int k0 = 0; k0 < n; k0 += NB) {
        const int nb = std::min(NB, n - k0), m = n - k0 - nb;
        double *Akk = A + k0 + (int64_t)k0 * lda;
        EIG_LAUNCH(0, (potrf_diag_kernel<<<1, NB, 0, st>>>(nb, Akk, lda, sc)));
        if (m > 0) {
            double *P = Akk + nb;
            EIG_LAUNCH(0, (trsm_panel_kernel<<<(m + 127) / 128, 128, 0, st>>>(m, nb, Akk, lda, P, lda, sc)));
            dim3 grid((m + 63) / 64, (m + 63) / 64);
            EIG_LAUNCH(0, (gemm_sub_kernel<false, true><<<grid, 256, 0, st>>>(m, m, nb, P, lda, P, lda, Akk + nb + (int64_t)nb * lda, lda, sc)));
        }
    }
    return SPARC_GPU_SUCCESS;
}

// L X = B in place (forward), B: n x nrhs
int trsm_lower_fwd(sparc_gpu_ctx *ctx, int n, int nrhs, const double *L, int64_t ldl, double *B, int64_t ldb, EigScalars *sc,
                   cudaStream_t st)
{
    for (int k0 = 0; k0 < n; k0 += NB) {
        const int nb = std::min(NB, n - k0), m = n - k0 - nb;
        const double *Lkk = L + k0 + (int64_t)k0 * ldl;
        EIG_LAUNCH(0, (trsm_diag_left_kernel<true><<<(nrhs + 127) / 128, 128, 0, st>>>(nb, nrhs, Lkk, ldl, B + k0, ldb, sc)));
        if (m > 0) {
            dim3 grid((m + 63) / 64, (nrhs + 63) / 64);
            EIG_LAUNCH(0, (gemm_sub_kernel<false, false><<<grid, 256, 0, st>>>(m, nrhs, nb, Lkk + nb, ldl, B + k0, ldb, B + k0 + nb, ldb, sc)));
        }
    }
    return SPARC_GPU_SUCCESS;
}

// L^T X = B in place (backward)
int trsm_lower_trans_bwd(sparc_gpu_ctx *ctx, int n, int nrhs, const double *L, int64_t ldl, double *B, int64_t ldb, EigScalars *sc,
                         cudaStream_t st)
{
    const int nblk = (n + NB - 1) / NB;
    for (int kb = nblk - 1; kb >= 0; --kb) {
        const int k0 = kb * NB, nb = std::min(NB, n - k0);
        const double *Lkk = L + k0 + (int64_t)k0 * ldl;
        EIG_LAUNCH(0, (trsm_diag_left_kernel<false><<<(nrhs + 127) / 128, 128, 0, st>>>(nb, nrhs, Lkk, ldl, B + k0, ldb, sc)));
        if (k0 > 0) {
            // B[0:k0, :] -= L[k0:k0+nb, 0:k0]^T X_k
            dim3 grid((k0 + 63) / 64, (nrhs + 63) / 64);
            EIG_LAUNCH(0, (gemm_sub_kernel<true, false><<<grid, 256, 0, st>>>(k0, nrhs, nb, L + k0, ldl, B + k0, ldb, B, ldb, sc)));
        }
    }
    return SPARC_GPU_SUCCESS;
}

}  // namespace

extern "C" int sparc_gpu_eigensolve(sparc_gpu_ctx *ctx, int64_t n64, const double *Hs, const double *Ms, double *Z, double *D,
                                    int32_t *info, void *ws, void *stream)
{
    if (!ctx || n64 < 0) return SPARC_GPU_INVALID_ARG;
    if (n64 == 0) return SPARC_GPU_SUCCESS;
    if (n64 > 12800) return SPARC_GPU_UNSUPPORTED;      // a column pair (2 n doubles) must fit 200 KB of shared memory
    if (!Hs || !Ms || !Z || !D || !ws) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    cudaStream_t st = (cudaStream_t)stream;
    const int n = (int)n64;
    WsLayout Lw;
    SPARC_TRY(ws_layout(ctx, SPARC_GPU_OP_EIGENSOLVE, n, 0, &Lw));
    SPARC_TRY(ws_check(ctx, Lw));
    const int64_t ld = Lw.ldw;
    double *B1 = (double *)ws, *B2 = B1 + ld * ld, *B3 = B2 + ld * ld, *B4 = B3 + ld * ld;
    double *mu = B4 + ld * ld;                          // [ld]
    int *rank = (int *)(mu + ld);                       // [ld] ints
    EigScalars *sc = (EigScalars *)(mu + 2 * ld);

    EIG_LAUNCH(0, (init_scalars_kernel<<<1, 1, 0, st>>>(sc)));
    // E1: B1 = L
    SPARC_CUDA_TRY(cudaMemcpy2DAsync(B1, (size_t)ld * 8, Ms, (size_t)n * 8, (size_t)n * 8, (size_t)n, cudaMemcpyDeviceToDevice, st));
    SPARC_TRY(potrf_lower(ctx, n, B1, ld, sc, st));
    // E2: B2 = L^-1 Hs; B3 = B2^T; B3 = L^-1 B3 = A; B2 = sym(B3)
    SPARC_CUDA_TRY(cudaMemcpy2DAsync(B2, (size_t)ld * 8, Hs, (size_t)n * 8, (size_t)n * 8, (size_t)n, cudaMemcpyDeviceToDevice, st));
    SPARC_TRY(trsm_lower_fwd(ctx, n, n, B1, ld, B2, ld, sc, st));
    dim3 tg((n + 31) / 32, (n + 31) / 32);
    EIG_LAUNCH(0, (transpose_kernel<false><<<tg, 256, 0, st>>>(n, B2, ld, B3, ld)));
    SPARC_TRY(trsm_lower_fwd(ctx, n, n, B1, ld, B3, ld, sc, st));
    EIG_LAUNCH(0, (symmetrize_kernel<<<n, 256, 0, st>>>(n, B3, ld, B2, ld, sc)));
    // E3: B3 <- A (kept for the Rayleigh quotients), B2 <- R = chol(A + sigma I), B4 = G = R^T.  The product of the rotations is
    // not accumulated (that would double the traffic of every round): G_final = G_0 V with G_0 = R^T, so V = R^-T G_final by one
    // blocked back substitution at the end.
    SPARC_CUDA_TRY(cudaMemcpyAsync(B3, B2, (size_t)ld * n * 8, cudaMemcpyDeviceToDevice, st));
    EIG_LAUNCH(0, (set_shift_kernel<<<(n + 255) / 256, 256, 0, st>>>(n, B2, ld, sc)));
    SPARC_TRY(potrf_lower(ctx, n, B2, ld, sc, st));
    EIG_LAUNCH(0, (transpose_kernel<true><<<tg, 256, 0, st>>>(n, B2, ld, B4, ld)));
    double *G = B4, *R = B2, *A = B3;
    {
        const int npad = n + (n & 1);
        const double tol = 2.3e-16 * sqrt((double)n) * 2.0;
        const size_t smem = (size_t)2 * n * sizeof(double);
        if (smem > 48 * 1024 && !(ctx->func_attr_done & (1ull << 40))) {
            SPARC_CUDA_TRY(cudaFuncSetAttribute(jacobi_round_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
            ctx->func_attr_done |= 1ull << 40;
        }
        if (smem > 48 * 1024 && !(ctx->func_attr_done & (1ull << 41))) {
            SPARC_CUDA_TRY(cudaFuncSetAttribute(jacobi_sweep_coop_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
            ctx->func_attr_done |= 1ull << 41;
        }
        // cooperative sweeps when the device supports them and at least one CTA per SM fits
        int coop = 0, occ = 0;
        if (ctx->opt_eig_coop && cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ctx->device) == cudaSuccess && coop &&
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, jacobi_sweep_coop_kernel, 256, smem) == cudaSuccess && occ >= 1) {
            const int grid = std::min(npad / 2, occ * ctx->sm_count);
            for (int sweep = 0; sweep < MAX_SWEEPS && n > 1; ++sweep) {
                int nn = n, np_ = npad, last = sweep == MAX_SWEEPS - 1;
                int64_t ldl = ld;
                double tl = tol;
                void *args[] = {&nn, &np_, &G, &ldl, &tl, &last, &sc};
                prof_begin(ctx, KK_EIG, st);
                SPARC_CUDA_TRY(cudaLaunchCooperativeKernel((const void *)jacobi_sweep_coop_kernel, dim3(grid), dim3(256), args, smem, st));
                prof_end(ctx, KK_EIG, st);
            }
        } else if (n > 1) {
            (void)cudaGetLastError();
            for (int sweep = 0; sweep < MAX_SWEEPS; ++sweep) {
                for (int r = 0; r < npad - 1; ++r)
                    EIG_LAUNCH(0, (jacobi_round_kernel<<<npad / 2, 256, smem, st>>>(n, npad, r, G, ld, nullptr, ld, tol, sc)));
                EIG_LAUNCH(0, (sweep_end_kernel<<<1, 1, 0, st>>>(tol, sweep == MAX_SWEEPS - 1, sc)));
            }
        }
    }
    SPARC_TRY(trsm_lower_trans_bwd(ctx, n, n, R, ld, G, ld, sc, st));          // G <- V = R^-T G
    double *V = G, *W = B2;                                                      // R is no longer needed: W = scratch
    // E4: mu = diag(V^T A V) with W = -(A V) through the subtracting kernel (the sign is undone in the quotient)
    SPARC_CUDA_TRY(cudaMemsetAsync(W, 0, (size_t)ld * n * 8, st));
    {
        dim3 grid((n + 63) / 64, (n + 63) / 64);
        EIG_LAUNCH(0, (gemm_sub_kernel<false, false><<<grid, 256, 0, st>>>(n, n, n, A, ld, V, ld, W, ld, nullptr)));
    }
    EIG_LAUNCH(0, (rayleigh_kernel<<<n, 256, 0, st>>>(n, V, ld, W, ld, -1.0, mu)));
    EIG_LAUNCH(0, (rank_kernel<<<(n + 255) / 256, 256, 0, st>>>(n, mu, rank, D)));
    EIG_LAUNCH(0, (permute_cols_kernel<<<dim3((n + 255) / 256 > 8 ? 8 : (n + 255) / 256, n), 256, 0, st>>>(n, V, ld, rank, W, ld)));
    SPARC_TRY(trsm_lower_trans_bwd(ctx, n, n, B1, ld, W, ld, sc, st));
    SPARC_CUDA_TRY(cudaMemcpy2DAsync(Z, (size_t)n * 8, W, (size_t)ld * 8, (size_t)n * 8, (size_t)n, cudaMemcpyDeviceToDevice, st));
    if (info) SPARC_CUDA_TRY(cudaMemcpyAsync(info, &sc->status, 2 * sizeof(int), cudaMemcpyDeviceToDevice, st));
    return SPARC_GPU_SUCCESS;
}
