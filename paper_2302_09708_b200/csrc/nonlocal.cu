// nonlocal.cu -- Kleinman-Bylander nonlocal term  V_nl X = sum_J S_J^T chi_J diag(gamma_J) chi_J^T S_J X
// ("nonlocal projectors for each atom, stored as a dense matrix, are applied on the
// appropriate components of X").  Two kernels:
//   nl_project : D_J = scale * diag(gamma_J) chi_J^T X[idx_J, cols]     warp-cooperative gather + small GEMM
//   nl_pull    : Out[i, col] += sum_{(J,t) covers i} chi_J[t,:] . D_J[:, col]
// The second is the scatter written in pull (gather) form through the point -> (atom,row) inverse map
// built at create: conflict-free without atomics and bitwise reproducible (R15).
#include <algorithm>

#include "internal.h"

namespace {

constexpr int NLP_WARPS = 8;      // warps per CTA in nl_project
constexpr int NLP_COLS = 4;       // columns per warp

// grid: (n_atoms, ceil(ncols / (NLP_WARPS*NLP_COLS))).  Lanes stride over the support rows t; each lane keeps
// PMAX x NLP_COLS partial sums; a shuffle tree reduces them; lane 0 scales by gamma and writes D.
template <int PMAX>
__global__ void __launch_bounds__(NLP_WARPS * 32)
nl_project_kernel(const int64_t *__restrict__ supp_ptr, const int32_t *__restrict__ supp_idx,
                  const int32_t *__restrict__ n_proj, const int32_t *__restrict__ proj_ofs,
                  const int64_t *__restrict__ chi_ptr, const double *__restrict__ chi,
                  const double *__restrict__ gamma, const double *__restrict__ X, int64_t ldx, int64_t ncols,
                  double scale, double *__restrict__ D, int ldD)
{
    const int J = blockIdx.x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t col0 = ((int64_t)blockIdx.y * NLP_WARPS + warp) * NLP_COLS;
    if (col0 >= ncols) return;
    const int P = n_proj[J];
    if (P == 0) return;
    const int64_t s0 = supp_ptr[J];
    const int nJ = (int)(supp_ptr[J + 1] - s0);
    const int32_t *idx = supp_idx + s0;
    const double *ch = chi + chi_ptr[J];
    const double *xc[NLP_COLS];
#pragma unroll
    for (int c = 0; c < NLP_COLS; ++c) xc[c] = X + (col0 + c < ncols ? col0 + c : col0) * ldx;

    double acc[PMAX][NLP_COLS];
#pragma unroll
    for (int q = 0; q < PMAX; ++q)
#pragma unroll
        for (int c = 0; c < NLP_COLS; ++c) acc[q][c] = 0.0;

    for (int t = lane; t < nJ; t += 32) {
        const int i = idx[t];
        double g[NLP_COLS];
#pragma unroll
        for (int c = 0; c < NLP_COLS; ++c) g[c] = xc[c][i];
#pragma unroll
        for (int q = 0; q < PMAX; ++q) {
            if (q < P) {
                const double cv = ch[t + (int64_t)q * nJ];
#pragma unroll
                for (int c = 0; c < NLP_COLS; ++c) acc[q][c] = fma(cv, g[c], acc[q][c]);
            }
        }
    }
    const int po = proj_ofs[J];
#pragma unroll
    for (int q = 0; q < PMAX; ++q) {
        if (q < P) {
#pragma unroll
            for (int c = 0; c < NLP_COLS; ++c) {
                double v = acc[q][c];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                if (lane == 0 && col0 + c < ncols) D[(int64_t)(po + q) + (col0 + c) * (int64_t)ldD] = gamma ? scale * gamma[po + q] * v : v;
            }
        }
    }
}

// grid: (ceil(n_covered/128), column chunks).  One thread per covered point, looping over the columns of
// its chunk: consecutive covered points are mostly consecutive grid indices -> coalesced read-modify-write.
__global__ void __launch_bounds__(128)
nl_pull_kernel(const int32_t *__restrict__ cov_idx, const int64_t *__restrict__ cov_ptr,
               const CoverEntry *__restrict__ ent, const double *__restrict__ chi, const double *__restrict__ D,
               int ldD, double *Out, int64_t ldo, int64_t n_covered, int64_t ncols, int cols_per_block)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_covered) return;
    const int i = cov_idx[k];
    const int64_t e0 = cov_ptr[k], e1 = cov_ptr[k + 1];
    const int64_t c0 = (int64_t)blockIdx.y * cols_per_block;
    const int64_t c1 = c0 + cols_per_block < ncols ? c0 + cols_per_block : ncols;
    for (int64_t col = c0; col < c1; ++col) {
        const double *d = D + col * (int64_t)ldD;
        double s = 0.0;
        for (int64_t e = e0; e < e1; ++e) {
            const CoverEntry en = ent[e];
            const int P = en.pofs_p & 0xff;
            const double *dj = d + (en.pofs_p >> 8);
            const double *ch = chi + en.chi_off;
            for (int q = 0; q < P; ++q) s = fma(ch[(int64_t)q * en.n_j], dj[q], s);
        }
        Out[i + col * ldo] += s;
    }
}


// ---- fused per-atom kernel (default path) ---------------------------------------------------------------------
// One CTA = one atom J x NLF_WARPS*NCW columns.  The chi_J rows and support indices are streamed through a
// double-buffered shared-memory tile (cp.async) that all warps of the CTA share; each warp owns NCW columns.
//   pass 1 (gather + small GEMM): lanes stride over the support rows t, gather X[idx[t], col] (coalesced along the
//           x-runs of the support) and accumulate C[q][c] += chi[t][q] X[idx[t]][c] in registers; a butterfly
//           all-reduce leaves D[q][c] = scale * gamma[q] * C[q][c] in every lane.
//   pass 2 (small GEMM + scatter): the tile stream is replayed (chi_J comes from L2) and each lane adds
//           sum_q chi[t][q] D[q][c] to Out[idx[t]][c] with an FP64 atomic add (RED): supports of different atoms
//           overlap, the atomics make the scatter conflict-free (north_star: "coloured or atomic").
constexpr int NLF_WARPS = 8;

__device__ __forceinline__ void cp_async8(void *smem, const void *gmem, int src_bytes)
{
    unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(sa), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async4(void *smem, const void *gmem, int src_bytes)
{
    unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;\n" ::"r"(sa), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::); }

template <int PMAX, int NCW, int NLF_TILE>      // NLF_TILE: support rows per shared-memory tile
__global__ void __launch_bounds__(NLF_WARPS * 32)
nl_fused_kernel(const int64_t *__restrict__ supp_ptr, const int32_t *__restrict__ supp_idx,
                const int32_t *__restrict__ n_proj, const int32_t *__restrict__ proj_ofs,
                const int64_t *__restrict__ chi_ptr, const double *__restrict__ chi,
                const double *__restrict__ gamma, const double *__restrict__ X, int64_t ldx, double *Out, int64_t ldo,
                int64_t ncols, double scale)
{
    __shared__ __align__(16) double chi_s[2][PMAX][NLF_TILE];
    __shared__ int32_t idx_s[2][NLF_TILE];
    const int J = blockIdx.x;
    const int P = n_proj[J];
    const int64_t s0 = supp_ptr[J];
    const int nJ = (int)(supp_ptr[J + 1] - s0);
    if (P == 0 || nJ == 0) return;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int64_t col0 = ((int64_t)blockIdx.y * NLF_WARPS + warp) * NCW;
    const bool warp_active = col0 < ncols;          // inactive warps still help loading tiles
    const int32_t *idx = supp_idx + s0;
    const double *ch = chi + chi_ptr[J];
    const int ntiles = (nJ + NLF_TILE - 1) / NLF_TILE;

    auto load_tile = [&](int tile, int buf) {
        const int t0 = tile * NLF_TILE;
        for (int k = tid; k < NLF_TILE; k += NLF_WARPS * 32) {
            const int t = t0 + k;
            const bool ok = t < nJ;
            cp_async4(&idx_s[buf][k], ok ? idx + t : idx, ok ? 4 : 0);
#pragma unroll
            for (int q = 0; q < PMAX; ++q)
                if (q < P) cp_async8(&chi_s[buf][q][k], ok ? ch + t + (int64_t)q * nJ : ch, ok ? 8 : 0);
        }
        cp_async_commit();
    };

    const double *xc[NCW];
    double *oc[NCW];
#pragma unroll
    for (int c = 0; c < NCW; ++c) {
        const int64_t col = (col0 + c < ncols) ? col0 + c : (warp_active ? col0 : 0);
        xc[c] = X + col * ldx;
        oc[c] = Out + col * ldo;
    }

    double acc[PMAX][NCW];
#pragma unroll
    for (int q = 0; q < PMAX; ++q)
#pragma unroll
        for (int c = 0; c < NCW; ++c) acc[q][c] = 0.0;

    // ---- pass 1: C = chi^T X[idx] -----------------------------------------------------------------------------
    load_tile(0, 0);
    for (int tile = 0; tile < ntiles; ++tile) {
        const int buf = tile & 1;
        cp_async_wait_all();
        __syncthreads();
        if (tile + 1 < ntiles) load_tile(tile + 1, buf ^ 1);
        if (warp_active) {
#pragma unroll 2
            for (int k = lane; k < NLF_TILE; k += 32) {
                const int i = idx_s[buf][k];          // rows beyond n_J: index 0 with chi = 0
                double g[NCW];
#pragma unroll
                for (int c = 0; c < NCW; ++c) g[c] = __ldg(xc[c] + i);
#pragma unroll
                for (int q = 0; q < PMAX; ++q) {
                    if (q < P) {
                        const double cv = chi_s[buf][q][k];
#pragma unroll
                        for (int c = 0; c < NCW; ++c) acc[q][c] = fma(cv, g[c], acc[q][c]);
                    }
                }
            }
        }
    }
    // butterfly all-reduce: every lane ends with D[q][c] = scale * gamma[q] * sum_t
    const int po = proj_ofs[J];
#pragma unroll
    for (int q = 0; q < PMAX; ++q) {
        if (q < P) {
            const double gq = scale * gamma[po + q];
#pragma unroll
            for (int c = 0; c < NCW; ++c) {
                double v = acc[q][c];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                acc[q][c] = gq * v;
            }
        }
    }
    // ---- pass 2: Out[idx] += chi D ------------------------------------------------------------------------------
    __syncthreads();
    load_tile(0, 0);
    for (int tile = 0; tile < ntiles; ++tile) {
        const int buf = tile & 1;
        cp_async_wait_all();
        __syncthreads();
        if (tile + 1 < ntiles) load_tile(tile + 1, buf ^ 1);
        if (warp_active) {
            const int t0 = tile * NLF_TILE;
#pragma unroll 2
            for (int k = lane; k < NLF_TILE; k += 32) {
                if (t0 + k < nJ) {
                    const int i = idx_s[buf][k];
                    double v[NCW];
#pragma unroll
                    for (int c = 0; c < NCW; ++c) v[c] = 0.0;
#pragma unroll
                    for (int q = 0; q < PMAX; ++q) {
                        if (q < P) {
                            const double cv = chi_s[buf][q][k];
#pragma unroll
                            for (int c = 0; c < NCW; ++c) v[c] = fma(cv, acc[q][c], v[c]);
                        }
                    }
#pragma unroll
                    for (int c = 0; c < NCW; ++c)
                        if (col0 + c < ncols) atomicAdd(oc[c] + i, v[c]);
                }
            }
        }
    }
}

}  // namespace

static int nl_project_impl(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, int64_t ncols, double scale, const double *gamma,
                           double *D, cudaStream_t st)
{
    const int cols_per_cta = NLP_WARPS * NLP_COLS;
    const int64_t max_y = 65535;
    for (int64_t j0 = 0; j0 < ncols; j0 += max_y * cols_per_cta) {
        const int64_t nb = std::min<int64_t>(ncols - j0, max_y * cols_per_cta);
        dim3 grid((unsigned)ctx->n_atoms, (unsigned)((nb + cols_per_cta - 1) / cols_per_cta));
        const double *Xb = X + j0 * ldx;
        double *Db = D + j0 * (int64_t)ctx->n_proj_total;
#define NLP_LAUNCH(PM)                                                                                         \
        nl_project_kernel<PM><<<grid, NLP_WARPS * 32, 0, st>>>(ctx->d_supp_ptr, ctx->d_supp_idx, ctx->d_n_proj, \
            ctx->d_proj_ofs, ctx->d_chi_ptr, ctx->d_chi, gamma, Xb, ldx, nb, scale, Db, ctx->n_proj_total)
        prof_begin(ctx, KK_NL_PROJECT, st);
        if (ctx->max_proj <= 4) NLP_LAUNCH(4);
        else if (ctx->max_proj <= 9) NLP_LAUNCH(9);
        else NLP_LAUNCH(16);
#undef NLP_LAUNCH
        prof_end(ctx, KK_NL_PROJECT, st);
    }
    SPARC_CUDA_TRY(cudaGetLastError());
    return SPARC_GPU_SUCCESS;
}

int launch_nl_project(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, int64_t ncols, double scale, double *D,
                      cudaStream_t st)
{
    return nl_project_impl(ctx, X, ldx, ncols, scale, ctx->d_gamma, D, st);
}

// W = chi^T X (no Gamma): the projector contraction of the force (gradient.cu)
int launch_nl_project_raw(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, int64_t ncols, double *W, cudaStream_t st)
{
    return nl_project_impl(ctx, X, ldx, ncols, 1.0, nullptr, W, st);
}

int launch_nl_pull(sparc_gpu_ctx *ctx, const double *D, double *Out, int64_t ldo, int64_t ncols, cudaStream_t st)
{
    if (ctx->n_covered == 0) return SPARC_GPU_SUCCESS;
    const int64_t bx = (ctx->n_covered + 127) / 128;
    // enough CTAs to fill the chip, but keep the (entry, chi) re-reads per thread amortised over columns
    int cols_per_block = 16;
    int64_t by = (ncols + cols_per_block - 1) / cols_per_block;
    while (by > 65535) { cols_per_block *= 2; by = (ncols + cols_per_block - 1) / cols_per_block; }
    dim3 grid((unsigned)bx, (unsigned)by);
    prof_begin(ctx, KK_NL_PULL, st);
    nl_pull_kernel<<<grid, 128, 0, st>>>(ctx->d_cov_idx, ctx->d_cov_ptr, ctx->d_cov_ent, ctx->d_chi, D,
                                         ctx->n_proj_total, Out, ldo, ctx->n_covered, ncols, cols_per_block);
    prof_end(ctx, KK_NL_PULL, st);
    SPARC_CUDA_TRY(cudaGetLastError());
    return SPARC_GPU_SUCCESS;
}

int launch_nl_fused(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, double *Out, int64_t ldo, int64_t ncols,
                    double scale, cudaStream_t st)
{
    const int ncw = ctx->max_proj <= 9 ? 4 : 2;
    const int cols_per_cta = NLF_WARPS * ncw;
    const int64_t max_y = 65535;
    for (int64_t j0 = 0; j0 < ncols; j0 += max_y * cols_per_cta) {
        const int64_t nb = std::min<int64_t>(ncols - j0, max_y * cols_per_cta);
        dim3 grid((unsigned)ctx->n_atoms, (unsigned)((nb + cols_per_cta - 1) / cols_per_cta));
#define NLF_LAUNCH(PM, NC, TL)                                                                                       \
        nl_fused_kernel<PM, NC, TL><<<grid, NLF_WARPS * 32, 0, st>>>(ctx->d_supp_ptr, ctx->d_supp_idx, ctx->d_n_proj,  \
            ctx->d_proj_ofs, ctx->d_chi_ptr, ctx->d_chi, ctx->d_gamma, X + j0 * ldx, ldx, Out + j0 * ldo, ldo, nb, scale)
        prof_begin(ctx, KK_NL_FUSED, st);
        if (ctx->max_proj <= 4) NLF_LAUNCH(4, 4, 256);
        else if (ctx->max_proj <= 9) NLF_LAUNCH(9, 4, 256);
        else NLF_LAUNCH(16, 2, 128);
#undef NLF_LAUNCH
        prof_end(ctx, KK_NL_FUSED, st);
    }
    SPARC_CUDA_TRY(cudaGetLastError());
    return SPARC_GPU_SUCCESS;
}
