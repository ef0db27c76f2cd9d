// stencil_generic.cu -- general-shape fused local pass:  Out = alpha (H_loc X + shift X) + beta Prev,
// H_loc = -1/2 Laplacian + Veff (3*n0+1 taps).
// Any grid size, any FD radius 1..6, periodic / Dirichlet per axis.  One thread per output point, neighbours
// read through L1/L2 (no tiling): this is the shape-agnostic path (odd sizes, tiny grids); the tuned path
// for the benchmark shapes is stencil_tma.cu.
#include "internal.h"

namespace {

struct GenericParams {
    StencilCoef coef;      // already multiplied by alpha
    double alpha, shift, beta;
    int nx, ny, nz, radius;
    int bcx, bcy, bcz;
};

__device__ __forceinline__ int wrap_or_neg(int q, int n, int bc)
{
    if (bc == 0) {
        if (q < 0) q += n;
        else if (q >= n) q -= n;
        return q;
    }
    return (q < 0 || q >= n) ? -1 : q;
}

__global__ void __launch_bounds__(256)
stencil_generic_kernel(GenericParams P, const double *__restrict__ veff, const double *__restrict__ X,
                       int64_t ldx, double *Out, int64_t ldo, const double *Prev, int64_t ldp)
{
    const int64_t nd = (int64_t)P.nx * P.ny * P.nz;
    const double *x = X + (int64_t)blockIdx.y * ldx;
    double *o = Out + (int64_t)blockIdx.y * ldo;
    const double *pv = Prev ? Prev + (int64_t)blockIdx.y * ldp : nullptr;
    const int64_t plane = (int64_t)P.nx * P.ny;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nd; i += (int64_t)gridDim.x * blockDim.x) {
        const int ix = (int)(i % P.nx);
        const int iy = (int)((i / P.nx) % P.ny);
        const int iz = (int)(i / plane);
        const double v = x[i];
        double acc = (P.coef.c0 + P.alpha * (veff[i] + P.shift)) * v;
        for (int p = 1; p <= P.radius; ++p) {
            double s = 0.0;
            int q = wrap_or_neg(ix - p, P.nx, P.bcx);
            if (q >= 0) s += x[i + (q - ix)];
            q = wrap_or_neg(ix + p, P.nx, P.bcx);
            if (q >= 0) s += x[i + (q - ix)];
            acc = fma(P.coef.cx[p], s, acc);
            s = 0.0;
            q = wrap_or_neg(iy - p, P.ny, P.bcy);
            if (q >= 0) s += x[i + (int64_t)(q - iy) * P.nx];
            q = wrap_or_neg(iy + p, P.ny, P.bcy);
            if (q >= 0) s += x[i + (int64_t)(q - iy) * P.nx];
            acc = fma(P.coef.cy[p], s, acc);
            s = 0.0;
            q = wrap_or_neg(iz - p, P.nz, P.bcz);
            if (q >= 0) s += x[i + (int64_t)(q - iz) * plane];
            q = wrap_or_neg(iz + p, P.nz, P.bcz);
            if (q >= 0) s += x[i + (int64_t)(q - iz) * plane];
            acc = fma(P.coef.cz[p], s, acc);
        }
        if (pv) acc = fma(P.beta, pv[i], acc);
        o[i] = acc;
    }
}

__global__ void __launch_bounds__(256)
copy_2d_kernel(double *dst, int64_t ldd, const double *__restrict__ src, int64_t lds, int64_t rows, int64_t cols)
{
    const int64_t total = rows * cols;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = k % rows, cidx = k / rows;
        dst[r + cidx * ldd] = src[r + cidx * lds];
    }
}

}  // namespace

int launch_stencil_generic(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, double *Out, int64_t ldo,
                           const double *Prev, int64_t ldp, int64_t ncols, double alpha, double shift,
                           double beta, cudaStream_t st)
{
    GenericParams P;
    for (int p = 0; p <= SPARC_MAX_RADIUS; ++p) {
        P.coef.cx[p] = alpha * ctx->coef.cx[p];
        P.coef.cy[p] = alpha * ctx->coef.cy[p];
        P.coef.cz[p] = alpha * ctx->coef.cz[p];
    }
    P.coef.c0 = alpha * ctx->coef.c0;
    P.alpha = alpha; P.shift = shift; P.beta = beta;
    P.nx = ctx->n[0]; P.ny = ctx->n[1]; P.nz = ctx->n[2]; P.radius = ctx->radius;
    P.bcx = ctx->bc[0]; P.bcy = ctx->bc[1]; P.bcz = ctx->bc[2];
    const int64_t max_cols = 65535;
    for (int64_t j0 = 0; j0 < ncols; j0 += max_cols) {
        const int64_t nb = ncols - j0 < max_cols ? ncols - j0 : max_cols;
        int64_t bx = (ctx->nd + 255) / 256;
        if (bx > 4096) bx = 4096;
        dim3 grid((unsigned)bx, (unsigned)nb);
        prof_begin(ctx, KK_STENCIL_GENERIC, st);
        stencil_generic_kernel<<<grid, 256, 0, st>>>(P, ctx->d_veff, X + j0 * ldx, ldx, Out + j0 * ldo, ldo,
                                                     (beta != 0.0 && Prev) ? Prev + j0 * ldp : nullptr, ldp);
        prof_end(ctx, KK_STENCIL_GENERIC, st);
    }
    SPARC_CUDA_TRY(cudaGetLastError());
    return SPARC_GPU_SUCCESS;
}

int launch_copy_2d(sparc_gpu_ctx *ctx, double *dst, int64_t ldd, const double *src, int64_t lds, int64_t rows,
                   int64_t cols, cudaStream_t st)
{
    if (rows <= 0 || cols <= 0) return SPARC_GPU_SUCCESS;
    int64_t blocks = (rows * cols + 255) / 256;
    if (blocks > (int64_t)ctx->sm_count * 32) blocks = (int64_t)ctx->sm_count * 32;
    prof_begin(ctx, KK_COPY2D, st);
    copy_2d_kernel<<<(unsigned)blocks, 256, 0, st>>>(dst, ldd, src, lds, rows, cols);
    prof_end(ctx, KK_COPY2D, st);
    SPARC_CUDA_TRY(cudaGetLastError());
    return SPARC_GPU_SUCCESS;
}
