// gradient.cu -- SURVEY.md section 8(f) NEXT-3: the kernels of the nonlocal Hellmann-Feynman force (PAPER.md:110, 188:
// "stencil operations and nonlocal projector multiplications ... the application of the gradient operator on the
// Kohn-Sham orbitals").
//
//   Y = D_a X        central first-derivative stencil of order n0 along one axis (radius n0/2, weights
//                    w_p = (-1)^{p+1} (n!)^2 / (p (n-p)! (n+p)!), reading R21), periodic wrap or zero outside a Dirichlet face
//   W = chi^T X      the projector contraction without Gamma (nonlocal.cu: nl_project_kernel with gamma = NULL)
//   F[J, a] = -2 sum_n g_n sum_q gamma_Jq (chi_Jq^T psi_n)(chi_Jq^T D_a psi_n)      (reading R22)
//
// The stencil is a 1-D, 2r-tap pass: 16 algorithmic bytes per point (one read, one write).  A thread owns U consecutive
// outputs ALONG the axis and keeps the U + 2r inputs they need in registers, so that every input is fetched U + 2r times per
// U outputs from L1 (1.75x at U = 16), once from DRAM.  Threads are laid out with x fastest (axis y, z) or with the
// x chunks fastest (axis x) so that the global loads and stores of a warp are contiguous runs.
#include <algorithm>

#include "internal.h"

namespace {

struct GradParams {
    double c[SPARC_MAX_RADIUS + 1];   // w_p / h_axis
    int n[3];
    int radius, bc;                   // boundary flag of the differentiated axis
};

template <int AXIS, int U, bool VEC>
__global__ void __launch_bounds__(256)
gradient_kernel(const GradParams P, const double *__restrict__ X, int64_t ldx, double *__restrict__ Y, int64_t ldy)
{
    constexpr int R = SPARC_MAX_RADIUS;
    const int nx = P.n[0], ny = P.n[1], nz = P.n[2];
    const int na = P.n[AXIS];
    const int nchunk = (na + U - 1) / U;
    // item -> (chunk along the axis, the two other coordinates); the fastest-varying item index is contiguous in memory
    const int64_t items = (int64_t)nchunk * (AXIS == 0 ? (int64_t)ny * nz : AXIS == 1 ? (int64_t)nx * nz : (int64_t)nx * ny);
    const int64_t it = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (it >= items) return;
    int a0;
    int64_t base, stride;
    if (AXIS == 0) {
        const int ch = (int)(it % nchunk);
        const int64_t row = it / nchunk;              // y + ny z
        a0 = ch * U; base = row * nx; stride = 1;
    } else if (AXIS == 1) {
        const int x = (int)(it % nx);
        const int64_t r = it / nx;
        const int ch = (int)(r % nchunk), z = (int)(r / nchunk);
        a0 = ch * U; base = x + (int64_t)nx * ny * z; stride = nx;
    } else {
        const int x = (int)(it % nx);
        const int64_t r = it / nx;
        const int y = (int)(r % ny), ch = (int)(r / ny);
        a0 = ch * U; base = x + (int64_t)nx * y; stride = (int64_t)nx * ny;
    }
    const double *x = X + (int64_t)blockIdx.y * ldx + base;
    double *y = Y + (int64_t)blockIdx.y * ldy + base;
    const int r = P.radius;

    double v[U + 2 * R];
    // x axis, even n_x, 16-byte aligned columns: the window starts at the even index a0 - 6, so (even, odd) pairs never
    // straddle the periodic wrap or a Dirichlet face: 16-byte loads (half the L1 wavefronts of the 8-byte ones)
    if (AXIS == 0 && VEC) {
#pragma unroll
        for (int k = 0; k < U + 2 * R; k += 2) {
            v[k] = v[k + 1] = 0.0;
            if (k + 1 >= R - r && k < U + R + r) {
                int q = a0 - R + k;
                bool ok = true;
                if (P.bc == 0) { q %= na; if (q < 0) q += na; }
                else ok = q >= 0 && q < na;
                if (ok) { const double2 t = *reinterpret_cast<const double2 *>(x + q); v[k] = t.x; v[k + 1] = t.y; }
            }
        }
    } else
#pragma unroll
    for (int k = 0; k < U + 2 * R; ++k) {
        v[k] = 0.0;
        if (k >= R - r && k < U + R + r) {
            int q = a0 - R + k;
            bool ok = true;
            if (P.bc == 0) { q %= na; if (q < 0) q += na; }
            else ok = q >= 0 && q < na;
            // outputs past the end of a ragged last chunk are never stored; their inputs need not exist
            if (ok && (P.bc == 0 || q < na)) v[k] = x[(int64_t)q * stride];
        }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
        if (a0 + u < na) {
            double s = 0.0;
#pragma unroll
            for (int p = 1; p <= R; ++p) s = fma(P.c[p], v[u + R + p] - v[u + R - p], s);
            y[(int64_t)(a0 + u) * stride] = s;
        }
    }
}

// F[3 J + a] += -2 sum_{n < ncols} occ[n] sum_q gamma[po_J + q] W[po_J + q, n] G[po_J + q, n]; one CTA per atom, fixed
// reduction tree (bitwise reproducible); the column blocks of a force call arrive in stream order.
__global__ void __launch_bounds__(128)
force_contract_kernel(const int32_t *__restrict__ n_proj, const int32_t *__restrict__ proj_ofs, const double *__restrict__ gamma,
                      const double *__restrict__ W, const double *__restrict__ G, int ldw, const double *__restrict__ occ,
                      int64_t ncols, int axis, double *F)
{
    __shared__ double red[128];
    const int J = blockIdx.x, P = n_proj[J], po = proj_ofs[J];
    double s = 0.0;
    for (int64_t n = threadIdx.x; n < ncols; n += blockDim.x) {
        double t = 0.0;
        for (int q = 0; q < P; ++q) t = fma(gamma[po + q] * W[po + q + n * ldw], G[po + q + n * ldw], t);
        s = fma(occ[n], t, s);
    }
    red[threadIdx.x] = s;
    __syncthreads();
    for (int o = 64; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) F[3 * J + axis] += -2.0 * red[0];
}

int launch_gradient(sparc_gpu_ctx *ctx, int axis, const double *X, int64_t ldx, double *Y, int64_t ldy, int64_t ncols,
                    cudaStream_t st)
{
    GradParams P;
    for (int p = 0; p <= SPARC_MAX_RADIUS; ++p) P.c[p] = p <= ctx->radius ? ctx->w1[p] / ctx->h[axis] : 0.0;
    P.n[0] = ctx->n[0]; P.n[1] = ctx->n[1]; P.n[2] = ctx->n[2];
    P.radius = ctx->radius; P.bc = ctx->bc[axis];
    constexpr int UX = 4, UYZ = 16;
    const int na = ctx->n[axis];
    const int U = axis == 0 ? UX : UYZ;
    const int64_t items = (int64_t)((na + U - 1) / U) * (ctx->nd / na);
    const int64_t bx = (items + 255) / 256;
    if (bx >= (int64_t)INT32_MAX) return SPARC_GPU_UNSUPPORTED;
    for (int64_t j0 = 0; j0 < ncols; j0 += 65535) {
        const int64_t nb = std::min<int64_t>(ncols - j0, 65535);
        dim3 grid((unsigned)bx, (unsigned)nb);
        prof_begin(ctx, KK_GRADIENT, st);
        const bool vec = (ctx->n[0] % 2 == 0) && (ldx % 2 == 0) && (((uintptr_t)X & 15) == 0);
        if (axis == 0 && vec) gradient_kernel<0, UX, true><<<grid, 256, 0, st>>>(P, X + j0 * ldx, ldx, Y + j0 * ldy, ldy);
        else if (axis == 0) gradient_kernel<0, UX, false><<<grid, 256, 0, st>>>(P, X + j0 * ldx, ldx, Y + j0 * ldy, ldy);
        else if (axis == 1) gradient_kernel<1, UYZ, false><<<grid, 256, 0, st>>>(P, X + j0 * ldx, ldx, Y + j0 * ldy, ldy);
        else gradient_kernel<2, UYZ, false><<<grid, 256, 0, st>>>(P, X + j0 * ldx, ldx, Y + j0 * ldy, ldy);
        prof_end(ctx, KK_GRADIENT, st);
    }
    SPARC_CUDA_TRY(cudaGetLastError());
    return SPARC_GPU_SUCCESS;
}

}  // namespace

extern "C" {

int sparc_gpu_gradient(sparc_gpu_ctx *ctx, int axis, const double *X, int64_t ldx, double *Y, int64_t ldy, int64_t ncols,
                       void *stream)
{
    if (!ctx || ncols < 0 || axis < 0 || axis > 2) return SPARC_GPU_INVALID_ARG;
    if (ncols == 0) return SPARC_GPU_SUCCESS;
    if (!X || !Y || ldx < ctx->nd || ldy < ctx->nd) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    return launch_gradient(ctx, axis, X, ldx, Y, ldy, ncols, (cudaStream_t)stream);
}

int sparc_gpu_nl_project(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, int64_t ncols, double *W, void *stream)
{
    if (!ctx || ncols < 0) return SPARC_GPU_INVALID_ARG;
    if (ncols == 0 || ctx->n_proj_total == 0) return SPARC_GPU_SUCCESS;
    if (!X || !W || ldx < ctx->nd) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    return launch_nl_project_raw(ctx, X, ldx, ncols, W, (cudaStream_t)stream);
}

int sparc_gpu_gradient_project(sparc_gpu_ctx *ctx, int axis, const double *X, int64_t ldx, int64_t ncols, double *W,
                               int64_t col_block, void *ws, void *stream)
{
    if (!ctx || ncols < 0 || axis < 0 || axis > 2) return SPARC_GPU_INVALID_ARG;
    if (ncols == 0 || ctx->n_proj_total == 0) return SPARC_GPU_SUCCESS;
    if (!X || !W || !ws || ldx < ctx->nd) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    cudaStream_t st = (cudaStream_t)stream;
    WsLayout L;
    SPARC_TRY(ws_layout(ctx, SPARC_GPU_OP_GRADIENT_PROJECT, ncols, col_block, &L));
    SPARC_TRY(ws_check(ctx, L));
    double *Y = (double *)((char *)ws + L.off_w);
    for (int64_t j0 = 0; j0 < ncols; j0 += L.block) {
        const int64_t nb = std::min(L.block, ncols - j0);
        SPARC_TRY(launch_gradient(ctx, axis, X + j0 * ldx, ldx, Y, L.ldw, nb, st));
        SPARC_TRY(launch_nl_project_raw(ctx, Y, L.ldw, nb, W + j0 * (int64_t)ctx->n_proj_total, st));
    }
    return SPARC_GPU_SUCCESS;
}

int sparc_gpu_nonlocal_force(sparc_gpu_ctx *ctx, const double *Psi, int64_t ld, int64_t ns, const double *occ, double *F,
                             int64_t col_block, void *ws, void *stream)
{
    if (!ctx || ns < 0) return SPARC_GPU_INVALID_ARG;
    if (ctx->n_atoms == 0) return SPARC_GPU_SUCCESS;
    if (!F) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    cudaStream_t st = (cudaStream_t)stream;
    SPARC_CUDA_TRY(cudaMemsetAsync(F, 0, (size_t)ctx->n_atoms * 3 * 8, st));
    if (ns == 0 || ctx->n_proj_total == 0) return SPARC_GPU_SUCCESS;
    if (!Psi || !occ || !ws || ld < ctx->nd) return SPARC_GPU_INVALID_ARG;
    WsLayout L;
    SPARC_TRY(ws_layout(ctx, SPARC_GPU_OP_NONLOCAL_FORCE, ns, col_block, &L));
    SPARC_TRY(ws_check(ctx, L));
    double *Y = (double *)((char *)ws + L.off_w);
    double *W = (double *)((char *)ws + L.off_d);
    double *G = W + (int64_t)ctx->n_proj_total * L.block;
    for (int64_t j0 = 0; j0 < ns; j0 += L.block) {
        const int64_t nb = std::min(L.block, ns - j0);
        SPARC_TRY(launch_nl_project_raw(ctx, Psi + j0 * ld, ld, nb, W, st));
        for (int a = 0; a < 3; ++a) {
            SPARC_TRY(launch_gradient(ctx, a, Psi + j0 * ld, ld, Y, L.ldw, nb, st));
            SPARC_TRY(launch_nl_project_raw(ctx, Y, L.ldw, nb, G, st));
            prof_begin(ctx, KK_GRADIENT, st);
            force_contract_kernel<<<(unsigned)ctx->n_atoms, 128, 0, st>>>(ctx->d_n_proj, ctx->d_proj_ofs, ctx->d_gamma, W, G,
                                                                          ctx->n_proj_total, occ + j0, nb, a, F);
            prof_end(ctx, KK_GRADIENT, st);
            SPARC_CUDA_TRY(cudaGetLastError());
        }
    }
    return SPARC_GPU_SUCCESS;
}

}  // extern "C"
