// kpoint.cu -- SURVEY.md section 8(f) NEXT-4: the complex (k-point) variant of the hot path ("complex-valued
// ... Bloch wavevectors", 126 / 146 / 166 the Zgemm forms, 176 Monkhorst-Pack grids).  Readings R24-R27:
//   * orbitals obey psi(r + L_a e_a) = exp(i theta_a) psi(r) on a periodic axis, theta_a = k_a L_a: a stencil tap that leaves
//     the cell through the upper face of axis a reads the wrapped point times exp(+i theta_a), through the lower face times
//     exp(-i theta_a); Dirichlet axes carry no phase;
//   * projector tables chi are real; a support row folded into the cell by the image shift w (per axis -1, 0, +1) acts as
//     chi~[t, q] = chi[t, q] exp(-i phi_t), phi_t = sum_a w_a[t] theta_a, and V_nl = sum_J chi~_J Gamma_J chi~_J^H;
//   * Hs = Psi^H H Psi and Ms = Psi^H Psi are Hermitian, the rotation is Psi Q with complex Q.
// Complex numbers are interleaved (re, im) doubles; a complex N_d x ncols block has its leading dimension counted in
// complex elements.
//
// Kernels.  The local pass is a one-thread-per-point complex stencil (any shape, 32 algorithmic bytes per point); the
// nonlocal term is the deterministic project + pull pair with the per-row phases.  The subspace products reuse the real
// FP64 tensor-core GEMMs of gemm.cu on the REAL VIEW of the interleaved arrays (a complex column of N_d entries is a real
// column of 2 N_d entries):
//   Re(A^H B) = view(A)^T view(B),   Im(A^H B) = view(A)^T view(-i B),   view(Psi Q) = [view(Psi) | view(i Psi)] [Re Q; Im Q],
// i.e. 4 real multiply-adds per complex one -- exactly the arithmetic of a complex GEMM, at the DMMA rate.
#include <math.h>

#include <algorithm>
#include <vector>

#include "internal.h"

namespace {

struct KStencilParams {
    StencilCoef coef;      // already multiplied by alpha
    double alpha, shift, beta;
    double ph[3][2];       // cos theta_a, sin theta_a (0 phase on Dirichlet axes)
    int n[3], radius, bc[3];
};

__device__ __forceinline__ double2 cmul(double2 a, double cr, double ci) { return make_double2(a.x * cr - a.y * ci, a.x * ci + a.y * cr); }

// Out = alpha (H_loc(k) X + shift X) + beta Prev on complex columns
__global__ void __launch_bounds__(256)
stencil_k_kernel(const KStencilParams P, const double *__restrict__ veff, const double2 *__restrict__ X, int64_t ldx,
                 double2 *Out, int64_t ldo, const double2 *Prev, int64_t ldp)
{
    const int nx = P.n[0], ny = P.n[1], nz = P.n[2];
    const int64_t nd = (int64_t)nx * ny * nz, plane = (int64_t)nx * ny;
    const double2 *x = X + (int64_t)blockIdx.y * ldx;
    double2 *o = Out + (int64_t)blockIdx.y * ldo;
    const double2 *pv = Prev ? Prev + (int64_t)blockIdx.y * ldp : nullptr;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nd; i += (int64_t)gridDim.x * blockDim.x) {
        const int c[3] = {(int)(i % nx), (int)((i / nx) % ny), (int)(i / plane)};
        const int64_t strd[3] = {1, nx, plane};
        const double2 v = x[i];
        const double d0 = P.coef.c0 + P.alpha * (veff[i] + P.shift);
        double ar = d0 * v.x, ai = d0 * v.y;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const double *cf = a == 0 ? P.coef.cx : a == 1 ? P.coef.cy : P.coef.cz;
            const int na = P.n[a];
            for (int p = 1; p <= P.radius; ++p) {
                double sr = 0.0, si = 0.0;
                int q = c[a] - p;
                if (q >= 0) { const double2 u = x[i - p * strd[a]]; sr += u.x; si += u.y; }
                else if (P.bc[a] == 0) {       // left the cell through the lower face: exp(-i theta)
                    const double2 u = cmul(x[i + (int64_t)(na - p) * strd[a]], P.ph[a][0], -P.ph[a][1]);
                    sr += u.x; si += u.y;
                }
                q = c[a] + p;
                if (q < na) { const double2 u = x[i + p * strd[a]]; sr += u.x; si += u.y; }
                else if (P.bc[a] == 0) {       // upper face: exp(+i theta)
                    const double2 u = cmul(x[i - (int64_t)(na - p) * strd[a]], P.ph[a][0], P.ph[a][1]);
                    sr += u.x; si += u.y;
                }
                ar = fma(cf[p], sr, ar); ai = fma(cf[p], si, ai);
            }
        }
        if (pv) { const double2 u = pv[i]; ar = fma(P.beta, u.x, ar); ai = fma(P.beta, u.y, ai); }
        o[i] = make_double2(ar, ai);
    }
}

constexpr int KP_WARPS = 8, KP_COLS = 2;

// D[po_J + q, col] = scale gamma_q sum_t chi[t, q] exp(+i phi_t) X[idx_t, col]      (chi~^H X, then Gamma)
template <int PMAX>
__global__ void __launch_bounds__(KP_WARPS * 32)
nl_project_k_kernel(const int64_t *__restrict__ supp_ptr, const int32_t *__restrict__ supp_idx, const int32_t *__restrict__ n_proj,
                    const int32_t *__restrict__ proj_ofs, const int64_t *__restrict__ chi_ptr, const double *__restrict__ chi,
                    const double *__restrict__ gamma, const double2 *__restrict__ phase, const double2 *__restrict__ X, int64_t ldx,
                    int64_t ncols, double scale, double2 *__restrict__ D, int ldD)
{
    const int J = blockIdx.x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t col0 = ((int64_t)blockIdx.y * KP_WARPS + warp) * KP_COLS;
    if (col0 >= ncols) return;
    const int P = n_proj[J];
    if (P == 0) return;
    const int64_t s0 = supp_ptr[J];
    const int nJ = (int)(supp_ptr[J + 1] - s0);
    const int32_t *idx = supp_idx + s0;
    const double2 *ph = phase + s0;
    const double *ch = chi + chi_ptr[J];
    const double2 *xc[KP_COLS];
#pragma unroll
    for (int c = 0; c < KP_COLS; ++c) xc[c] = X + (col0 + c < ncols ? col0 + c : col0) * ldx;
    double2 acc[PMAX][KP_COLS];
#pragma unroll
    for (int q = 0; q < PMAX; ++q)
#pragma unroll
        for (int c = 0; c < KP_COLS; ++c) acc[q][c] = make_double2(0.0, 0.0);
    for (int t = lane; t < nJ; t += 32) {
        const int i = idx[t];
        const double2 e = ph[t];
        double2 g[KP_COLS];
#pragma unroll
        for (int c = 0; c < KP_COLS; ++c) g[c] = cmul(xc[c][i], e.x, e.y);
#pragma unroll
        for (int q = 0; q < PMAX; ++q) {
            if (q < P) {
                const double cv = ch[t + (int64_t)q * nJ];
#pragma unroll
                for (int c = 0; c < KP_COLS; ++c) { acc[q][c].x = fma(cv, g[c].x, acc[q][c].x); acc[q][c].y = fma(cv, g[c].y, acc[q][c].y); }
            }
        }
    }
    const int po = proj_ofs[J];
#pragma unroll
    for (int q = 0; q < PMAX; ++q) {
        if (q < P) {
#pragma unroll
            for (int c = 0; c < KP_COLS; ++c) {
                double vr = acc[q][c].x, vi = acc[q][c].y;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) { vr += __shfl_xor_sync(0xffffffffu, vr, o); vi += __shfl_xor_sync(0xffffffffu, vi, o); }
                const double g = scale * gamma[po + q];
                if (lane == 0 && col0 + c < ncols) D[(int64_t)(po + q) + (col0 + c) * (int64_t)ldD] = make_double2(g * vr, g * vi);
            }
        }
    }
}

// Out[i, col] += sum_{(J,t) covering i} exp(-i phi_t) sum_q chi_J[t, q] D[po_J + q, col]
__global__ void __launch_bounds__(128)
nl_pull_k_kernel(const int32_t *__restrict__ cov_idx, const int64_t *__restrict__ cov_ptr, const CoverEntry *__restrict__ ent,
                 const double2 *__restrict__ cov_phase, const double *__restrict__ chi, const double2 *__restrict__ D, int ldD,
                 double2 *Out, int64_t ldo, int64_t n_covered, int64_t ncols, int cols_per_block)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_covered) return;
    const int i = cov_idx[k];
    const int64_t e0 = cov_ptr[k], e1 = cov_ptr[k + 1];
    const int64_t c0 = (int64_t)blockIdx.y * cols_per_block;
    const int64_t c1 = c0 + cols_per_block < ncols ? c0 + cols_per_block : ncols;
    for (int64_t col = c0; col < c1; ++col) {
        const double2 *d = D + col * (int64_t)ldD;
        double sr = 0.0, si = 0.0;
        for (int64_t e = e0; e < e1; ++e) {
            const CoverEntry en = ent[e];
            const int P = en.pofs_p & 0xff;
            const double2 *dj = d + (en.pofs_p >> 8);
            const double *ch = chi + en.chi_off;
            double tr = 0.0, ti = 0.0;
            for (int q = 0; q < P; ++q) { const double cv = ch[(int64_t)q * en.n_j]; tr = fma(cv, dj[q].x, tr); ti = fma(cv, dj[q].y, ti); }
            const double2 ph = cov_phase[e];            // exp(+i phi): conjugate applied here
            sr += tr * ph.x + ti * ph.y;
            si += ti * ph.x - tr * ph.y;
        }
        double2 o = Out[i + col * ldo];
        o.x += sr; o.y += si;
        Out[i + col * ldo] = o;
    }
}

// dst = -i src (MINUS_I) or +i src, elementwise on a rows x cols complex block
template <bool MINUS_I>
__global__ void __launch_bounds__(256)
rot_i_kernel(double2 *dst, int64_t ldd, const double2 *__restrict__ src, int64_t lds, int64_t rows, int64_t cols)
{
    const int64_t total = rows * cols;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = k % rows, c = k / rows;
        const double2 v = src[r + c * lds];
        dst[r + c * ldd] = MINUS_I ? make_double2(v.y, -v.x) : make_double2(-v.y, v.x);
    }
}

// C (complex m x n, ldc) = Re + i Im from two real m x n blocks (ld m)
__global__ void __launch_bounds__(256)
combine_kernel(double2 *C, int64_t ldc, const double *__restrict__ Re, const double *__restrict__ Im, int64_t m, int64_t n)
{
    const int64_t total = m * n;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = k % m, c = k / m;
        C[r + c * ldc] = make_double2(Re[k], Im[k]);
    }
}

// B2 (2 ns x ns real) = [Re Q; Im Q] from complex Q (ns x ns)
__global__ void __launch_bounds__(256)
split_q_kernel(double *B2, const double2 *__restrict__ Q, int64_t ns)
{
    const int64_t total = ns * ns;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = k % ns, j = k / ns;
        const double2 v = Q[k];
        B2[i + j * 2 * ns] = v.x;
        B2[ns + i + j * 2 * ns] = v.y;
    }
}

// A2 (2 nr x 2 ns real, ld lda2) = [view(P) | view(i P)] for the complex panel P (nr x ns, ld in complex elements)
__global__ void __launch_bounds__(256)
pack_panel_kernel(double *A2, int64_t lda2, const double2 *__restrict__ Pn, int64_t ld, int64_t nr, int64_t ns)
{
    const int64_t total = nr * ns;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = k % nr, c = k / nr;
        const double2 v = Pn[r + c * ld];
        *reinterpret_cast<double2 *>(A2 + 2 * r + c * lda2) = v;
        *reinterpret_cast<double2 *>(A2 + 2 * r + (ns + c) * lda2) = make_double2(-v.y, v.x);
    }
}

int grid_for(const sparc_gpu_ctx *ctx, int64_t total)
{
    return (int)std::min<int64_t>((total + 255) / 256, (int64_t)ctx->sm_count * 32);
}

int local_pass_k(sparc_gpu_ctx *c, const double2 *X, int64_t ldx, double2 *Out, int64_t ldo, const double2 *Prev, int64_t ldp,
                 int64_t ncols, double alpha, double shift, double beta, cudaStream_t st)
{
    KStencilParams P;
    for (int p = 0; p <= SPARC_MAX_RADIUS; ++p) {
        P.coef.cx[p] = alpha * c->coef.cx[p]; P.coef.cy[p] = alpha * c->coef.cy[p]; P.coef.cz[p] = alpha * c->coef.cz[p];
    }
    P.coef.c0 = alpha * c->coef.c0;
    P.alpha = alpha; P.shift = shift; P.beta = beta;
    for (int a = 0; a < 3; ++a) {
        P.n[a] = c->n[a]; P.bc[a] = c->bc[a];
        P.ph[a][0] = cos(c->k_theta[a]); P.ph[a][1] = sin(c->k_theta[a]);
    }
    P.radius = c->radius;
    for (int64_t j0 = 0; j0 < ncols; j0 += 65535) {
        const int64_t nb = std::min<int64_t>(ncols - j0, 65535);
        dim3 grid((unsigned)std::min<int64_t>((c->nd + 255) / 256, 4096), (unsigned)nb);
        prof_begin(c, KK_KPOINT, st);
        stencil_k_kernel<<<grid, 256, 0, st>>>(P, c->d_veff, X + j0 * ldx, ldx, Out + j0 * ldo, ldo,
                                               (beta != 0.0 && Prev) ? Prev + j0 * ldp : nullptr, ldp);
        prof_end(c, KK_KPOINT, st);
    }
    SPARC_CUDA_TRY(cudaGetLastError());
    return SPARC_GPU_SUCCESS;
}

// Out += scale V_nl(k) X  (D: n_proj_total x ncols complex scratch)
int nl_pass_k(sparc_gpu_ctx *c, const double2 *X, int64_t ldx, double2 *Out, int64_t ldo, int64_t ncols, double scale, double2 *D,
              cudaStream_t st)
{
    if (c->n_atoms <= 0 || c->n_proj_total <= 0 || c->supp_total <= 0 || !c->opt_nonlocal) return SPARC_GPU_SUCCESS;
    const int cols_per_cta = KP_WARPS * KP_COLS;
    for (int64_t j0 = 0; j0 < ncols; j0 += 65535LL * cols_per_cta) {
        const int64_t nb = std::min<int64_t>(ncols - j0, 65535LL * cols_per_cta);
        dim3 grid((unsigned)c->n_atoms, (unsigned)((nb + cols_per_cta - 1) / cols_per_cta));
#define KP_LAUNCH(PM)                                                                                                   \
        nl_project_k_kernel<PM><<<grid, KP_WARPS * 32, 0, st>>>(c->d_supp_ptr, c->d_supp_idx, c->d_n_proj, c->d_proj_ofs,  \
            c->d_chi_ptr, c->d_chi, c->d_gamma, c->d_k_phase, X + j0 * ldx, ldx, nb, scale, D + j0 * c->n_proj_total, c->n_proj_total)
        prof_begin(c, KK_KPOINT, st);
        if (c->max_proj <= 4) KP_LAUNCH(4);
        else if (c->max_proj <= 9) KP_LAUNCH(9);
        else KP_LAUNCH(16);
#undef KP_LAUNCH
        prof_end(c, KK_KPOINT, st);
    }
    SPARC_CUDA_TRY(cudaGetLastError());
    if (c->n_covered > 0) {
        int cols_per_block = 16;
        int64_t by = (ncols + cols_per_block - 1) / cols_per_block;
        while (by > 65535) { cols_per_block *= 2; by = (ncols + cols_per_block - 1) / cols_per_block; }
        dim3 grid((unsigned)((c->n_covered + 127) / 128), (unsigned)by);
        prof_begin(c, KK_KPOINT, st);
        nl_pull_k_kernel<<<grid, 128, 0, st>>>(c->d_cov_idx, c->d_cov_ptr, c->d_cov_ent, c->d_k_cov_phase, c->d_chi, D,
                                               c->n_proj_total, Out, ldo, c->n_covered, ncols, cols_per_block);
        prof_end(c, KK_KPOINT, st);
        SPARC_CUDA_TRY(cudaGetLastError());
    }
    return SPARC_GPU_SUCCESS;
}

int h_apply_block_k(sparc_gpu_ctx *c, const double2 *X, int64_t ldx, double2 *Y, int64_t ldy, int64_t ncols, double2 *D,
                    cudaStream_t st)
{
    SPARC_TRY(local_pass_k(c, X, ldx, Y, ldy, nullptr, 0, ncols, 1.0, 0.0, 0.0, st));
    SPARC_TRY(nl_pass_k(c, X, ldx, Y, ldy, ncols, 1.0, D, st));
    return SPARC_GPU_SUCCESS;
}

}  // namespace

// workspace carving of the k-point operators (called from ws_layout in context.cu)
int ws_layout_k(const sparc_gpu_ctx *c, int op, int64_t ns, int64_t block, WsLayout *L)
{
    const int64_t A = 256;
    int64_t off = 0;
    const int64_t n1 = std::max<int64_t>(ns, 1);
    if (op == SPARC_GPU_OP_ROTATE_K) {
        // A2 = [view(P) | view(iP)] (2 rp x 2 ns real), T (2 rp x ns real), B2 = [Re Q; Im Q] (2 ns x ns real)
        int64_t rp = block > 0 ? block : std::max<int64_t>(128, ((1024LL << 20) / (32 * n1)) / 128 * 128);
        rp = std::min<int64_t>(rp, c->nd);
        L->block = rp;
        L->ldw = round_up_i64(2 * rp, 16);
        L->off_w = off; off += round_up_i64(L->ldw * 2 * n1 * 8, A);
        L->off_d = off; off += round_up_i64(L->ldw * n1 * 8, A);
        L->off_g = off; off += round_up_i64(2 * n1 * n1 * 8, A);
    } else {
        const int64_t cb = block > 0 ? std::min(block, n1) : std::min<int64_t>(n1, 512);
        L->block = cb;
        L->ldw = round_up_i64(c->nd, 16);                      // complex elements
        L->off_w = off;                                        // W / Y block (complex)
        if (op != SPARC_GPU_OP_HAMILTONIAN_APPLY_K) off += round_up_i64(L->ldw * cb * 16, A);
        L->off_d = off; off += round_up_i64((int64_t)std::max(c->n_proj_total, 1) * cb * 16, A);
        L->off_g = off;
        if (op == SPARC_GPU_OP_PROJECT_K) {
            off += round_up_i64(L->ldw * cb * 16, A);          // -i Y block
            off += 2 * round_up_i64(n1 * cb * 8, A);           // Re, Im (ns x cb real each)
            off += round_up_i64(gemm_tn_ws_bytes(c, n1, cb, 2 * c->nd), A);
        }
    }
    L->total = std::max<int64_t>(off, A);
    return SPARC_GPU_SUCCESS;
}

void kpoint_free(sparc_gpu_ctx *c)
{
    cudaFree(c->d_k_phase); cudaFree(c->d_k_cov_phase);
    c->d_k_phase = c->d_k_cov_phase = nullptr;
}

extern "C" {

int sparc_gpu_set_kpoint(sparc_gpu_ctx *ctx, const double *theta, const int8_t *supp_shift)
{
    if (!ctx || !theta) return SPARC_GPU_INVALID_ARG;
    for (int a = 0; a < 3; ++a) if (!std::isfinite(theta[a])) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    // validate and build the new tables on the host FIRST: a bad shift leaves the previous k-point fully in place
    if (supp_shift)
        for (int64_t t = 0; t < 3 * ctx->supp_total; ++t)
            if (supp_shift[t] < -1 || supp_shift[t] > 1) return SPARC_GPU_BAD_DESCRIPTOR;
    double th[3];
    for (int a = 0; a < 3; ++a) th[a] = ctx->bc[a] == 0 ? theta[a] : 0.0;
    // exp(+i phi_t) per support row, and the same numbers in the order of the point -> (atom, row) cover entries
    std::vector<double> ph((size_t)ctx->supp_total * 2), cph((size_t)ctx->supp_total * 2);
    for (int64_t t = 0; t < ctx->supp_total; ++t) {
        double phi = 0.0;
        if (supp_shift)
            for (int a = 0; a < 3; ++a) phi += supp_shift[3 * t + a] * th[a];
        ph[2 * t] = cos(phi); ph[2 * t + 1] = sin(phi);
    }
    for (int64_t e = 0; e < ctx->supp_total; ++e) {
        const int64_t t = ctx->h_cov_row[(size_t)e];
        cph[2 * e] = ph[2 * t]; cph[2 * e + 1] = ph[2 * t + 1];
    }
    SPARC_CUDA_TRY(cudaDeviceSynchronize());             // a previous k-point's tables may still be in use
    // from here on the old k-point is gone; k_set goes back to 1 only once BOTH new tables are on the device, so that a failed
    // upload can never leave *_k calls with k_set = 1 and NULL tables
    ctx->k_set = 0;
    kpoint_free(ctx);
    for (int a = 0; a < 3; ++a) ctx->k_theta[a] = th[a];
    if (ctx->supp_total > 0) {
        double2 *p0 = nullptr, *p1 = nullptr;
        cudaError_t e = cudaMalloc((void **)&p0, ph.size() * 8);
        if (e == cudaSuccess) e = cudaMalloc((void **)&p1, cph.size() * 8);
        if (e == cudaSuccess) e = cudaMemcpy(p0, ph.data(), ph.size() * 8, cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(p1, cph.data(), cph.size() * 8, cudaMemcpyHostToDevice);
        if (e != cudaSuccess) {
            (void)cudaGetLastError();
            cudaFree(p0); cudaFree(p1);
            return e == cudaErrorMemoryAllocation ? SPARC_GPU_OUT_OF_MEMORY : SPARC_GPU_CUDA_ERROR;
        }
        ctx->d_k_phase = p0;
        ctx->d_k_cov_phase = p1;
    }
    ctx->k_set = 1;
    return SPARC_GPU_SUCCESS;
}

int sparc_gpu_hamiltonian_apply_k(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, double *Y, int64_t ldy, int64_t ncols,
                                  void *ws, void *stream)
{
    if (!ctx || ncols < 0) return SPARC_GPU_INVALID_ARG;
    if (ncols == 0) return SPARC_GPU_SUCCESS;
    if (!X || !Y || !ws || ldx < ctx->nd || ldy < ctx->nd || !ctx->k_set) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    WsLayout L;
    SPARC_TRY(ws_layout(ctx, SPARC_GPU_OP_HAMILTONIAN_APPLY_K, ncols, 0, &L));
    SPARC_TRY(ws_check(ctx, L));
    double2 *D = (double2 *)((char *)ws + L.off_d);
    const double2 *Xc = (const double2 *)X;
    double2 *Yc = (double2 *)Y;
    for (int64_t j0 = 0; j0 < ncols; j0 += L.block) {
        const int64_t nb = std::min(L.block, ncols - j0);
        SPARC_TRY(h_apply_block_k(ctx, Xc + j0 * ldx, ldx, Yc + j0 * ldy, ldy, nb, D, (cudaStream_t)stream));
    }
    return SPARC_GPU_SUCCESS;
}

int sparc_gpu_chebyshev_filter_k(sparc_gpu_ctx *ctx, double *Psi, int64_t ld, int64_t ns, int degree, double a, double b,
                                 double a0, int64_t col_block, void *ws, void *stream)
{
    if (!ctx || ns < 0 || degree < 0) return SPARC_GPU_INVALID_ARG;
    if (!(a0 < a && a < b)) return SPARC_GPU_BAD_BOUNDS;
    if (ns == 0 || degree == 0) return SPARC_GPU_SUCCESS;
    if (!Psi || !ws || ld < ctx->nd || !ctx->k_set) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    cudaStream_t st = (cudaStream_t)stream;
    WsLayout L;
    SPARC_TRY(ws_layout(ctx, SPARC_GPU_OP_CHEBYSHEV_FILTER_K, ns, col_block, &L));
    SPARC_TRY(ws_check(ctx, L));
    double2 *W = (double2 *)((char *)ws + L.off_w);
    double2 *D = (double2 *)((char *)ws + L.off_d);
    const double e = 0.5 * (b - a), c = 0.5 * (b + a);
    const double sigma1 = e / (a0 - c), tau = 2.0 / sigma1;
    double2 *P = (double2 *)Psi;
    for (int64_t j0 = 0; j0 < ns; j0 += L.block) {
        const int64_t nb = std::min(L.block, ns - j0);
        double2 *bufA = P + j0 * ld;
        double2 *cur = bufA, *oth = W;
        int64_t ldc = ld, ldo = L.ldw;
        double sigma = sigma1;
        for (int k = 1; k <= degree; ++k) {           // oth <- alpha (H cur - c cur) + beta oth   (R3)
            const double sigma2 = 1.0 / (tau - sigma);
            const double alpha = (k == 1) ? sigma1 / e : 2.0 * sigma2 / e;
            const double beta = (k == 1) ? 0.0 : -(sigma * sigma2);
            SPARC_TRY(local_pass_k(ctx, cur, ldc, oth, ldo, k == 1 ? nullptr : oth, ldo, nb, alpha, -c, beta, st));
            SPARC_TRY(nl_pass_k(ctx, cur, ldc, oth, ldo, nb, alpha, D, st));
            if (k > 1) sigma = sigma2;
            std::swap(cur, oth); std::swap(ldc, ldo);
        }
        if (cur != bufA) SPARC_TRY(launch_copy_2d(ctx, (double *)bufA, 2 * ld, (const double *)cur, 2 * ldc, 2 * ctx->nd, nb, st));
    }
    return SPARC_GPU_SUCCESS;
}

int sparc_gpu_project_k(sparc_gpu_ctx *ctx, const double *Psi, int64_t ld, int64_t ns, double *Hs, double *Ms,
                        int64_t col_block, void *ws, void *stream)
{
    if (!ctx || ns < 0) return SPARC_GPU_INVALID_ARG;
    if (ns == 0) return SPARC_GPU_SUCCESS;
    if (!Psi || !Hs || !Ms || !ws || ld < ctx->nd || !ctx->k_set) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    cudaStream_t st = (cudaStream_t)stream;
    WsLayout L;
    SPARC_TRY(ws_layout(ctx, SPARC_GPU_OP_PROJECT_K, ns, col_block, &L));
    SPARC_TRY(ws_check(ctx, L));
    const int64_t A = 256, cb = L.block, nd = ctx->nd;
    double2 *Y = (double2 *)((char *)ws + L.off_w);
    double2 *D = (double2 *)((char *)ws + L.off_d);
    char *p = (char *)ws + L.off_g;
    double2 *Yr = (double2 *)p; p += round_up_i64(L.ldw * cb * 16, A);
    double *Re = (double *)p; p += round_up_i64(ns * cb * 8, A);
    double *Im = (double *)p; p += round_up_i64(ns * cb * 8, A);
    void *G = p;
    const double2 *Pc = (const double2 *)Psi;
    // Re(A^H B) = view(A)^T view(B), Im(A^H B) = view(A)^T view(-i B): two real TN products over the 2 N_d real rows
    auto gram_block = [&](const double2 *B, int64_t ldb, int64_t nb, double2 *Cout) -> int {
        SPARC_TRY(launch_gemm_tn(ctx, (const double *)Pc, 2 * ld, (const double *)B, 2 * ldb, Re, ns, ns, nb, 2 * nd, G, -1, st));
        prof_begin(ctx, KK_KPOINT, st);
        rot_i_kernel<true><<<grid_for(ctx, nd * nb), 256, 0, st>>>(Yr, L.ldw, B, ldb, nd, nb);
        prof_end(ctx, KK_KPOINT, st);
        SPARC_CUDA_TRY(cudaGetLastError());
        SPARC_TRY(launch_gemm_tn(ctx, (const double *)Pc, 2 * ld, (const double *)Yr, 2 * L.ldw, Im, ns, ns, nb, 2 * nd, G, -1, st));
        prof_begin(ctx, KK_KPOINT, st);
        combine_kernel<<<grid_for(ctx, ns * nb), 256, 0, st>>>(Cout, ns, Re, Im, ns, nb);
        prof_end(ctx, KK_KPOINT, st);
        SPARC_CUDA_TRY(cudaGetLastError());
        return SPARC_GPU_SUCCESS;
    };
    for (int64_t j0 = 0; j0 < ns; j0 += cb) {
        const int64_t nb = std::min(cb, ns - j0);
        SPARC_TRY(h_apply_block_k(ctx, Pc + j0 * ld, ld, Y, L.ldw, nb, D, st));
        SPARC_TRY(gram_block(Y, L.ldw, nb, (double2 *)Hs + j0 * ns));
        SPARC_TRY(gram_block(Pc + j0 * ld, ld, nb, (double2 *)Ms + j0 * ns));
    }
    return SPARC_GPU_SUCCESS;
}

int sparc_gpu_rotate_k(sparc_gpu_ctx *ctx, double *Psi, int64_t ld, int64_t ns, const double *Q, int64_t row_panel, void *ws,
                       void *stream)
{
    if (!ctx || ns < 0) return SPARC_GPU_INVALID_ARG;
    if (ns == 0) return SPARC_GPU_SUCCESS;
    if (!Psi || !Q || !ws || ld < ctx->nd) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    cudaStream_t st = (cudaStream_t)stream;
    WsLayout L;
    SPARC_TRY(ws_layout(ctx, SPARC_GPU_OP_ROTATE_K, ns, row_panel, &L));
    SPARC_TRY(ws_check(ctx, L));
    double *A2 = (double *)((char *)ws + L.off_w);
    double *T = (double *)((char *)ws + L.off_d);
    double *B2 = (double *)((char *)ws + L.off_g);
    prof_begin(ctx, KK_KPOINT, st);
    split_q_kernel<<<grid_for(ctx, ns * ns), 256, 0, st>>>(B2, (const double2 *)Q, ns);
    prof_end(ctx, KK_KPOINT, st);
    SPARC_CUDA_TRY(cudaGetLastError());
    double2 *Pc = (double2 *)Psi;
    for (int64_t r0 = 0; r0 < ctx->nd; r0 += L.block) {
        const int64_t nr = std::min(L.block, ctx->nd - r0);
        prof_begin(ctx, KK_KPOINT, st);
        pack_panel_kernel<<<grid_for(ctx, nr * ns), 256, 0, st>>>(A2, L.ldw, Pc + r0, ld, nr, ns);
        prof_end(ctx, KK_KPOINT, st);
        SPARC_CUDA_TRY(cudaGetLastError());
        // view(P Q) = [view(P) | view(i P)] [Re Q; Im Q]
        SPARC_TRY(launch_gemm_nn(ctx, A2, L.ldw, B2, 2 * ns, T, L.ldw, 2 * nr, ns, 2 * ns, st));
        SPARC_TRY(launch_copy_2d(ctx, (double *)(Pc + r0), 2 * ld, T, L.ldw, 2 * nr, ns, st));
    }
    return SPARC_GPU_SUCCESS;
}

}  // extern "C"
