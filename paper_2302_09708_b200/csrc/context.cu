// context.cu -- C-ABI entry points: context lifetime, validation, host-side orchestration of the
// filter / project / rotate passes.  All arithmetic of the method runs in the kernels launched from
// here (stencil_*.cu, nonlocal.cu, gemm.cu); this file only sequences them.
#include <cuda.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <new>
#include <vector>

#include "internal.h"

struct ProfRec { int kind; cudaEvent_t a, b; };
struct ProfState {
    bool on = false;
    std::vector<ProfRec> recs;
    std::vector<cudaEvent_t> pool;
    double ns[KK_COUNT] = {0};
    int64_t count[KK_COUNT] = {0};
    cudaEvent_t cur = nullptr;
};

void prof_begin(sparc_gpu_ctx *ctx, int kind, cudaStream_t st)
{
    ctx->kernel_launches++;
    ProfState *p = ctx->prof;
    if (!p) return;
    p->count[kind]++;
    if (!p->on) return;
    cudaEvent_t a;
    if (p->pool.empty()) { if (cudaEventCreate(&a) != cudaSuccess) { (void)cudaGetLastError(); p->cur = nullptr; return; } }
    else { a = p->pool.back(); p->pool.pop_back(); }
    cudaEventRecord(a, st);
    p->cur = a;
}

void prof_end(sparc_gpu_ctx *ctx, int kind, cudaStream_t st)
{
    ProfState *p = ctx->prof;
    if (!p || !p->on || !p->cur) return;
    cudaEvent_t b;
    if (p->pool.empty()) { if (cudaEventCreate(&b) != cudaSuccess) { (void)cudaGetLastError(); return; } }
    else { b = p->pool.back(); p->pool.pop_back(); }
    cudaEventRecord(b, st);
    p->recs.push_back({kind, p->cur, b});
    p->cur = nullptr;
}

namespace {

// fold finished event pairs into the per-kind totals (caller has synchronised the stream)
void prof_collect(ProfState *p)
{
    for (auto &r : p->recs) {
        float ms = 0.f;
        if (cudaEventSynchronize(r.b) == cudaSuccess && cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess)
            p->ns[r.kind] += (double)ms * 1e6;
        else
            (void)cudaGetLastError();
        p->pool.push_back(r.a);
        p->pool.push_back(r.b);
    }
    p->recs.clear();
}

// O(1) host arithmetic: central FD weights of the second derivative, radius r (R1).
void fd_weights_host(int r, double *w)
{
    long double w0 = 0.0L;
    for (int p = 1; p <= r; ++p) {
        long double ratio = 1.0L;   // (r!)^2 / ((r-p)! (r+p)!)
        for (int j = 1; j <= p; ++j) ratio *= (long double)(r - p + j) / (long double)(r + j);
        long double v = 2.0L / ((long double)p * p) * ratio;
        w[p] = (double)((p & 1) ? v : -v);
        w0 -= 2.0L / ((long double)p * p);
    }
    w[0] = (double)w0;
}

// central FD weights of the first derivative, radius r (reading R21): w_p = (-1)^{p+1} (r!)^2 / (p (r-p)! (r+p)!)
void fd1_weights_host(int r, double *w)
{
    w[0] = 0.0;
    for (int p = 1; p <= r; ++p) {
        long double ratio = 1.0L;
        for (int j = 1; j <= p; ++j) ratio *= (long double)(r - p + j) / (long double)(r + j);
        w[p] = (double)(((p & 1) ? ratio : -ratio) / (long double)p);
    }
}

template <typename T>
int upload(T **dst, const T *src, size_t count)
{
    *dst = nullptr;
    if (count == 0) return SPARC_GPU_SUCCESS;
    SPARC_CUDA_TRY(cudaMalloc((void **)dst, count * sizeof(T)));
    SPARC_CUDA_TRY(cudaMemcpy(*dst, src, count * sizeof(T), cudaMemcpyHostToDevice));
    return SPARC_GPU_SUCCESS;
}

void free_tables(sparc_gpu_ctx *c)
{
    cudaFree(c->d_supp_ptr); cudaFree(c->d_supp_idx); cudaFree(c->d_n_proj); cudaFree(c->d_proj_ofs);
    cudaFree(c->d_chi_ptr); cudaFree(c->d_chi); cudaFree(c->d_gamma); cudaFree(c->d_cov_idx);
    cudaFree(c->d_cov_ptr); cudaFree(c->d_cov_ent); cudaFree(c->d_veff);
    for (int k = 0; k < 2; ++k) if (c->copy_stream[k]) { cudaStreamDestroy(c->copy_stream[k]); c->copy_stream[k] = nullptr; }
    nlb_free(c);
    kpoint_free(c);
}

int validate_desc(const sparc_gpu_desc *d)
{
    for (int a = 0; a < 3; ++a) {
        if (d->n[a] < 1 || !(d->h[a] > 0.0) || !std::isfinite(d->h[a])) return SPARC_GPU_INVALID_ARG;
        if (d->bc[a] != 0 && d->bc[a] != 1) return SPARC_GPU_INVALID_ARG;
    }
    if ((int64_t)d->n[0] * d->n[1] * d->n[2] >= (int64_t)INT32_MAX) return SPARC_GPU_UNSUPPORTED;   // R20
    if (d->fd_order < 2 || d->fd_order > 2 * SPARC_MAX_RADIUS || (d->fd_order & 1)) return SPARC_GPU_UNSUPPORTED;
    for (int a = 0; a < 3; ++a)
        if (d->bc[a] == 0 && d->n[a] < d->fd_order + 1) return SPARC_GPU_UNSUPPORTED;               // R10
    if (d->n_atoms < 0) return SPARC_GPU_INVALID_ARG;
    if (d->n_atoms > 0) {
        if (!d->supp_ptr || !d->supp_idx || !d->n_proj || !d->chi_ptr || !d->chi || !d->gamma)
            return SPARC_GPU_INVALID_ARG;
        const int64_t nd = (int64_t)d->n[0] * d->n[1] * d->n[2];
        if (d->supp_ptr[0] != 0 || d->chi_ptr[0] != 0) return SPARC_GPU_BAD_DESCRIPTOR;
        for (int J = 0; J < d->n_atoms; ++J) {
            const int64_t s0 = d->supp_ptr[J], s1 = d->supp_ptr[J + 1];
            const int P = d->n_proj[J];
            if (s1 < s0 || P < 0 || P > SPARC_MAX_PROJ) return SPARC_GPU_BAD_DESCRIPTOR;
            if (d->chi_ptr[J + 1] - d->chi_ptr[J] != (s1 - s0) * P) return SPARC_GPU_BAD_DESCRIPTOR;
            for (int64_t t = s0; t < s1; ++t) {
                const int32_t i = d->supp_idx[t];
                if (i < 0 || i >= nd) return SPARC_GPU_BAD_DESCRIPTOR;
                if (t > s0 && i <= d->supp_idx[t - 1]) return SPARC_GPU_BAD_DESCRIPTOR;             // R8
            }
        }
    }
    return SPARC_GPU_SUCCESS;
}

// Out = alpha (H_loc X + shift X) + beta Prev on one column block: the fused local pass (stencil + Veff + axpy).
int local_pass(sparc_gpu_ctx *c, const double *X, int64_t ldx, double *Out, int64_t ldo, const double *Prev,
               int64_t ldp, int64_t ncols, double alpha, double shift, double beta, cudaStream_t st)
{
    int path = c->opt_stencil_path;
    if (path == 0) {
        // wide grids (12 x-blocks): the hybrid DMMA kernel is ~5 % ahead (configs 3-4); otherwise the DFMA kernel
        if (c->n[0] >= 64 && stencil_dmma_supported(c, X, ldx, Out, ldo, Prev, ldp)) path = 3;
        else path = stencil_tma_supported(c, X, ldx, Out, ldo, Prev, ldp) ? 2 : 1;
    }
    if (path == 3) {
        SPARC_TRY(launch_stencil_dmma(c, X, ldx, Out, ldo, Prev, ldp, ncols, alpha, shift, beta, st));
    } else if (path == 2) {
        SPARC_TRY(launch_stencil_tma(c, X, ldx, Out, ldo, Prev, ldp, ncols, alpha, shift, beta, st));
    } else {
        SPARC_TRY(launch_stencil_generic(c, X, ldx, Out, ldo, Prev, ldp, ncols, alpha, shift, beta, st));
    }
    c->stencil_path_last = path;
    return SPARC_GPU_SUCCESS;
}

// Nonlocal path of a pass that reads X and updates Out: -1 none, 1 project + pull, 2 per-atom fused, 3 brick.
int effective_nl_mode(const sparc_gpu_ctx *c, const double *X, int64_t ldx, const double *Out, int64_t ldo)
{
    if (!c->opt_nonlocal || c->n_atoms <= 0 || c->n_proj_total <= 0 || c->supp_total <= 0) return -1;
    if (c->opt_nonlocal_mode != 0) return c->opt_nonlocal_mode;
    return (nlb_supported(c, X, ldx) && nlb_supported(c, Out, ldo)) ? 3 : 2;
}

// Out += alpha V_nl X with the per-atom kernels (modes 1, 2)
int nl_pass_per_atom(sparc_gpu_ctx *c, int mode, const double *X, int64_t ldx, double *Out, int64_t ldo, int64_t ncols,
                     double alpha, double *D, cudaStream_t st)
{
    if (mode == 1) {
        SPARC_TRY(launch_nl_project(c, X, ldx, ncols, alpha, D, st));
        SPARC_TRY(launch_nl_pull(c, D, Out, ldo, ncols, st));
    } else {
        SPARC_TRY(launch_nl_fused(c, X, ldx, Out, ldo, ncols, alpha, st));
    }
    return SPARC_GPU_SUCCESS;
}

// Y = H X on one column block (D: workspace of 2 * n_proj_total * ncols doubles)
int h_apply_block(sparc_gpu_ctx *c, const double *X, int64_t ldx, double *Y, int64_t ldy, int64_t ncols, double *D,
                  cudaStream_t st)
{
    const int mode = effective_nl_mode(c, X, ldx, Y, ldy);
    if (mode == 3) {      // chi^T X first (X may not be read after Y is written when they alias; they never do here)
        SPARC_CUDA_TRY(cudaMemsetAsync(D, 0, (size_t)nlb_c_doubles(c, ncols) * 8, st));
        SPARC_TRY(launch_nl_brick(c, 1, const_cast<double *>(X), ldx, ncols, 1.0, nullptr, D, st));
    }
    SPARC_TRY(local_pass(c, X, ldx, Y, ldy, nullptr, 0, ncols, 1.0, 0.0, 0.0, st));
    if (mode == 3) SPARC_TRY(launch_nl_brick(c, 2, Y, ldy, ncols, 1.0, D, nullptr, st));
    else if (mode > 0) SPARC_TRY(nl_pass_per_atom(c, mode, X, ldx, Y, ldy, ncols, 1.0, D, st));
    return SPARC_GPU_SUCCESS;
}

}  // namespace


static int64_t default_col_block(const sparc_gpu_ctx *c, int64_t ns) { (void)c; return std::min<int64_t>(ns, 1024); }

static int64_t default_row_panel(const sparc_gpu_ctx *c, int64_t ns)
{
    // stage of at most ~2 GiB, at least 128 rows, multiple of 128
    int64_t r = (int64_t)(2048LL << 20) / (8 * std::max<int64_t>(ns, 1));
    r = std::max<int64_t>(128, r / 128 * 128);
    return std::min<int64_t>(r, round_up_i64(c->nd, 128));
}

int ws_layout(const sparc_gpu_ctx *c, int op, int64_t ns, int64_t block, WsLayout *L)
{
    if (ns < 0) return SPARC_GPU_INVALID_ARG;
    memset(L, 0, sizeof(*L));
    const int64_t A = 256;
    int64_t off = 0;
    switch (op) {
    case SPARC_GPU_OP_HAMILTONIAN_APPLY:
    case SPARC_GPU_OP_CHEBYSHEV_FILTER:
    case SPARC_GPU_OP_PROJECT: {
        int64_t cb = block > 0 ? std::min(block, std::max<int64_t>(ns, 1)) : default_col_block(c, std::max<int64_t>(ns, 1));
        L->block = cb;
        L->ldw = round_up_i64(c->nd, 16);
        L->off_w = off;
        if (op != SPARC_GPU_OP_HAMILTONIAN_APPLY) off += round_up_i64(L->ldw * cb * 8, A);
        L->off_d = off;
        off += round_up_i64(2 * std::max<int64_t>((int64_t)std::max(c->n_proj_total, 1) * nlb_c_cols(cb), nlb_c_doubles(c, cb)) * 8, A);
        L->off_g = off;
        if (op == SPARC_GPU_OP_PROJECT) {
            off += round_up_i64(std::max(gemm_tn_ws_bytes(c, ns, cb, c->nd), gemm_tn_ws_bytes(c, ns, ns, c->nd)), A);
        }
        break;
    }
    case SPARC_GPU_OP_GRADIENT_PROJECT:
    case SPARC_GPU_OP_NONLOCAL_FORCE: {
        // one gradient block Y = D_a X, and (force) the two projection blocks W = chi^T X, G = chi^T Y
        int64_t cb = block > 0 ? std::min(block, std::max<int64_t>(ns, 1)) : default_col_block(c, std::max<int64_t>(ns, 1));
        L->block = cb;
        L->ldw = round_up_i64(c->nd, 16);
        L->off_w = off;
        off += round_up_i64(L->ldw * cb * 8, A);
        L->off_d = off;
        if (op == SPARC_GPU_OP_NONLOCAL_FORCE) off += round_up_i64(2 * (int64_t)std::max(c->n_proj_total, 1) * cb * 8, A);
        break;
    }
    case SPARC_GPU_OP_EIGENSOLVE: {
        // A, V (n x n each, the Jacobi iterate and the accumulated rotations), L (Cholesky factor), 2 n scalars
        const int64_t n = std::max<int64_t>(ns, 1), np = round_up_i64(n, 32);
        L->block = np;
        L->ldw = np;
        L->off_w = off;
        off += round_up_i64(4 * np * np * 8 + 8 * np * 8 + 4096, A);
        break;
    }
    case SPARC_GPU_OP_HAMILTONIAN_APPLY_K:
    case SPARC_GPU_OP_CHEBYSHEV_FILTER_K:
    case SPARC_GPU_OP_PROJECT_K:
    case SPARC_GPU_OP_ROTATE_K:
        return ws_layout_k(c, op, ns, block, L);
    case SPARC_GPU_OP_GRAM: {
        const int64_t n = std::max<int64_t>(ns, 1);
        L->block = n; L->ldw = n; L->off_w = off; L->off_g = off;
        off += round_up_i64(gemm_tn_ws_bytes(c, n, n, c->nd), A);
        break;
    }
    case SPARC_GPU_OP_ROTATE: {
        int64_t rp = block > 0 ? block : default_row_panel(c, ns);
        rp = std::min<int64_t>(rp, c->nd);
        L->block = rp;
        L->ldw = round_up_i64(rp, 16);
        L->off_w = off;
        off += round_up_i64(L->ldw * std::max<int64_t>(ns, 1) * 8, A);
        break;
    }
    default:
        return SPARC_GPU_INVALID_ARG;
    }
    L->total = std::max<int64_t>(off, A);
    return SPARC_GPU_SUCCESS;
}

// the caller declared the size of its workspace (sparc_gpu_set_workspace_size): refuse a call that would overrun it
int ws_check(const sparc_gpu_ctx *c, const WsLayout &L)
{
    return (c->ws_bytes > 0 && L.total > c->ws_bytes) ? SPARC_GPU_WORKSPACE_TOO_SMALL : SPARC_GPU_SUCCESS;
}


// row panel and stage pitch a rotation of ns columns uses (and the workspace check that goes with them)
int rotate_layout(const sparc_gpu_ctx *c, int64_t ns, int64_t row_panel, int64_t *rp, int64_t *ldw)
{
    WsLayout L;
    SPARC_TRY(ws_layout(c, SPARC_GPU_OP_ROTATE, ns, row_panel, &L));
    SPARC_TRY(ws_check(c, L));
    *rp = L.block; *ldw = L.ldw;
    return SPARC_GPU_SUCCESS;
}

// rows [0, nr) of Psi_rows <- the same rows times Q, staged through T (the product must not overwrite rows it still reads)
int rotate_panel(sparc_gpu_ctx *c, double *Psi_rows, int64_t ld, int64_t nr, int64_t ns, const double *Q, double *T,
                 int64_t ldw, cudaStream_t st)
{
    SPARC_TRY(launch_gemm_nn(c, Psi_rows, ld, Q, ns, T, ldw, nr, ns, ns, st));
    SPARC_TRY(launch_copy_2d(c, Psi_rows, ld, T, ldw, nr, ns, st));
    return SPARC_GPU_SUCCESS;
}

extern "C" {

const char *sparc_gpu_version(void) { return "sparc_gpu 0.1.0 (sm_100a)"; }

const char *sparc_gpu_error_string(int code)
{
    switch (code) {
    case SPARC_GPU_SUCCESS: return "success";
    case SPARC_GPU_INVALID_ARG: return "invalid argument";
    case SPARC_GPU_UNSUPPORTED: return "unsupported configuration or device";
    case SPARC_GPU_BAD_BOUNDS: return "filter bounds must satisfy a0 < a < b";
    case SPARC_GPU_BAD_DESCRIPTOR: return "inconsistent projector descriptor";
    case SPARC_GPU_WORKSPACE_TOO_SMALL: return "workspace too small";
    case SPARC_GPU_OUT_OF_MEMORY: return "out of device memory";
    case SPARC_GPU_CUDA_ERROR: return "CUDA error";
    case SPARC_GPU_STATIC_SCRATCH_EXCEEDED: return "m * n exceeds the built-in static scratch of sparc_gpu_gram_static (2097152 doubles)";
    default: return "unknown status";
    }
}

int sparc_gpu_create(const sparc_gpu_desc *desc, sparc_gpu_ctx **out)
{
    if (!desc || !out) return SPARC_GPU_INVALID_ARG;
    *out = nullptr;
    SPARC_TRY(validate_desc(desc));
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) { (void)cudaGetLastError(); return SPARC_GPU_UNSUPPORTED; }
    if (desc->device < 0 || desc->device >= ndev) return SPARC_GPU_INVALID_ARG;
    cudaDeviceProp prop;
    SPARC_CUDA_TRY(cudaGetDeviceProperties(&prop, desc->device));
    if (prop.major != 10) return SPARC_GPU_UNSUPPORTED;     // sm_100a only, no fallback
    DeviceGuard dg(desc->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;

    sparc_gpu_ctx *c = new (std::nothrow) sparc_gpu_ctx();
    if (!c) return SPARC_GPU_OUT_OF_MEMORY;
    c->device = desc->device;
    c->sm_count = prop.multiProcessorCount;
    for (int a = 0; a < 3; ++a) { c->n[a] = desc->n[a]; c->h[a] = desc->h[a]; c->bc[a] = desc->bc[a]; }
    c->radius = desc->fd_order / 2;
    c->nd = (int64_t)desc->n[0] * desc->n[1] * desc->n[2];
    c->prof = new (std::nothrow) ProfState();
    fd_weights_host(c->radius, c->w);
    fd1_weights_host(c->radius, c->w1);
    double isum = 0.0;
    for (int p = 0; p <= SPARC_MAX_RADIUS; ++p) { c->coef.cx[p] = c->coef.cy[p] = c->coef.cz[p] = 0.0; }
    for (int p = 1; p <= c->radius; ++p) {
        c->coef.cx[p] = -0.5 * c->w[p] / (c->h[0] * c->h[0]);
        c->coef.cy[p] = -0.5 * c->w[p] / (c->h[1] * c->h[1]);
        c->coef.cz[p] = -0.5 * c->w[p] / (c->h[2] * c->h[2]);
    }
    for (int a = 0; a < 3; ++a) isum += 1.0 / (c->h[a] * c->h[a]);
    c->coef.c0 = -0.5 * c->w[0] * isum;

    // resolve cuTensorMapEncodeTiled without linking libcuda
    {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            c->fn_encode_tiled = fn;
        else
            (void)cudaGetLastError();
    }

    int st = SPARC_GPU_SUCCESS;
    do {
        // local potential
        if ((st = (cudaMalloc((void **)&c->d_veff, (size_t)c->nd * 8) == cudaSuccess) ? 0 : SPARC_GPU_OUT_OF_MEMORY)) break;
        if (desc->veff) {
            if (cudaMemcpy(c->d_veff, desc->veff, (size_t)c->nd * 8, cudaMemcpyHostToDevice) != cudaSuccess) { st = SPARC_GPU_CUDA_ERROR; break; }
        } else if (cudaMemset(c->d_veff, 0, (size_t)c->nd * 8) != cudaSuccess) { st = SPARC_GPU_CUDA_ERROR; break; }

        c->n_atoms = desc->n_atoms;
        if (c->n_atoms == 0) break;
        const int na = c->n_atoms;
        c->supp_total = desc->supp_ptr[na];
        std::vector<int32_t> pofs(na + 1, 0);
        for (int J = 0; J < na; ++J) {
            pofs[J + 1] = pofs[J] + desc->n_proj[J];
            c->max_proj = std::max<int32_t>(c->max_proj, desc->n_proj[J]);
        }
        c->n_proj_total = pofs[na];
        if ((st = upload(&c->d_supp_ptr, desc->supp_ptr, (size_t)na + 1))) break;
        if ((st = upload(&c->d_supp_idx, desc->supp_idx, (size_t)c->supp_total))) break;
        if ((st = upload(&c->d_n_proj, desc->n_proj, (size_t)na))) break;
        if ((st = upload(&c->d_proj_ofs, pofs.data(), (size_t)na + 1))) break;
        if ((st = upload(&c->d_chi_ptr, desc->chi_ptr, (size_t)na + 1))) break;
        if ((st = upload(&c->d_chi, desc->chi, (size_t)desc->chi_ptr[na]))) break;
        if ((st = upload(&c->d_gamma, desc->gamma, (size_t)c->n_proj_total))) break;

        // inverse map point -> list of (atom, row): counting sort by grid index
        std::vector<int64_t> cnt((size_t)c->nd + 1, 0);
        for (int64_t t = 0; t < c->supp_total; ++t) cnt[(size_t)desc->supp_idx[t] + 1]++;
        std::vector<int32_t> cov_idx;
        std::vector<int64_t> cov_ptr;
        std::vector<int64_t> slot((size_t)c->nd, -1);
        cov_ptr.push_back(0);
        for (int64_t i = 0; i < c->nd; ++i) {
            if (cnt[(size_t)i + 1] > 0) {
                slot[(size_t)i] = cov_ptr.back();
                cov_idx.push_back((int32_t)i);
                cov_ptr.push_back(cov_ptr.back() + cnt[(size_t)i + 1]);
            }
        }
        c->n_covered = (int64_t)cov_idx.size();
        std::vector<CoverEntry> ent((size_t)c->supp_total);
        c->h_cov_row.assign((size_t)c->supp_total, 0);
        for (int J = 0; J < na; ++J) {
            const int64_t s0 = desc->supp_ptr[J], nJ = desc->supp_ptr[J + 1] - s0;
            for (int64_t t = 0; t < nJ; ++t) {
                const int32_t i = desc->supp_idx[s0 + t];
                CoverEntry e;
                e.chi_off = desc->chi_ptr[J] + t;
                e.n_j = (int32_t)nJ;
                e.pofs_p = (pofs[J] << 8) | desc->n_proj[J];
                c->h_cov_row[(size_t)slot[(size_t)i]] = s0 + t;
                ent[(size_t)slot[(size_t)i]++] = e;      // atoms in ascending J order per point: deterministic
            }
        }
        if ((st = upload(&c->d_cov_idx, cov_idx.data(), cov_idx.size()))) break;
        if ((st = upload(&c->d_cov_ptr, cov_ptr.data(), cov_ptr.size()))) break;
        if ((st = upload(&c->d_cov_ent, ent.data(), ent.size()))) break;
        if ((st = nlb_build(c, desc))) break;
    } while (0);
    if (st != SPARC_GPU_SUCCESS) { (void)cudaGetLastError(); free_tables(c); delete c->prof; delete c; return st; }
    *out = c;
    return SPARC_GPU_SUCCESS;
}

int sparc_gpu_destroy(sparc_gpu_ctx *ctx)
{
    if (!ctx) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    free_tables(ctx);
    if (ctx->prof) {
        prof_collect(ctx->prof);
        for (auto e : ctx->prof->pool) cudaEventDestroy(e);
        delete ctx->prof;
    }
    delete ctx;
    return SPARC_GPU_SUCCESS;
}

int sparc_gpu_set_veff(sparc_gpu_ctx *ctx, const double *veff_dev, void *stream)
{
    if (!ctx || !veff_dev) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    SPARC_CUDA_TRY(cudaMemcpyAsync(ctx->d_veff, veff_dev, (size_t)ctx->nd * 8, cudaMemcpyDeviceToDevice,
                                   (cudaStream_t)stream));
    return SPARC_GPU_SUCCESS;
}

int sparc_gpu_set_option(sparc_gpu_ctx *ctx, const char *key, int64_t value)
{
    if (!ctx || !key) return SPARC_GPU_INVALID_ARG;
    if (!strcmp(key, "stencil_path")) { if (value < 0 || value > 3) return SPARC_GPU_INVALID_ARG; ctx->opt_stencil_path = (int)value; return 0; }
    if (!strcmp(key, "nonlocal_mode")) { if (value < 0 || value > 3) return SPARC_GPU_INVALID_ARG; ctx->opt_nonlocal_mode = (int)value; return 0; }
    if (!strcmp(key, "nonlocal")) { ctx->opt_nonlocal = value ? 1 : 0; return 0; }
    if (!strcmp(key, "profile")) { if (!ctx->prof) return SPARC_GPU_OUT_OF_MEMORY; ctx->prof->on = value != 0; return 0; }
    if (!strcmp(key, "profile_reset")) {
        if (!ctx->prof) return SPARC_GPU_OUT_OF_MEMORY;
        prof_collect(ctx->prof);
        for (int k = 0; k < KK_COUNT; ++k) { ctx->prof->ns[k] = 0; ctx->prof->count[k] = 0; }
        ctx->gemm_flop[0] = ctx->gemm_flop[1] = 0.0;
        return 0;
    }
    if (!strcmp(key, "stencil_ay")) { if (value < 0 || value > 2) return SPARC_GPU_INVALID_ARG; ctx->opt_stencil_ay = (int)value; ctx->tma_choice.valid = 0; return 0; }
    if (!strcmp(key, "stencil_ty")) { if (value < 0) return SPARC_GPU_INVALID_ARG; ctx->opt_stencil_ty = (int)value; ctx->tma_choice.valid = 0; return 0; }
    // ring depth 2..8 (a one-stage ring cannot overlap the TMA copy with the arithmetic: rejected here, not at launch)
    if (!strcmp(key, "stencil_stages")) { if (value != 0 && (value < 2 || value > 8)) return SPARC_GPU_INVALID_ARG; ctx->opt_stencil_stages = (int)value; ctx->tma_choice.valid = 0; return 0; }
    if (!strcmp(key, "eig_coop")) { ctx->opt_eig_coop = value ? 1 : 0; return 0; }
    if (!strcmp(key, "stencil_xt")) { if (value != 0 && (value < 32 || value > 96 || value % 8)) return SPARC_GPU_INVALID_ARG; ctx->opt_stencil_xt = (int)value; return 0; }
    if (!strcmp(key, "stencil_zchunks")) { if (value < 0) return SPARC_GPU_INVALID_ARG; ctx->opt_stencil_zchunks = (int)value; return 0; }
    if (!strcmp(key, "nlb_dbg")) { ctx->opt_nlb_dbg = (int)value; return 0; }
    if (!strcmp(key, "nlb_kernel")) { if (value < 0 || value > 2) return SPARC_GPU_INVALID_ARG; ctx->opt_nlb_kernel = (int)value; return 0; }
    if (!strcmp(key, "nlb_cap")) { if (value < 0) return SPARC_GPU_INVALID_ARG; ctx->opt_nlb_cap = (int)value; return 0; }
    if (!strcmp(key, "gemm_full")) { ctx->opt_gemm_full = value ? 1 : 0; return 0; }
    if (!strcmp(key, "gemm_path")) { if (value < 0 || value > 2) return SPARC_GPU_INVALID_ARG; ctx->opt_gemm_path = (int)value; return 0; }
    return SPARC_GPU_INVALID_ARG;
}

int sparc_gpu_get_info(const sparc_gpu_ctx *ctx, const char *key, int64_t *value)
{
    if (!ctx || !key || !value) return SPARC_GPU_INVALID_ARG;
    if (!strcmp(key, "kernel_launches")) { *value = ctx->kernel_launches; return 0; }
    if (!strcmp(key, "nd")) { *value = ctx->nd; return 0; }
    if (!strcmp(key, "n_proj_total")) { *value = ctx->n_proj_total; return 0; }
    if (!strcmp(key, "covered_points")) { *value = ctx->n_covered; return 0; }
    if (!strcmp(key, "stencil_path_last")) { *value = ctx->stencil_path_last; return 0; }
    if (!strcmp(key, "sm_count")) { *value = ctx->sm_count; return 0; }
    if (!strcmp(key, "gemm_tn_mflop")) { *value = (int64_t)(ctx->gemm_flop[0] / 1e6); return 0; }
    if (!strcmp(key, "gemm_nn_mflop")) { *value = (int64_t)(ctx->gemm_flop[1] / 1e6); return 0; }
    if (!strcmp(key, "nl_brick")) { *value = ctx->nlb.ok; return 0; }
    if (!strcmp(key, "nl_brick_blocks")) { *value = ctx->nlb.n_blocks; return 0; }
    if (!strcmp(key, "nl_brick_active")) { *value = ctx->nlb.n_active; return 0; }
    if (!strcmp(key, "nl_brick_max_blocks")) { *value = ctx->nlb.max_blocks; return 0; }
    if (!strcmp(key, "nl_brick_max_jobs")) { *value = ctx->nlb.max_jobs; return 0; }
    if (!strncmp(key, "prof_ns:", 8) || !strncmp(key, "prof_count:", 11)) {
        if (!ctx->prof) return SPARC_GPU_OUT_OF_MEMORY;
        const bool is_ns = key[5] == 'n';
        const int kind = atoi(key + (is_ns ? 8 : 11));
        if (kind < 0 || kind >= KK_COUNT) return SPARC_GPU_INVALID_ARG;
        if (is_ns) { prof_collect(ctx->prof); *value = (int64_t)ctx->prof->ns[kind]; }
        else *value = ctx->prof->count[kind];
        return 0;
    }
    return SPARC_GPU_INVALID_ARG;
}

int sparc_gpu_set_workspace_size(sparc_gpu_ctx *ctx, int64_t bytes)
{
    if (!ctx || bytes < 0) return SPARC_GPU_INVALID_ARG;
    ctx->ws_bytes = bytes;
    return SPARC_GPU_SUCCESS;
}

int sparc_gpu_workspace_bytes(const sparc_gpu_ctx *ctx, int op, int64_t ns, int64_t block, int64_t *bytes)
{
    if (!ctx || !bytes) return SPARC_GPU_INVALID_ARG;
    WsLayout L;
    SPARC_TRY(ws_layout(ctx, op, ns, block, &L));
    *bytes = L.total;
    return SPARC_GPU_SUCCESS;
}

int sparc_gpu_hamiltonian_apply(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, double *Y, int64_t ldy,
                                int64_t ncols, void *ws, void *stream)
{
    if (!ctx || ncols < 0) return SPARC_GPU_INVALID_ARG;
    if (ncols == 0) return SPARC_GPU_SUCCESS;
    if (!X || !Y || !ws || ldx < ctx->nd || ldy < ctx->nd) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    WsLayout L;
    SPARC_TRY(ws_layout(ctx, SPARC_GPU_OP_HAMILTONIAN_APPLY, ncols, 0, &L));
    SPARC_TRY(ws_check(ctx, L));
    double *D = (double *)((char *)ws + L.off_d);
    for (int64_t j0 = 0; j0 < ncols; j0 += L.block) {
        const int64_t nb = std::min(L.block, ncols - j0);
        SPARC_TRY(h_apply_block(ctx, X + j0 * ldx, ldx, Y + j0 * ldy, ldy, nb, D, (cudaStream_t)stream));
    }
    return SPARC_GPU_SUCCESS;
}

int sparc_gpu_chebyshev_filter(sparc_gpu_ctx *ctx, double *Psi, int64_t ld, int64_t ns, int degree, double a,
                               double b, double a0, int64_t col_block, void *ws, void *stream)
{
    if (!ctx || ns < 0 || degree < 0) return SPARC_GPU_INVALID_ARG;
    if (!(a0 < a && a < b)) return SPARC_GPU_BAD_BOUNDS;
    if (ns == 0 || degree == 0) return SPARC_GPU_SUCCESS;
    if (!Psi || !ws || ld < ctx->nd) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    cudaStream_t st = (cudaStream_t)stream;
    WsLayout L;
    SPARC_TRY(ws_layout(ctx, SPARC_GPU_OP_CHEBYSHEV_FILTER, ns, col_block, &L));
    SPARC_TRY(ws_check(ctx, L));
    double *W = (double *)((char *)ws + L.off_w);
    double *D = (double *)((char *)ws + L.off_d);
    const double e = 0.5 * (b - a), c = 0.5 * (b + a);
    const double sigma1 = e / (a0 - c), tau = 2.0 / sigma1;
    for (int64_t j0 = 0; j0 < ns; j0 += L.block) {
        const int64_t nb = std::min(L.block, ns - j0);
        double *bufA = Psi + j0 * ld;     // holds Y_{k-1} (k odd) / Y_k (k even)
        double *cur = bufA, *oth = W;
        int64_t ldc = ld, ldo = L.ldw;
        // one degree step: oth <- alpha (H cur - c cur) + beta oth.  With the brick kernel the nonlocal term of step k
        // and the projection chi^T Psi_k needed by step k + 1 share one read-modify-write of oth.
        const int mode = effective_nl_mode(ctx, cur, ldc, oth, ldo);
        const size_t cbytes = (size_t)nlb_c_doubles(ctx, nb) * 8;
        double *Cb[2] = {D, D + nlb_c_doubles(ctx, nb)};
        if (mode == 3) {     // D_0 = alpha_1 Gamma chi^T Psi_0: the projection folds in the alpha of the step that pulls it
            SPARC_CUDA_TRY(cudaMemsetAsync(Cb[0], 0, cbytes, st));
            SPARC_TRY(launch_nl_brick(ctx, 1, cur, ldc, nb, sigma1 / e, nullptr, Cb[0], st));
        }
        double sigma = sigma1;
        for (int k = 1; k <= degree; ++k) {
            const double sigma2 = 1.0 / (tau - sigma);
            const double alpha = (k == 1) ? sigma1 / e : 2.0 * sigma2 / e;
            const double beta = (k == 1) ? 0.0 : -(sigma * sigma2);
            SPARC_TRY(local_pass(ctx, cur, ldc, oth, ldo, k == 1 ? nullptr : oth, ldo, nb, alpha, -c, beta, st));
            if (mode == 3) {
                const bool last = (k == degree);
                if (!last) SPARC_CUDA_TRY(cudaMemsetAsync(Cb[k & 1], 0, cbytes, st));
                // alpha_{k+1} = 2 sigma_{k+1} / e, sigma_{k+1} = 1 / (tau - sigma_k), sigma_k = sigma1 (k = 1) or sigma2
                const double alpha_next = 2.0 / (tau - (k == 1 ? sigma1 : sigma2)) / e;
                SPARC_TRY(launch_nl_brick(ctx, last ? 2 : 3, oth, ldo, nb, alpha_next, Cb[(k - 1) & 1], Cb[k & 1], st));
            } else if (mode > 0) {
                SPARC_TRY(nl_pass_per_atom(ctx, mode, cur, ldc, oth, ldo, nb, alpha, D, st));
            }
            if (k > 1) sigma = sigma2;
            std::swap(cur, oth); std::swap(ldc, ldo);
        }
        if (cur != bufA) SPARC_TRY(launch_copy_2d(ctx, bufA, ld, cur, ldc, ctx->nd, nb, st));
    }
    return SPARC_GPU_SUCCESS;
}

int sparc_gpu_project(sparc_gpu_ctx *ctx, const double *Psi, int64_t ld, int64_t ns, double *Hs, double *Ms,
                      int64_t col_block, void *ws, void *stream)
{
    if (!ctx || ns < 0) return SPARC_GPU_INVALID_ARG;
    if (ns == 0) return SPARC_GPU_SUCCESS;
    if (!Psi || !Hs || !Ms || !ws || ld < ctx->nd) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    cudaStream_t st = (cudaStream_t)stream;
    WsLayout L;
    SPARC_TRY(ws_layout(ctx, SPARC_GPU_OP_PROJECT, ns, col_block, &L));
    SPARC_TRY(ws_check(ctx, L));
    double *Y = (double *)((char *)ws + L.off_w);
    double *D = (double *)((char *)ws + L.off_d);
    void *G = (char *)ws + L.off_g;
    // Hs and Ms are symmetric (H is): only tiles at or above the diagonal are computed, then mirrored (reading R12)
    const bool sym = ctx->opt_gemm_full == 0;
    for (int64_t j0 = 0; j0 < ns; j0 += L.block) {
        const int64_t nb = std::min(L.block, ns - j0);
        SPARC_TRY(h_apply_block(ctx, Psi + j0 * ld, ld, Y, L.ldw, nb, D, st));
        // Hs[:, j0:j0+nb] = Psi^T Y_block
        SPARC_TRY(launch_gemm_tn(ctx, Psi, ld, Y, L.ldw, Hs + j0 * ns, ns, ns, nb, ctx->nd, G, sym ? j0 : -1, st));
    }
    SPARC_TRY(launch_gemm_tn(ctx, Psi, ld, Psi, ld, Ms, ns, ns, ns, ctx->nd, G, sym ? 0 : -1, st));
    if (sym) {
        SPARC_TRY(launch_mirror_upper(ctx, Hs, ns, ns, st));
        SPARC_TRY(launch_mirror_upper(ctx, Ms, ns, ns, st));
    }
    return SPARC_GPU_SUCCESS;
}

int sparc_gpu_rotate(sparc_gpu_ctx *ctx, double *Psi, int64_t ld, int64_t ns, const double *Q, int64_t row_panel,
                     void *ws, void *stream)
{
    if (!ctx || ns < 0) return SPARC_GPU_INVALID_ARG;
    if (ns == 0) return SPARC_GPU_SUCCESS;
    if (!Psi || !Q || !ws || ld < ctx->nd) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    cudaStream_t st = (cudaStream_t)stream;
    WsLayout L;
    SPARC_TRY(ws_layout(ctx, SPARC_GPU_OP_ROTATE, ns, row_panel, &L));
    SPARC_TRY(ws_check(ctx, L));
    double *T = (double *)((char *)ws + L.off_w);
    for (int64_t r0 = 0; r0 < ctx->nd; r0 += L.block) {
        const int64_t nr = std::min(L.block, ctx->nd - r0);
        SPARC_TRY(rotate_panel(ctx, Psi + r0, ld, nr, ns, Q, T, L.ldw, st));
    }
    return SPARC_GPU_SUCCESS;
}

// ---- building blocks of the row-partitioned (multi-GPU) projection and rotation, SURVEY.md section 8(f) NEXT-2 -------------

int sparc_gpu_gram(sparc_gpu_ctx *ctx, const double *A, int64_t lda, const double *B, int64_t ldb, int64_t nrows, int64_t m,
                   int64_t n, double *C, int symmetric, void *ws, void *stream)
{
    if (!ctx || nrows < 0 || m < 0 || n < 0) return SPARC_GPU_INVALID_ARG;
    if (m == 0 || n == 0) return SPARC_GPU_SUCCESS;
    if (!C || (symmetric && m != n)) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    cudaStream_t st = (cudaStream_t)stream;
    // a rank that owns no rows passes empty blocks (NULL data pointers, no workspace): its contribution is C = 0, as
    // sparc_gpu_rotate_rows treats nrows = 0 as a no-op
    if (nrows == 0) { SPARC_CUDA_TRY(cudaMemsetAsync(C, 0, (size_t)m * n * 8, st)); return SPARC_GPU_SUCCESS; }
    if (!A || !B || !ws || lda < nrows || ldb < nrows) return SPARC_GPU_INVALID_ARG;
    WsLayout L;
    SPARC_TRY(ws_layout(ctx, SPARC_GPU_OP_GRAM, std::max(m, n), 0, &L));
    SPARC_TRY(ws_check(ctx, L));
    const bool sym = symmetric && ctx->opt_gemm_full == 0;
    SPARC_TRY(launch_gemm_tn(ctx, A, lda, B, ldb, C, m, m, n, nrows, (char *)ws + L.off_g, sym ? 0 : -1, st));
    if (sym) SPARC_TRY(launch_mirror_upper(ctx, C, m, m, st));
    return SPARC_GPU_SUCCESS;
}

int sparc_gpu_rotate_rows(sparc_gpu_ctx *ctx, double *X, int64_t ld, int64_t nrows, int64_t ns, const double *Q,
                          int64_t row_panel, void *ws, void *stream)
{
    if (!ctx || ns < 0 || nrows < 0) return SPARC_GPU_INVALID_ARG;
    if (ns == 0 || nrows == 0) return SPARC_GPU_SUCCESS;
    if (!X || !Q || !ws || ld < nrows) return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    int64_t rp = 0, ldw = 0;
    SPARC_TRY(rotate_layout(ctx, ns, row_panel, &rp, &ldw));
    for (int64_t r0 = 0; r0 < nrows; r0 += rp) {
        const int64_t nr = std::min(rp, nrows - r0);
        SPARC_TRY(rotate_panel(ctx, X + r0, ld, nr, ns, Q, (double *)ws, ldw, (cudaStream_t)stream));
    }
    return SPARC_GPU_SUCCESS;
}

}  // extern "C"
