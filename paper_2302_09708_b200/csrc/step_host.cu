// step_host.cu -- the whole CheFSI step for a caller whose orbitals live in HOST memory (the situation of the paper's
// implementation, which stages X, H~, M~, Z~ through the host around every step: PAPER.md:118, 128, 138, 146, 158, 166).
// Plumbing only: the arithmetic is the same operator calls as the device-resident path; what this file adds is the
// overlap of the PCIe copies with them.
//
//   columns in  : Psi_host -> Psi_dev by column chunks on a copy stream; the filter of chunk j (independent columns,
//                 PAPER.md:120) runs while chunk j + 1 is in flight
//   project     : Hs, Ms -> host as soon as they are complete (copy stream)
//   rotate      : row panel by row panel; the rows of a finished panel leave for the host (2-D copy)
//                 while the next panel is multiplied
#include <algorithm>
#include <vector>

#include "internal.h"

namespace {

struct EventPool {
    std::vector<cudaEvent_t> ev;
    ~EventPool() { for (auto e : ev) cudaEventDestroy(e); }
    cudaEvent_t get()
    {
        cudaEvent_t e = nullptr;
        if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
        ev.push_back(e);
        return e;
    }
};

// Whatever way the call ends, nothing of it is still in flight afterwards: an early error return would otherwise leave
// async copies into the caller's host buffers (and kernels on three streams) running while the events are destroyed.
struct SyncOnExit {
    cudaStream_t s[3];
    ~SyncOnExit() { for (auto q : s) if (cudaStreamSynchronize(q) != cudaSuccess) (void)cudaGetLastError(); }
};

// Q_host != NULL: rotate by the caller's Q.  Q_host == NULL: Algorithm 1 as written -- the subspace
// eigenproblem Hs Z = Ms Z D is solved on the device between projection and rotation, D and info go to the host.
int step_host_impl(sparc_gpu_ctx *ctx, const double *Psi_in_host, double *Psi_out_host, int64_t ld_host, int64_t ns, int degree,
                   double a, double b, double a0, const double *Q_host, double *D_host, int32_t *info_host, double *Hs_host,
                   double *Ms_host, double *Psi_dev, int64_t ld_dev, double *mats_dev, int64_t col_block, int64_t row_panel,
                   void *ws_dev, void *stream)
{
    const bool solve = Q_host == nullptr;
    if (!ctx || ns < 0 || degree < 0) return SPARC_GPU_INVALID_ARG;
    if (!(a0 < a && a < b)) return SPARC_GPU_BAD_BOUNDS;
    if (ns == 0) return SPARC_GPU_SUCCESS;
    if (!Psi_in_host || !Psi_out_host || !Hs_host || !Ms_host || !Psi_dev || !mats_dev || !ws_dev ||
        ld_host < ctx->nd || ld_dev < ctx->nd || (solve && (!D_host || !info_host)))
        return SPARC_GPU_INVALID_ARG;
    DeviceGuard dg(ctx->device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    cudaStream_t st = (cudaStream_t)stream;
    if (!ctx->copy_stream[0] || !ctx->copy_stream[1]) {          // both or neither: a half-made pair is never kept
        cudaStream_t s0 = nullptr, s1 = nullptr;
        SPARC_CUDA_TRY(cudaStreamCreateWithFlags(&s0, cudaStreamNonBlocking));
        const cudaError_t e1 = cudaStreamCreateWithFlags(&s1, cudaStreamNonBlocking);
        if (e1 != cudaSuccess) { (void)cudaGetLastError(); (void)cudaStreamDestroy(s0); return SPARC_GPU_CUDA_ERROR; }
        ctx->copy_stream[0] = s0;
        ctx->copy_stream[1] = s1;
    }
    cudaStream_t s_in = ctx->copy_stream[0], s_out = ctx->copy_stream[1];
    EventPool pool;                      // destroyed after `drain` below has synchronised the three streams
    SyncOnExit drain{{st, s_in, s_out}};
    const int64_t nd = ctx->nd;
    double *Hs_dev = mats_dev, *Ms_dev = mats_dev + ns * ns, *Q_dev = mats_dev + 2 * ns * ns;
    double *D_dev = mats_dev + 3 * ns * ns;                      // solve only: D[ns], then 2 x int32 info
    int32_t *info_dev = (int32_t *)(D_dev + ns);

    // the copy streams start after whatever the caller queued on `stream`
    cudaEvent_t ev0 = pool.get();
    if (!ev0) return SPARC_GPU_CUDA_ERROR;
    SPARC_CUDA_TRY(cudaEventRecord(ev0, st));
    SPARC_CUDA_TRY(cudaStreamWaitEvent(s_in, ev0, 0));
    SPARC_CUDA_TRY(cudaStreamWaitEvent(s_out, ev0, 0));

    // ---- columns in, filter ----------------------------------------------------------------------------------------
    int64_t blk = 0;
    {
        int64_t bytes = 0;   // (validates ns / col_block the same way the filter call will)
        SPARC_TRY(sparc_gpu_workspace_bytes(ctx, SPARC_GPU_OP_CHEBYSHEV_FILTER, ns, col_block, &bytes));
        blk = col_block > 0 ? std::min(col_block, ns) : std::min<int64_t>(ns, 1024);
        // a block that fits one chunk is cut into up to four chunks of at least 64 columns, so that copies and kernels overlap
        if (blk >= ns) blk = std::max<int64_t>(std::min<int64_t>(ns, 64), (ns + 3) / 4);
    }
    for (int64_t j0 = 0; j0 < ns; j0 += blk) {
        const int64_t nb = std::min(blk, ns - j0);
        SPARC_CUDA_TRY(cudaMemcpy2DAsync(Psi_dev + j0 * ld_dev, (size_t)ld_dev * 8, Psi_in_host + j0 * ld_host,
                                         (size_t)ld_host * 8, (size_t)nd * 8, (size_t)nb, cudaMemcpyHostToDevice, s_in));
        cudaEvent_t e = pool.get();
        if (!e) return SPARC_GPU_CUDA_ERROR;
        SPARC_CUDA_TRY(cudaEventRecord(e, s_in));
        SPARC_CUDA_TRY(cudaStreamWaitEvent(st, e, 0));
        SPARC_TRY(sparc_gpu_chebyshev_filter(ctx, Psi_dev + j0 * ld_dev, ld_dev, nb, degree, a, b, a0, col_block, ws_dev, st));
    }
    cudaEvent_t ev_q = nullptr;
    if (!solve) {                        // Q rides behind the columns
        SPARC_CUDA_TRY(cudaMemcpyAsync(Q_dev, Q_host, (size_t)ns * ns * 8, cudaMemcpyHostToDevice, s_in));
        ev_q = pool.get();
        if (!ev_q) return SPARC_GPU_CUDA_ERROR;
        SPARC_CUDA_TRY(cudaEventRecord(ev_q, s_in));
    }

    // ---- project; Hs, Ms out -----------------------------------------------------------------------------------------
    SPARC_TRY(sparc_gpu_project(ctx, Psi_dev, ld_dev, ns, Hs_dev, Ms_dev, col_block, ws_dev, st));
    cudaEvent_t ev_p = pool.get();
    if (!ev_p) return SPARC_GPU_CUDA_ERROR;
    SPARC_CUDA_TRY(cudaEventRecord(ev_p, st));
    SPARC_CUDA_TRY(cudaStreamWaitEvent(s_out, ev_p, 0));
    SPARC_CUDA_TRY(cudaMemcpyAsync(Hs_host, Hs_dev, (size_t)ns * ns * 8, cudaMemcpyDeviceToHost, s_out));
    SPARC_CUDA_TRY(cudaMemcpyAsync(Ms_host, Ms_dev, (size_t)ns * ns * 8, cudaMemcpyDeviceToHost, s_out));

    // ---- solve (Q_host == NULL): Z -> Q_dev, D and info -> host; the one point where the host waits mid-step, because a
    // pencil whose Ms is not positive definite must not be rotated by what the solver left in Z
    bool rotate = true;
    if (solve) {
        SPARC_TRY(sparc_gpu_eigensolve(ctx, ns, Hs_dev, Ms_dev, Q_dev, D_dev, info_dev, ws_dev, st));
        cudaEvent_t ev_s = pool.get();
        if (!ev_s) return SPARC_GPU_CUDA_ERROR;
        SPARC_CUDA_TRY(cudaEventRecord(ev_s, st));
        SPARC_CUDA_TRY(cudaStreamWaitEvent(s_out, ev_s, 0));
        SPARC_CUDA_TRY(cudaMemcpyAsync(D_host, D_dev, (size_t)ns * 8, cudaMemcpyDeviceToHost, s_out));
        SPARC_CUDA_TRY(cudaMemcpyAsync(info_host, info_dev, 2 * sizeof(int32_t), cudaMemcpyDeviceToHost, s_out));
        SPARC_CUDA_TRY(cudaStreamSynchronize(s_out));
        rotate = info_host[0] != 1;
    } else {
        SPARC_CUDA_TRY(cudaStreamWaitEvent(st, ev_q, 0));
    }

    // ---- rotate by row panels; finished rows out -----------------------------------------------------------------------
    int64_t rp = 0, ldw = 0;
    SPARC_TRY(rotate_layout(ctx, ns, row_panel, &rp, &ldw));
    for (int64_t r0 = 0; r0 < nd; r0 += rp) {
        const int64_t nr = std::min(rp, nd - r0);
        if (rotate) SPARC_TRY(rotate_panel(ctx, Psi_dev + r0, ld_dev, nr, ns, Q_dev, (double *)ws_dev, ldw, st));
        cudaEvent_t e = pool.get();
        if (!e) return SPARC_GPU_CUDA_ERROR;
        SPARC_CUDA_TRY(cudaEventRecord(e, st));
        SPARC_CUDA_TRY(cudaStreamWaitEvent(s_out, e, 0));
        SPARC_CUDA_TRY(cudaMemcpy2DAsync(Psi_out_host + r0, (size_t)ld_host * 8, Psi_dev + r0, (size_t)ld_dev * 8,
                                         (size_t)nr * 8, (size_t)ns, cudaMemcpyDeviceToHost, s_out));
    }
    SPARC_CUDA_TRY(cudaStreamSynchronize(s_out));
    SPARC_CUDA_TRY(cudaStreamSynchronize(s_in));
    SPARC_CUDA_TRY(cudaStreamSynchronize(st));
    return SPARC_GPU_SUCCESS;
}

}  // namespace

extern "C" int sparc_gpu_chefsi_step_host(sparc_gpu_ctx *ctx, const double *Psi_in_host, double *Psi_out_host,
                                          int64_t ld_host, int64_t ns, int degree, double a, double b, double a0,
                                          const double *Q_host, double *Hs_host, double *Ms_host, double *Psi_dev,
                                          int64_t ld_dev, double *mats_dev, int64_t col_block, int64_t row_panel,
                                          void *ws_dev, void *stream)
{
    if (ns > 0 && !Q_host) return SPARC_GPU_INVALID_ARG;        // the solving variant is sparc_gpu_chefsi_step_host_solve
    return step_host_impl(ctx, Psi_in_host, Psi_out_host, ld_host, ns, degree, a, b, a0, Q_host, nullptr, nullptr, Hs_host,
                          Ms_host, Psi_dev, ld_dev, mats_dev, col_block, row_panel, ws_dev, stream);
}

extern "C" int sparc_gpu_chefsi_step_host_solve(sparc_gpu_ctx *ctx, const double *Psi_in_host, double *Psi_out_host,
                                                int64_t ld_host, int64_t ns, int degree, double a, double b, double a0,
                                                double *D_host, int32_t *info_host, double *Hs_host, double *Ms_host,
                                                double *Psi_dev, int64_t ld_dev, double *mats_dev, int64_t col_block,
                                                int64_t row_panel, void *ws_dev, void *stream)
{
    return step_host_impl(ctx, Psi_in_host, Psi_out_host, ld_host, ns, degree, a, b, a0, nullptr, D_host, info_host, Hs_host,
                          Ms_host, Psi_dev, ld_dev, mats_dev, col_block, row_panel, ws_dev, stream);
}
