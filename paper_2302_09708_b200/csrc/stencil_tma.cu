// stencil_tma.cu -- placeholder until the TMA-tiled kernel lands (next commit).
#include "internal.h"

bool stencil_tma_supported(const sparc_gpu_ctx *, const double *, int64_t, const double *, int64_t, const double *, int64_t)
{
    return false;
}

int launch_stencil_tma(sparc_gpu_ctx *, const double *, int64_t, double *, int64_t, const double *, int64_t, int64_t,
                       double, double, double, cudaStream_t)
{
    return SPARC_GPU_UNSUPPORTED;
}
