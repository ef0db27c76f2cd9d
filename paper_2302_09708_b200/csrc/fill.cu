// fill.cu -- device restatement of the workloads' counter-based uniform generator:
//   key = mix64(seed*C_SEED + stream*C_STREAM + GOLDEN);  u = (mix64(key + GOLDEN*index) >> 11) * 2^-53
// Input generation only (not an operator of the method): lets an 82 GB Psi be created in HBM directly.
#include "internal.h"

namespace {

__host__ __device__ inline uint64_t mix64(uint64_t z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

__global__ void __launch_bounds__(256)
fill_uniform_kernel(double *dst, int64_t count, uint64_t key, uint64_t index0, double lo, double span)
{
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < count; k += (int64_t)gridDim.x * blockDim.x) {
        const uint64_t z = mix64(key + 0x9E3779B97F4A7C15ULL * (index0 + (uint64_t)k));
        dst[k] = lo + span * ((double)(z >> 11) * (1.0 / 9007199254740992.0));
    }
}

}  // namespace

extern "C" int sparc_gpu_fill_uniform(double *dst_dev, int64_t count, uint64_t seed, uint64_t stream_id,
                                      uint64_t index0, double lo, double hi, int device, void *stream)
{
    if (count < 0 || (count > 0 && !dst_dev)) return SPARC_GPU_INVALID_ARG;
    if (count == 0) return SPARC_GPU_SUCCESS;
    DeviceGuard dg(device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    const uint64_t key = mix64(seed * 0xD1B54A32D192ED03ULL + stream_id * 0x8CB92BA72F3D8DD7ULL + 0x9E3779B97F4A7C15ULL);
    int64_t blocks = (count + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    fill_uniform_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(dst_dev, count, key, index0, lo, hi - lo);
    SPARC_CUDA_TRY(cudaGetLastError());
    return SPARC_GPU_SUCCESS;
}
