// peaks.cu -- register-resident FP64 throughput probes: the roofline denominators of the FP64-bound kernels
// ("FP64 DMMA peak measured on the box by a register-resident DMMA microbenchmark").
// Not an operator of the method.  kind 0: independent DFMA chains; kind 1: independent DMMA.8x8x4 chains
// (mma.sync.m8n8k4.f64 -- on sm_100a every PTX f64 mma shape lowers to it); kind 2: device-to-device copy GB/s.
#include "internal.h"

namespace {

constexpr int PROBE_THREADS = 256;
constexpr int PROBE_CHAINS = 16;

__global__ void __launch_bounds__(PROBE_THREADS)
probe_dfma_kernel(double *sink, int iters, double a, double b)
{
    double acc[PROBE_CHAINS];
#pragma unroll
    for (int k = 0; k < PROBE_CHAINS; ++k) acc[k] = (double)(threadIdx.x + k);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < PROBE_CHAINS; ++k) acc[k] = fma(acc[k], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < PROBE_CHAINS; ++k) s += acc[k];
    if (s == 12345.678) sink[0] = s;        // never true for the probe's constants; keeps the chains alive
}

__global__ void __launch_bounds__(PROBE_THREADS)
probe_dmma_kernel(double *sink, int iters, double a, double b)
{
    double c0[PROBE_CHAINS], c1[PROBE_CHAINS];
#pragma unroll
    for (int k = 0; k < PROBE_CHAINS; ++k) { c0[k] = (double)k; c1[k] = (double)threadIdx.x; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < PROBE_CHAINS; ++k)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(c0[k]), "+d"(c1[k])
                         : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < PROBE_CHAINS; ++k) s += c0[k] + c1[k];
    if (s == 12345.678) sink[0] = s;
}

__global__ void __launch_bounds__(256)
probe_copy_kernel(double2 *dst, const double2 *src, int64_t n)
{
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x)
        dst[k] = src[k];
}

}  // namespace

extern "C" int sparc_gpu_probe_peak(int device, int kind, double *value_out, void *scratch_dev, int64_t scratch_bytes,
                                    void *stream)
{
    if (!value_out || kind < 0 || kind > 2) return SPARC_GPU_INVALID_ARG;
    if (!scratch_dev || scratch_bytes < 64) return SPARC_GPU_WORKSPACE_TOO_SMALL;
    DeviceGuard dg(device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    cudaDeviceProp prop;
    SPARC_CUDA_TRY(cudaGetDeviceProperties(&prop, device));
    if (prop.major != 10) return SPARC_GPU_UNSUPPORTED;
    cudaStream_t st = (cudaStream_t)stream;
    cudaEvent_t e0, e1;
    SPARC_CUDA_TRY(cudaEventCreate(&e0));
    SPARC_CUDA_TRY(cudaEventCreate(&e1));
    const int sms = prop.multiProcessorCount;
    double best = 0.0;
    int status = SPARC_GPU_SUCCESS;
    for (int rep = 0; rep < 5 && status == SPARC_GPU_SUCCESS; ++rep) {       // rep 0 is the warm-up
        double work = 0.0;                                                   // flop or bytes
        cudaEventRecord(e0, st);
        if (kind == 0) {
            const int iters = 1 << 14, grid = sms * 8;
            probe_dfma_kernel<<<grid, PROBE_THREADS, 0, st>>>((double *)scratch_dev, iters, 0.999999, 1e-9);
            work = 2.0 * PROBE_CHAINS * (double)iters * PROBE_THREADS * grid;
        } else if (kind == 1) {
            const int iters = 1 << 12, grid = sms * 8;
            probe_dmma_kernel<<<grid, PROBE_THREADS, 0, st>>>((double *)scratch_dev, iters, 0.5, 1e-9);
            work = 2.0 * 256.0 * PROBE_CHAINS * (double)iters * (PROBE_THREADS / 32) * grid;
        } else {
            const int64_t n = scratch_bytes / 32;                            // double2 elements per half
            probe_copy_kernel<<<sms * 16, 256, 0, st>>>((double2 *)scratch_dev + n, (const double2 *)scratch_dev, n);
            work = 2.0 * 16.0 * (double)n;
        }
        cudaEventRecord(e1, st);
        if (cudaGetLastError() != cudaSuccess || cudaEventSynchronize(e1) != cudaSuccess) { status = SPARC_GPU_CUDA_ERROR; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms > 0.f) best = best > work / (ms * 1e-3) ? best : work / (ms * 1e-3);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    (void)cudaGetLastError();
    *value_out = (kind == 2) ? best / 1e9 : best / 1e12;                     // GB/s or TFLOP/s
    return status;
}
