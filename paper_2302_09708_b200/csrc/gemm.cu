// gemm.cu -- FP64 tensor-core (DMMA m8n8k4) tiled GEMMs for the subspace steps:
//   TN:  C = A^T B  with the contraction over the N_d grid rows   (Hs = Psi^T Y, Ms = Psi^T Psi)
//   NN:  C = A B    row panel of Psi times Q                      (X = X~ Z~)
// On sm_100a every PTX f64 mma.sync shape lowers to DMMA.8x8x4, so m8n8k4 is used directly.  Operands are
// staged global -> shared with cp.async (double-buffered 32-deep k-tiles), fragments are read with conflict-free LDS.64 (row pitch
// == 4 mod 16 doubles).  tcgen05/TMEM have no f64 kind and do not apply here.
// Small-output TN products (N_s = 32, 256) are split over K across the chip and reduced in a fixed order
// (deterministic).
#include <algorithm>
#include <mutex>

#include "internal.h"

namespace {

// BK = 32 with a double buffer (round 2): half as many barriers per DMMA as BK = 16 x 3 stages, same 2 CTAs per SM
// (110 KB of shared memory each): 32.7 -> 33.4 TFLOP/s at config 3
constexpr int BM = 128, BK = 32, STAGES = 2;
// CTA tile 128 x (32 NWN): 2 x NWN warps of 64 x 32.  NWN = 2 (128 x 64, 128 threads) lets two CTAs share an SM so that
// one CTA's pipeline barriers are covered by the other's DMMAs; NWN = 4 is the 128 x 128 tile.
constexpr int NWN_DEFAULT = 2;
constexpr int PITCH_K = BK + 4;     // rows of BK doubles (k contiguous)
constexpr int PITCH_M = BM + 4;     // rows of BM doubles (m contiguous)

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem, int src_bytes)
{
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async8(void *smem, const void *gmem, int src_bytes)
{
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

constexpr size_t smem_bytes(bool a_mmajor, int nwn)
{
    return (size_t)STAGES * ((a_mmajor ? BK * PITCH_M : BM * PITCH_K) + 32 * nwn * PITCH_K) * sizeof(double);
}

// Load a tile whose contiguous global direction is "inner" (length INNER doubles per row, ROWS rows).
// Global element (inner i, row r) lives at g[i + r*ld]; rows beyond `rows_valid` and inner beyond
// `inner_valid` are zero-filled.  Shared layout: s[r*PITCH + i].
template <int ROWS, int INNER, int PITCH, bool VEC16, int GEMM_THREADS>
__device__ __forceinline__ void load_tile(double *s, const double *g, int64_t ld, int64_t rows_valid,
                                          int64_t inner_valid, int tid)
{
    if (VEC16) {
        constexpr int CH = INNER / 2;
        for (int c = tid; c < ROWS * CH; c += GEMM_THREADS) {
            const int r = c / CH, i = (c % CH) * 2;
            int bytes = 0;
            if (r < rows_valid) bytes = (i + 1 < inner_valid) ? 16 : ((i < inner_valid) ? 8 : 0);
            const double *src = bytes ? g + i + (int64_t)r * ld : g;
            cp_async16(s + r * PITCH + i, src, bytes);
        }
    } else {
        for (int c = tid; c < ROWS * INNER; c += GEMM_THREADS) {
            const int r = c / INNER, i = c % INNER;
            const int bytes = (r < rows_valid && i < inner_valid) ? 8 : 0;
            const double *src = bytes ? g + i + (int64_t)r * ld : g;
            cp_async8(s + r * PITCH + i, src, bytes);
        }
    }
}

// A_MMAJOR = false: A is K x M col-major (A[k + m*lda]) -> C = A^T B           (TN)
// A_MMAJOR = true : A is M x K col-major (A[m + k*lda]) -> C = A B             (NN)
// B is always K x N col-major (B[k + n*ldb]).  C is M x N col-major; with splits > 1, blockIdx.z writes its
// partial product to Cpart + z*M*N (ld = M).
template <bool A_MMAJOR, bool VEC16, int NWN>
__global__ void __launch_bounds__(64 * NWN, NWN == 2 ? 2 : 1)
gemm_dmma_kernel(const double *__restrict__ A, int64_t lda, const double *__restrict__ B, int64_t ldb, double *C,
                 int64_t ldc, int64_t M, int64_t N, int64_t K, int64_t k_chunk, int tiles_m, int64_t diag)
{
    extern __shared__ __align__(16) double smem[];
    constexpr int BN = 32 * NWN, GEMM_THREADS = 64 * NWN;
    constexpr int A_STAGE = A_MMAJOR ? BK * PITCH_M : BM * PITCH_K;
    constexpr int B_STAGE = BN * PITCH_K;
    double *As = smem;
    double *Bs = smem + STAGES * A_STAGE;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp / NWN, wn = warp % NWN;       // 2 x NWN warps, warp tile 64 x 32
    const int tile_m = blockIdx.x % tiles_m, tile_n = blockIdx.x / tiles_m;
    const int64_t m0 = (int64_t)tile_m * BM, n0 = (int64_t)tile_n * BN;
    // symmetric result (diag >= 0: global column index of column 0): tiles strictly below the diagonal are skipped,
    // the caller mirrors the upper triangle afterwards
    if (diag >= 0 && m0 >= diag + n0 + BN) return;
    const int64_t k_begin = (int64_t)blockIdx.z * k_chunk;
    const int64_t k_end = (k_begin + k_chunk < K) ? k_begin + k_chunk : K;
    if (gridDim.z > 1) { C += (int64_t)blockIdx.z * M * N; ldc = M; }
    const int nkt = (k_end > k_begin) ? (int)((k_end - k_begin + BK - 1) / BK) : 0;

    double acc[8][4][2];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    auto issue = [&](int kt) {
        const int s = kt % STAGES;
        const int64_t k0 = k_begin + (int64_t)kt * BK;
        const int64_t kv = k_end - k0;      // valid k in this tile (may exceed BK)
        if (A_MMAJOR)
            load_tile<BK, BM, PITCH_M, VEC16, GEMM_THREADS>(As + s * A_STAGE, A + m0 + k0 * lda, lda, kv, M - m0, tid);
        else
            load_tile<BM, BK, PITCH_K, VEC16, GEMM_THREADS>(As + s * A_STAGE, A + k0 + m0 * lda, lda, M - m0, kv, tid);
        load_tile<BN, BK, PITCH_K, VEC16, GEMM_THREADS>(Bs + s * B_STAGE, B + k0 + n0 * ldb, ldb, N - n0, kv, tid);
    };

#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nkt) issue(s);
        cp_async_commit();
    }
    const int lr = lane >> 2, lk = lane & 3;
    for (int kt = 0; kt < nkt; ++kt) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        if (kt + STAGES - 1 < nkt) issue(kt + STAGES - 1);
        cp_async_commit();
        const double *as = As + (kt % STAGES) * A_STAGE;
        const double *bs = Bs + (kt % STAGES) * B_STAGE;
#pragma unroll
        for (int kk = 0; kk < BK; kk += 4) {
            double a[8], b[4];
#pragma unroll
            for (int mi = 0; mi < 8; ++mi) {
                const int m = wm * 64 + mi * 8 + lr;
                a[mi] = A_MMAJOR ? as[(kk + lk) * PITCH_M + m] : as[m * PITCH_K + kk + lk];
            }
#pragma unroll
            for (int ni = 0; ni < 4; ++ni) b[ni] = bs[(wn * 32 + ni * 8 + lr) * PITCH_K + kk + lk];
#pragma unroll
            for (int mi = 0; mi < 8; ++mi)
#pragma unroll
                for (int ni = 0; ni < 4; ++ni) dmma884(acc[mi][ni][0], acc[mi][ni][1], a[mi], b[ni]);
        }
    }
    cp_async_wait<0>();

#pragma unroll
    for (int mi = 0; mi < 8; ++mi) {
        const int64_t row = m0 + wm * 64 + mi * 8 + lr;
        if (row >= M) continue;
#pragma unroll
        for (int ni = 0; ni < 4; ++ni) {
            const int64_t col = n0 + wn * 32 + ni * 8 + 2 * lk;
            if (col < N) C[row + col * ldc] = acc[mi][ni][0];
            if (col + 1 < N) C[row + (col + 1) * ldc] = acc[mi][ni][1];
        }
    }
}

// diag >= 0: the GEMM skipped the 128 x BN tiles strictly below the diagonal of a symmetric result (m0 >= diag + n0 + BN);
// their partials were never written and are not read here (launch_mirror_upper fills those elements of C afterwards)
__global__ void __launch_bounds__(256)
splitk_reduce_kernel(const double *__restrict__ part, int splits, int64_t M, int64_t N, double *C, int64_t ldc, int64_t diag,
                     int bn)
{
    const int64_t total = M * N;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        if (diag >= 0 && ((e % M) / BM) * BM >= diag + ((e / M) / bn) * bn + bn) continue;
        double s = 0.0;
        for (int z = 0; z < splits; ++z) s += part[(int64_t)z * total + e];     // fixed order: deterministic
        C[(e % M) + (e / M) * ldc] = s;
    }
}

// Reference-shaped simple kernel (option gemm_path = 1): one thread per output element, plain FMA loop.
template <bool A_MMAJOR>
__global__ void __launch_bounds__(256)
gemm_simple_kernel(const double *__restrict__ A, int64_t lda, const double *__restrict__ B, int64_t ldb, double *C,
                   int64_t ldc, int64_t M, int64_t N, int64_t K)
{
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= M * N) return;
    const int64_t m = e % M, n = e / M;
    double s = 0.0;
    for (int64_t k = 0; k < K; ++k) s = fma(A_MMAJOR ? A[m + k * lda] : A[k + m * lda], B[k + n * ldb], s);
    C[m + n * ldc] = s;
}

// C[i, j] = C[j, i] for i > j (n x n, column-major): 32 x 32 tiles through shared memory, both sides coalesced
__global__ void __launch_bounds__(256)
mirror_upper_kernel(double *C, int64_t ldc, int64_t n)
{
    __shared__ double t[32][33];
    const int64_t bi = blockIdx.x, bj = blockIdx.y;          // destination tile (rows bi, columns bj), bi >= bj
    if (bi < bj) return;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int r = ty; r < 32; r += 8) {                        // source tile: rows bj*32.., columns bi*32..
        const int64_t row = bj * 32 + tx, col = bi * 32 + r;
        t[r][tx] = (row < n && col < n) ? C[row + col * ldc] : 0.0;
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        const int64_t row = bi * 32 + tx, col = bj * 32 + r;  // destination element (row, col) = source (col, row)
        if (row < n && col < n && row > col) C[row + col * ldc] = t[tx][r];
    }
}

struct SplitPlan { int splits; int64_t k_chunk; };

// Split-K plan for the tall contraction (K = N_d >> M, N): the number of CTAs (tiles x splits) is chosen as the
// nearest-to-whole number of waves over the SMs (one CTA per SM), preferring few splits; partial products go to the
// workspace and are summed in a fixed order (deterministic).
// number of 128 x 64 tiles a launch computes (all, or those at / above the diagonal of a symmetric result)
int64_t tiles_computed(int64_t M, int64_t N, int64_t diag)
{
    const int BN = 32 * NWN_DEFAULT;
    const int64_t tm = (M + BM - 1) / BM, tn = (N + BN - 1) / BN;
    if (diag < 0) return tm * tn;
    int64_t c = 0;
    for (int64_t n = 0; n < tn; ++n) c += std::min<int64_t>(tm, (diag + n * BN + BN + BM - 1) / BM);   // tiles with m0 < diag + n0 + BN
    return c;
}

int64_t splitk_ws_cap(int64_t M, int64_t N) { return std::min<int64_t>((int64_t)2 << 30, 64 * M * N * 8); }

SplitPlan plan_tn(const sparc_gpu_ctx *ctx, int64_t M, int64_t N, int64_t K, int64_t diag)
{
    const int64_t tiles = std::max<int64_t>(1, tiles_computed(M, N, diag));
    const int64_t sms = std::max(1, ctx->sm_count) * (NWN_DEFAULT == 2 ? 2 : 1);      // CTA slots
    const int64_t max_splits = std::max<int64_t>(1, std::min<int64_t>(64, K / (16 * BK)));
    const int64_t ws_cap = splitk_ws_cap(M, N);                   // at most 2 GiB of partial products
    int64_t best_s = 1;
    double best_cost = 1e300;
    for (int64_t s = 1; s <= max_splits; ++s) {
        if (s > 1 && s * M * N * 8 > ws_cap) break;
        const int64_t ctas = tiles * s;
        const int64_t waves = (ctas + sms - 1) / sms;
        // time ~ waves * (K / s) per CTA, plus the reduction traffic (s partials of M x N) relative to the main loop
        const double cost = (double)waves * ((double)K / (double)s + 64.0) + (s > 1 ? 0.02 * (double)s * (double)K / 64.0 / (double)std::max<int64_t>(1, tiles / 8 + 1) : 0.0);
        if (cost < best_cost * 0.995) { best_cost = cost; best_s = s; }
    }
    int64_t chunk = (K + best_s - 1) / best_s;
    chunk = round_up_i64(std::max<int64_t>(chunk, 1), BK);
    int64_t splits = (K + chunk - 1) / chunk;
    if (splits < 1) splits = 1;
    return {(int)splits, chunk};
}

bool aligned16(const void *p) { return ((uintptr_t)p & 15) == 0; }

template <bool A_MMAJOR>
int launch_dmma(sparc_gpu_ctx *ctx, const double *A, int64_t lda, const double *B, int64_t ldb, double *C, int64_t ldc,
                int64_t M, int64_t N, int64_t K, SplitPlan plan, int64_t diag, cudaStream_t st)
{
    constexpr int NWN = NWN_DEFAULT, BN = 32 * NWN, GEMM_THREADS = 64 * NWN;
    const int tiles_m = (int)((M + BM - 1) / BM), tiles_n = (int)((N + BN - 1) / BN);
    dim3 grid((unsigned)(tiles_m * tiles_n), 1, (unsigned)plan.splits);
    const bool vec = aligned16(A) && aligned16(B) && (lda % 2 == 0) && (ldb % 2 == 0);
    const size_t smem = smem_bytes(A_MMAJOR, NWN);
    const int kind = A_MMAJOR ? KK_GEMM_NN : KK_GEMM_TN;
    {   // flop actually issued (tiles below the diagonal of a symmetric result are skipped; edge tiles count in full)
        const int64_t computed = tiles_computed(M, N, diag);
        ctx->gemm_flop[A_MMAJOR ? 1 : 0] += 2.0 * (double)K * (double)(BM * BN) * (double)computed;
    }
    // the dynamic shared-memory attribute is set once per context and kernel variant (bits 42..45 of func_attr_done)
    const uint64_t attr_bit = 1ull << (42 + (A_MMAJOR ? 2 : 0) + (vec ? 1 : 0));
    if (vec) {
        auto kern = gemm_dmma_kernel<A_MMAJOR, true, NWN>;
        if (!(ctx->func_attr_done & attr_bit)) {
            SPARC_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            ctx->func_attr_done |= attr_bit;
        }
        prof_begin(ctx, kind, st);
        kern<<<grid, GEMM_THREADS, smem, st>>>(A, lda, B, ldb, C, ldc, M, N, K, plan.k_chunk, tiles_m, diag);
    } else {
        auto kern = gemm_dmma_kernel<A_MMAJOR, false, NWN>;
        if (!(ctx->func_attr_done & attr_bit)) {
            SPARC_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            ctx->func_attr_done |= attr_bit;
        }
        prof_begin(ctx, kind, st);
        kern<<<grid, GEMM_THREADS, smem, st>>>(A, lda, B, ldb, C, ldc, M, N, K, plan.k_chunk, tiles_m, diag);
    }
    prof_end(ctx, kind, st);
    SPARC_CUDA_TRY(cudaGetLastError());
    return SPARC_GPU_SUCCESS;
}

}  // namespace

int64_t gemm_tn_ws_bytes(const sparc_gpu_ctx *ctx, int64_t M, int64_t N, int64_t K)
{
    (void)ctx; (void)K;
    return splitk_ws_cap(M, N);        // upper bound of any split-K plan (the plan depends on the tiles actually computed)
}

int launch_gemm_tn(sparc_gpu_ctx *ctx, const double *A, int64_t lda, const double *B, int64_t ldb, double *C,
                   int64_t ldc, int64_t M, int64_t N, int64_t K, void *ws, int64_t diag, cudaStream_t st)
{
    if (M <= 0 || N <= 0) return SPARC_GPU_SUCCESS;
    if (ctx->opt_gemm_path == 1) {
        const int64_t blocks = (M * N + 255) / 256;
        prof_begin(ctx, KK_GEMM_TN, st);
        gemm_simple_kernel<false><<<(unsigned)blocks, 256, 0, st>>>(A, lda, B, ldb, C, ldc, M, N, K);
        prof_end(ctx, KK_GEMM_TN, st);
        SPARC_CUDA_TRY(cudaGetLastError());
        return SPARC_GPU_SUCCESS;
    }
    SplitPlan plan = plan_tn(ctx, M, N, K, diag);
    if (plan.splits > 1) {
        double *part = (double *)ws;
        SPARC_TRY(launch_dmma<false>(ctx, A, lda, B, ldb, part, M, M, N, K, plan, diag, st));     // skipped tiles stay undefined
        int64_t blocks = std::min<int64_t>((M * N + 255) / 256, (int64_t)ctx->sm_count * 8);
        prof_begin(ctx, KK_SPLITK_REDUCE, st);
        splitk_reduce_kernel<<<(unsigned)blocks, 256, 0, st>>>(part, plan.splits, M, N, C, ldc, diag, 32 * NWN_DEFAULT);
        prof_end(ctx, KK_SPLITK_REDUCE, st);
        SPARC_CUDA_TRY(cudaGetLastError());
        return SPARC_GPU_SUCCESS;
    }
    return launch_dmma<false>(ctx, A, lda, B, ldb, C, ldc, M, N, K, plan, diag, st);
}

int launch_gemm_nn(sparc_gpu_ctx *ctx, const double *A, int64_t lda, const double *B, int64_t ldb, double *C,
                   int64_t ldc, int64_t M, int64_t N, int64_t K, cudaStream_t st)
{
    if (M <= 0 || N <= 0) return SPARC_GPU_SUCCESS;
    if (ctx->opt_gemm_path == 1) {
        const int64_t blocks = (M * N + 255) / 256;
        prof_begin(ctx, KK_GEMM_NN, st);
        gemm_simple_kernel<true><<<(unsigned)blocks, 256, 0, st>>>(A, lda, B, ldb, C, ldc, M, N, K);
        prof_end(ctx, KK_GEMM_NN, st);
        SPARC_CUDA_TRY(cudaGetLastError());
        return SPARC_GPU_SUCCESS;
    }
    SplitPlan plan{1, round_up_i64(std::max<int64_t>(K, 1), BK)};
    return launch_dmma<true>(ctx, A, lda, B, ldb, C, ldc, M, N, K, plan, -1, st);
}

int launch_mirror_upper(sparc_gpu_ctx *ctx, double *C, int64_t ldc, int64_t n, cudaStream_t st)
{
    if (n <= 1) return SPARC_GPU_SUCCESS;
    const unsigned nt = (unsigned)((n + 31) / 32);
    prof_begin(ctx, KK_COPY2D, st);
    mirror_upper_kernel<<<dim3(nt, nt), 256, 0, st>>>(C, ldc, n);
    prof_end(ctx, KK_COPY2D, st);
    SPARC_CUDA_TRY(cudaGetLastError());
    return SPARC_GPU_SUCCESS;
}

// ---- sparc_gpu_gram_static: C = A^T B for callers that cannot allocate (include/sparc_gpu.h) ------------------------------------
// Same DMMA kernel, same fixed-order reduction and same mirror kernel as sparc_gpu_gram; what differs is where the split-K
// partial products live (the file-scope array below instead of the caller's workspace), that no context is needed, and that
// the split plan is limited to what the array holds.  Nothing above this line is touched by it.

namespace {

constexpr int64_t GRAM_STATIC_ELEMS = SPARC_GPU_GRAM_STATIC_MAX_ELEMS;      // 2 Mi doubles = 16 MiB

// The scratch itself.  It is part of the library's device image: each GPU on which this library's code is loaded sets
// 16 MiB aside for it and keeps them until the process ends, whether or not sparc_gpu_gram_static is ever called.
// In HOST code the identifier below is only a handle for cudaGetSymbolAddress -- it is NOT a device address and must never
// be handed to a kernel as such (the kernel would fault, or on a system where the GPU can read host memory, quietly work
// on the wrong bytes).  gram_static_setup() asks the runtime for the real address once per device.
static __device__ __align__(256) double g_gram_static_scratch[GRAM_STATIC_ELEMS];

constexpr int GRAM_STATIC_MAX_DEVICES = 64;
struct GramStaticDevice {
    bool ready = false;
    double *scratch = nullptr;      // device address of g_gram_static_scratch on this GPU
    int sm_count = 0;
};
GramStaticDevice g_gram_static_device[GRAM_STATIC_MAX_DEVICES];
std::mutex g_gram_static_mutex;

// One-time set-up for `device`, which the caller has made current: resolve the array's address on this GPU, read the SM
// count, raise the kernels' dynamic shared-memory limit.  No allocation (the array came with the module).
int gram_static_setup(int device, GramStaticDevice *out)
{
    std::lock_guard<std::mutex> lock(g_gram_static_mutex);
    GramStaticDevice &d = g_gram_static_device[device];
    if (!d.ready) {
        int major = 0, sms = 0;
        SPARC_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device));
        if (major != 10) return SPARC_GPU_UNSUPPORTED;                       // the library holds sm_100a code only
        SPARC_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
        double *ptr = nullptr;
        SPARC_CUDA_TRY(cudaGetSymbolAddress((void **)&ptr, g_gram_static_scratch));
        if (!ptr) return SPARC_GPU_CUDA_ERROR;
        const int smem = (int)smem_bytes(false, NWN_DEFAULT);
        SPARC_CUDA_TRY(cudaFuncSetAttribute(gemm_dmma_kernel<false, true, NWN_DEFAULT>,
                                            cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        SPARC_CUDA_TRY(cudaFuncSetAttribute(gemm_dmma_kernel<false, false, NWN_DEFAULT>,
                                            cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        d.scratch = ptr;
        d.sm_count = std::max(1, sms);
        d.ready = true;
    }
    *out = d;
    return SPARC_GPU_SUCCESS;
}

// plan_tn's cost model with the static array as the cap on the partial products (splits * M * N <= GRAM_STATIC_ELEMS)
SplitPlan plan_tn_static(int sm_count, int64_t M, int64_t N, int64_t K, int64_t diag)
{
    const int64_t tiles = std::max<int64_t>(1, tiles_computed(M, N, diag));
    const int64_t slots = (int64_t)sm_count * (NWN_DEFAULT == 2 ? 2 : 1);
    const int64_t max_splits = std::max<int64_t>(1, std::min<int64_t>(64, K / (16 * BK)));
    const int64_t cap_elems = std::min<int64_t>(GRAM_STATIC_ELEMS, 64 * M * N);
    int64_t best_s = 1;
    double best_cost = 1e300;
    for (int64_t s = 1; s <= max_splits; ++s) {
        if (s > 1 && s * M * N > cap_elems) break;
        const int64_t waves = (tiles * s + slots - 1) / slots;
        const double cost = (double)waves * ((double)K / (double)s + 64.0)
                            + (s > 1 ? 0.02 * (double)s * (double)K / 64.0 / (double)std::max<int64_t>(1, tiles / 8 + 1) : 0.0);
        if (cost < best_cost * 0.995) { best_cost = cost; best_s = s; }
    }
    const int64_t chunk = round_up_i64(std::max<int64_t>((K + best_s - 1) / best_s, 1), BK);
    return {(int)std::max<int64_t>(1, (K + chunk - 1) / chunk), chunk};
}

}  // namespace

extern "C" int sparc_gpu_gram_static(int device, const double *A, int64_t lda, const double *B, int64_t ldb, int64_t nrows,
                                     int64_t m, int64_t n, double *C, int symmetric, void *stream)
{
    if (device < 0 || device >= GRAM_STATIC_MAX_DEVICES || nrows < 0 || m < 0 || n < 0) return SPARC_GPU_INVALID_ARG;
    if (m == 0 || n == 0) return SPARC_GPU_SUCCESS;
    if (!C || (symmetric && m != n)) return SPARC_GPU_INVALID_ARG;
    if (nrows > 0 && (!A || !B || lda < nrows || ldb < nrows)) return SPARC_GPU_INVALID_ARG;
    if (m > GRAM_STATIC_ELEMS || n > GRAM_STATIC_ELEMS || m * n > GRAM_STATIC_ELEMS) return SPARC_GPU_STATIC_SCRATCH_EXCEEDED;
    DeviceGuard dg(device);
    if (!dg.ok) return SPARC_GPU_CUDA_ERROR;
    GramStaticDevice dev;
    SPARC_TRY(gram_static_setup(device, &dev));
    cudaStream_t st = (cudaStream_t)stream;
    if (nrows == 0) { SPARC_CUDA_TRY(cudaMemsetAsync(C, 0, (size_t)m * n * 8, st)); return SPARC_GPU_SUCCESS; }

    constexpr int BN = 32 * NWN_DEFAULT, GEMM_THREADS = 64 * NWN_DEFAULT;
    const int64_t diag = symmetric ? 0 : -1;
    const SplitPlan plan = plan_tn_static(dev.sm_count, m, n, nrows, diag);
    // every partial element that the reduction reads is written by this call's GEMM launch first, so nothing in the
    // array has to be cleared: what an earlier call left there is never read
    double *out = plan.splits > 1 ? dev.scratch : C;
    const int tiles_m = (int)((m + BM - 1) / BM), tiles_n = (int)((n + BN - 1) / BN);
    const dim3 grid((unsigned)(tiles_m * tiles_n), 1, (unsigned)plan.splits);
    const size_t smem = smem_bytes(false, NWN_DEFAULT);
    if (aligned16(A) && aligned16(B) && lda % 2 == 0 && ldb % 2 == 0)
        gemm_dmma_kernel<false, true, NWN_DEFAULT><<<grid, GEMM_THREADS, smem, st>>>(A, lda, B, ldb, out, m, m, n, nrows,
                                                                                    plan.k_chunk, tiles_m, diag);
    else
        gemm_dmma_kernel<false, false, NWN_DEFAULT><<<grid, GEMM_THREADS, smem, st>>>(A, lda, B, ldb, out, m, m, n, nrows,
                                                                                     plan.k_chunk, tiles_m, diag);
    SPARC_CUDA_TRY(cudaGetLastError());
    if (plan.splits > 1) {
        const int64_t blocks = std::min<int64_t>((m * n + 255) / 256, (int64_t)dev.sm_count * 8);
        splitk_reduce_kernel<<<(unsigned)blocks, 256, 0, st>>>(dev.scratch, plan.splits, m, n, C, m, diag, BN);
        SPARC_CUDA_TRY(cudaGetLastError());
    }
    if (symmetric && m > 1) {
        const unsigned nt = (unsigned)((m + 31) / 32);
        mirror_upper_kernel<<<dim3(nt, nt), 256, 0, st>>>(C, m, m);
        SPARC_CUDA_TRY(cudaGetLastError());
    }
    return SPARC_GPU_SUCCESS;
}
