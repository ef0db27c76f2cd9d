// stencil_tma.cu -- the tuned fused local pass for sm_100a:
//     Out = alpha (H_loc X + shift X) + beta Prev,   H_loc = -1/2 Laplacian(radius 6) + Veff
// i.e. stencil + Veff multiply + Chebyshev three-term axpy in ONE
// pass: each degree step reads Psi_k once, Psi_{k-1} once and writes Psi_{k+1} once (24 B per grid point).
//
// Design (differs from the paper's Micikevicius-style kernel):
//   * work item = (orbital column, y-tile of TY rows, z-chunk); the tile spans the WHOLE x extent, so the x halo
//     never leaves the SM; the CTA marches through z.
//   * warp 0 is the producer: it streams one z-plane of the tile per step into a shared-memory ring with TMA
//     (cp.async.bulk.tensor.4d over the (x, y, z, column) tensor, boxes of W x 6 rows; out-of-range rows / planes
//     are zero-filled by TMA = Dirichlet; periodic y / z by wrapping the box coordinate; periodic x by patching the
//     6+6 halo columns inside shared memory), then hands the plane to the consumers through an mbarrier.
//   * the other warps are consumers.  Each thread owns 2 (x) x AY (y) points of the tile and keeps the 13 partial
//     z-sums of each of them in registers ("register-blocked z-column", accumulate form): an arriving plane adds
//     its centre/x/y taps to the output plane it is the centre of and one z tap to each of the 12 neighbouring
//     output planes; the output plane that just received its last tap gets + beta*Prev and is stored.  Shared
//     memory traffic is 1 + 6/1 + 12/AY vector loads per 2 outputs; coefficients sit in the constant bank.
//   * Veff and Prev are read straight from global (L2 / HBM) with 16-byte loads, Out is written with 16-byte stores.
#include <cuda.h>

#include <algorithm>

#include "internal.h"

namespace {

constexpr int R = 6;             // stencil radius of the tuned path (FD order 12)
constexpr int NSLOT = 2 * R + 1; // 13 partial sums per point
constexpr int NSTAGE = 6;        // shared-memory ring depth (planes)
constexpr int LAG = 2;           // producer refills a stage LAG planes after it was handed out
constexpr int BOX_ROWS = 6;      // TMA box height (= halo height)

struct TmaParams {
    double cx[R + 1], cy[R + 1], cz[R + 1];   // alpha * (-1/2 w_p / h^2)
    double c0a;                                // alpha * (c0 + shift)
    double alpha, beta;
    const double *veff;
    double *out;
    const double *prev;
    int64_t ldo, ldp;
    int nx, ny, nz;
    int W;            // smem row pitch in doubles (>= nx + 12, multiple of 8)
    int TY;           // tile rows
    int ntx;          // nx / 2 consumer threads along x
    int n_consumers;  // ntx * (TY / AY)
    int ytiles, zchunks, zchunk_len;
    int per_x, per_y, per_z;
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra WAIT_DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "WAIT_DONE:\n\t"
        "}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *tmap, uint64_t *bar, int x, int y, int z, int c)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(
            smem_u32(dst)),
        "l"(tmap), "r"(x), "r"(y), "r"(z), "r"(c), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ double2 ldg_stream(const double *p)
{
    double2 v;
    asm volatile("ld.global.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}

template <int AY, bool HAS_PREV>
__global__ void __launch_bounds__(AY == 2 ? 384 : 288, 1)
stencil_tma_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ TmaParams P)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t *bar_full = reinterpret_cast<uint64_t *>(smem_raw);   // [NSTAGE] TMA landed
    uint64_t *bar_ready = bar_full + NSTAGE;                       // [NSTAGE] halo patched, consumers may read
    uint64_t *bar_empty = bar_ready + NSTAGE;                      // [NSTAGE] consumers done
    unsigned char *stages = smem_raw + 256;
    const int rows = P.TY + 2 * R;
    const uint32_t stage_bytes = (uint32_t)(P.W * rows * 8);

    const int tid = threadIdx.x;
    const int n_cwarps = (P.n_consumers + 31) >> 5;
    if (tid == 0) {
        for (int s = 0; s < NSTAGE; ++s) {
            mbar_init(&bar_full[s], 1);
            mbar_init(&bar_ready[s], 1);
            mbar_init(&bar_empty[s], (uint32_t)n_cwarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // ---- work item -------------------------------------------------------------------------------------
    const int per_col = P.ytiles * P.zchunks;
    const int col = blockIdx.x / per_col;
    const int rem = blockIdx.x - col * per_col;
    const int ytile = rem / P.zchunks;
    const int zc = rem - ytile * P.zchunks;
    const int y0 = ytile * P.TY;
    const int z0 = zc * P.zchunk_len;
    const int z1 = min(z0 + P.zchunk_len, P.nz);
    const int nzc = z1 - z0;
    const int nsteps = nzc + 2 * R;          // input planes z0-6 .. z1+5

    if (tid < 32) {
        // ================================ producer warp ================================================
        const int lane = tid;
        const int nboxes = rows / BOX_ROWS;
        auto issue_plane = [&](int s) {
            const int stage = s % NSTAGE;
            int zin = z0 - R + s;
            if (P.per_z) { if (zin < 0) zin += P.nz; else if (zin >= P.nz) zin -= P.nz; }
            unsigned char *dst = stages + (size_t)stage * stage_bytes;
            mbar_arrive_expect_tx(&bar_full[stage], stage_bytes);
            for (int b = 0; b < nboxes; ++b) {
                int y = y0 - R + b * BOX_ROWS;
                if (P.per_y) { if (y < 0) y += P.ny; else if (y >= P.ny) y -= P.ny; }
                tma_load_4d(dst + (size_t)b * BOX_ROWS * P.W * 8, &tmap, &bar_full[stage], -R, y, zin, col);
            }
        };
        if (lane == 0) {
            asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap) : "memory");
            for (int s = 0; s < NSTAGE - LAG && s < nsteps; ++s) issue_plane(s);
        }
        for (int i = 0; i < nsteps; ++i) {
            const int snew = i + NSTAGE - LAG;
            if (snew < nsteps && lane == 0) {
                if (i >= LAG) {
                    const int sold = i - LAG;    // plane that used the stage before
                    mbar_wait(&bar_empty[sold % NSTAGE], (uint32_t)((sold / NSTAGE) & 1));
                }
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                issue_plane(snew);
            }
            const int stage = i % NSTAGE;
            mbar_wait(&bar_full[stage], (uint32_t)((i / NSTAGE) & 1));
            if (P.per_x) {
                double *pl = reinterpret_cast<double *>(stages + (size_t)stage * stage_bytes);
                for (int k = lane; k < rows * 2 * R; k += 32) {
                    const int r = k / (2 * R), j = k - r * (2 * R);
                    double *row = pl + r * P.W;
                    if (j < R) row[j] = row[j + P.nx];                 // left halo  <- last 6 of the row
                    else row[P.nx + j] = row[j];                       // right halo <- first 6 (j in 6..11 -> sx nx+6..nx+11)
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&bar_ready[stage]);
        }
        return;
    }

    // ==================================== consumer warps ====================================================
    const int ct = tid - 32;
    const bool active = ct < P.n_consumers;
    const int cta = active ? ct : 0;                 // inactive lanes shadow thread 0 and never store
    const int ty = cta / P.ntx, tx = cta - ty * P.ntx;
    const int lane = tid & 31;
    const int pitchB = P.W * 8;
    // byte offset of the thread's first own point inside a stage: row (ty*AY + 6), column (2*tx + 6)
    const uint32_t thr_off = (uint32_t)(((ty * AY + R) * P.W + 2 * tx + R) * 8);
    const int64_t plane = (int64_t)P.nx * P.ny;
    const int64_t pt_off = (int64_t)(y0 + ty * AY) * P.nx + 2 * tx;     // offset of the own point inside a plane
    const double *veff_p = P.veff + pt_off;
    double *out_p = P.out + (int64_t)col * P.ldo + pt_off;
    const double *prev_p = HAS_PREV ? P.prev + (int64_t)col * P.ldp + pt_off : nullptr;

    double acc[NSLOT][AY][2];
#pragma unroll
    for (int s = 0; s < NSLOT; ++s)
#pragma unroll
        for (int a = 0; a < AY; ++a) acc[s][a][0] = acc[s][a][1] = 0.0;

    int s = 0;
    for (int sb = 0; sb < nsteps; sb += NSLOT) {
#pragma unroll
        for (int ph = 0; ph < NSLOT; ++ph) {
            if (s >= nsteps) break;
            const int stage = s % NSTAGE;
            const int zin = z0 - R + s;              // plane arriving (unwrapped index)
            const int zo = zin - R;                  // plane completed by this step
            const bool do_xy = (s >= R) && (s < R + nzc);
            const bool do_store = (s >= 2 * R);

            // early global loads for this step
            double2 pv[AY], vf[AY];
            if (HAS_PREV && do_store) {
#pragma unroll
                for (int a = 0; a < AY; ++a) pv[a] = ldg_stream(prev_p + (int64_t)zo * plane + a * P.nx);
            }
            if (do_xy) {
#pragma unroll
                for (int a = 0; a < AY; ++a)
                    vf[a] = *reinterpret_cast<const double2 *>(veff_p + (int64_t)zin * plane + a * P.nx);
            }

            mbar_wait(&bar_ready[stage], (uint32_t)((s / NSTAGE) & 1));
            const unsigned char *sp = stages + (size_t)stage * stage_bytes + thr_off;
#define LD2(ptr) (*reinterpret_cast<const double2 *>(ptr))
            double2 own[AY];
#pragma unroll
            for (int a = 0; a < AY; ++a) own[a] = LD2(sp + a * pitchB);

            // ---- z taps: this plane feeds the 12 neighbouring output planes --------------------------------
#pragma unroll
            for (int d = -R; d <= R; ++d) {
                if (d == 0) continue;
                const int slot = (ph - d + NSLOT) % NSLOT;
                const double c = P.cz[d < 0 ? -d : d];
#pragma unroll
                for (int a = 0; a < AY; ++a) {
                    if (d == -R) {            // first contribution to output plane zin + 6: opens the slot
                        acc[slot][a][0] = c * own[a].x;
                        acc[slot][a][1] = c * own[a].y;
                    } else {
                        acc[slot][a][0] = fma(c, own[a].x, acc[slot][a][0]);
                        acc[slot][a][1] = fma(c, own[a].y, acc[slot][a][1]);
                    }
                }
            }

            // ---- centre, x and y taps of the plane this one is the centre of --------------------------------
            if (do_xy) {
#pragma unroll
                for (int a = 0; a < AY; ++a) {
                    const unsigned char *rp = sp + a * pitchB;
                    double h[2 * R + 2];       // x - 6 .. x + 7
                    {
                        const double2 m3 = LD2(rp - 48), m2 = LD2(rp - 32), m1 = LD2(rp - 16);
                        const double2 p1 = LD2(rp + 16), p2 = LD2(rp + 32), p3 = LD2(rp + 48);
                        h[0] = m3.x; h[1] = m3.y; h[2] = m2.x; h[3] = m2.y; h[4] = m1.x; h[5] = m1.y;
                        h[6] = own[a].x; h[7] = own[a].y;
                        h[8] = p1.x; h[9] = p1.y; h[10] = p2.x; h[11] = p2.y; h[12] = p3.x; h[13] = p3.y;
                    }
                    double s0 = fma(P.alpha, vf[a].x, P.c0a) * own[a].x;
                    double s1 = fma(P.alpha, vf[a].y, P.c0a) * own[a].y;
#pragma unroll
                    for (int p = 1; p <= R; ++p) {
                        s0 = fma(P.cx[p], h[6 - p], s0);
                        s0 = fma(P.cx[p], h[6 + p], s0);
                        s1 = fma(P.cx[p], h[7 - p], s1);
                        s1 = fma(P.cx[p], h[7 + p], s1);
                    }
                    acc[ph][a][0] += s0;
                    acc[ph][a][1] += s1;
                }
#pragma unroll
                for (int rr = -R; rr < AY + R; ++rr) {
                    const double2 yv = (rr >= 0 && rr < AY) ? own[rr >= 0 && rr < AY ? rr : 0] : LD2(sp + rr * pitchB);
#pragma unroll
                    for (int a = 0; a < AY; ++a) {
                        const int dist = rr > a ? rr - a : a - rr;
                        if (dist >= 1 && dist <= R) {
                            acc[ph][a][0] = fma(P.cy[dist], yv.x, acc[ph][a][0]);
                            acc[ph][a][1] = fma(P.cy[dist], yv.y, acc[ph][a][1]);
                        }
                    }
                }
            }
#undef LD2
            // ---- this stage is free again ---------------------------------------------------------------------
            __syncwarp();
            if (lane == 0) mbar_arrive(&bar_empty[stage]);

            // ---- output plane zo has all 37 taps: recurrence axpy + store --------------------------------------
            if (do_store) {
                const int cs = (ph + R + 1) % NSLOT;      // slot of plane zin - 6
                if (active) {
#pragma unroll
                    for (int a = 0; a < AY; ++a) {
                        double2 o;
                        if (HAS_PREV) {
                            o.x = fma(P.beta, pv[a].x, acc[cs][a][0]);
                            o.y = fma(P.beta, pv[a].y, acc[cs][a][1]);
                        } else {
                            o.x = acc[cs][a][0];
                            o.y = acc[cs][a][1];
                        }
                        *reinterpret_cast<double2 *>(out_p + (int64_t)zo * plane + a * P.nx) = o;
                    }
                }
            }
            ++s;
        }
    }
}

struct TileChoice { int TY, AY; };

// tile rows: a multiple of 6 dividing ny, as tall as the register budget allows (consumers <= cap)
bool choose_tile(int nx, int ny, TileChoice *tc)
{
    const int ntx = nx / 2;
    int best_ty = 0, best_ay = 0;
    for (int ay = 2; ay <= 2; ++ay) {     // AY = 3 spills at the 224-register cap: not instantiated
        const int cap = (ay == 2) ? 352 : 256;
        for (int ty = ny; ty >= 6; --ty) {
            if (ny % ty || ty % BOX_ROWS || ty % ay) continue;
            if (ntx * (ty / ay) > cap) continue;
            if (ty > best_ty) { best_ty = ty; best_ay = ay; }
            break;
        }
    }
    if (!best_ty) return false;
    tc->TY = best_ty; tc->AY = best_ay;
    return true;
}

bool a16(const void *p) { return ((uintptr_t)p & 15) == 0; }

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

}  // namespace

bool stencil_tma_supported(const sparc_gpu_ctx *ctx, const double *X, int64_t ldx, const double *Out, int64_t ldo,
                           const double *Prev, int64_t ldp)
{
    if (!ctx->fn_encode_tiled || ctx->radius != R) return false;
    const int nx = ctx->n[0], ny = ctx->n[1];
    if (nx & 1) return false;
    if (nx < 2 * R + 2 || round_up_i64(nx + 2 * R, 8) > 256) return false;
    if (ny % BOX_ROWS) return false;
    if (!a16(X) || !a16(Out) || (Prev && !a16(Prev)) || (ldx & 1) || (ldo & 1) || (Prev && (ldp & 1))) return false;
    TileChoice tc;
    return choose_tile(nx, ny, &tc);
}

int launch_stencil_tma(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, double *Out, int64_t ldo, const double *Prev,
                       int64_t ldp, int64_t ncols, double alpha, double shift, double beta, cudaStream_t st)
{
    const bool has_prev = (beta != 0.0) && Prev;
    if (!stencil_tma_supported(ctx, X, ldx, Out, ldo, has_prev ? Prev : nullptr, ldp)) return SPARC_GPU_UNSUPPORTED;
    const int nx = ctx->n[0], ny = ctx->n[1], nz = ctx->n[2];
    TileChoice tc;
    choose_tile(nx, ny, &tc);

    TmaParams P;
    for (int p = 0; p <= R; ++p) { P.cx[p] = alpha * ctx->coef.cx[p]; P.cy[p] = alpha * ctx->coef.cy[p]; P.cz[p] = alpha * ctx->coef.cz[p]; }
    P.c0a = alpha * (ctx->coef.c0 + shift);
    P.alpha = alpha; P.beta = beta;
    P.veff = ctx->d_veff;
    P.ldo = ldo; P.ldp = ldp;
    P.nx = nx; P.ny = ny; P.nz = nz;
    P.W = (int)round_up_i64(nx + 2 * R, 8);
    P.TY = tc.TY;
    P.ntx = nx / 2;
    P.n_consumers = P.ntx * (tc.TY / tc.AY);
    P.ytiles = ny / tc.TY;
    P.per_x = ctx->bc[0] == 0; P.per_y = ctx->bc[1] == 0; P.per_z = ctx->bc[2] == 0;

    const int threads = 32 + (P.n_consumers + 31) / 32 * 32;
    const size_t smem = 256 + (size_t)NSTAGE * P.W * (tc.TY + 2 * R) * 8;
    if (smem > 227 * 1024) return SPARC_GPU_UNSUPPORTED;

    // z chunks: split the march only as far as needed to give the chip about two waves of CTAs
    const int64_t max_cols_per_launch = std::max<int64_t>(1, (int64_t)INT32_MAX / ((int64_t)P.ytiles * nz));
    for (int64_t j0 = 0; j0 < ncols; j0 += max_cols_per_launch) {
        const int64_t nb = std::min<int64_t>(max_cols_per_launch, ncols - j0);
        int zchunks = 1;
        const int64_t base = nb * P.ytiles;
        const int64_t want = 2LL * ctx->sm_count;
        if (base < want) zchunks = (int)std::min<int64_t>((want + base - 1) / base, std::max(1, nz / 12));
        P.zchunk_len = (nz + zchunks - 1) / zchunks;
        P.zchunks = (nz + P.zchunk_len - 1) / P.zchunk_len;
        P.out = Out + j0 * ldo;
        P.prev = has_prev ? Prev + j0 * ldp : nullptr;

        CUtensorMap tmap;
        const cuuint64_t gdim[4] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)nz, (cuuint64_t)nb};
        const cuuint64_t gstr[3] = {(cuuint64_t)nx * 8, (cuuint64_t)nx * ny * 8, (cuuint64_t)ldx * 8};
        const cuuint32_t box[4] = {(cuuint32_t)P.W, BOX_ROWS, 1, 1};
        const cuuint32_t estr[4] = {1, 1, 1, 1};
        CUresult cr = ((EncodeTiledFn)ctx->fn_encode_tiled)(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4,
                                                            (void *)(X + j0 * ldx), gdim, gstr, box, estr,
                                                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                                            CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (cr != CUDA_SUCCESS) return SPARC_GPU_CUDA_ERROR;

        const unsigned grid = (unsigned)(nb * P.ytiles * P.zchunks);
#define LAUNCH_TMA(AYV, HP)                                                                                          \
        do {                                                                                                         \
            auto kern = stencil_tma_kernel<AYV, HP>;                                                                 \
            SPARC_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));      \
            prof_begin(ctx, KK_STENCIL_TMA, st);                                                                     \
            kern<<<grid, threads, smem, st>>>(tmap, P);                                                              \
            prof_end(ctx, KK_STENCIL_TMA, st);                                                                       \
        } while (0)
        if (has_prev) LAUNCH_TMA(2, true); else LAUNCH_TMA(2, false);
#undef LAUNCH_TMA
    }
    SPARC_CUDA_TRY(cudaGetLastError());
    return SPARC_GPU_SUCCESS;
}
