// stencil_tma.cu -- the tuned fused local pass for sm_100a:
//     Out = alpha (H_loc X + shift X) + beta Prev,   H_loc = -1/2 Laplacian(radius 6) + Veff
// i.e. stencil + Veff multiply + Chebyshev three-term axpy in ONE
// pass: each degree step reads Psi_k once, Psi_{k-1} once and writes Psi_{k+1} once (24 B per grid point).
//
// Design (differs from the paper's Micikevicius-style kernel):
//   * work item = (orbital column, y-tile of TY rows, z-chunk); the tile spans the WHOLE x extent, so the x halo
//     never leaves the SM; the CTA marches through z.  Tiles are small (about 150 consumer threads) so that two or
//     three CTAs share an SM and overlap each other's pipeline bubbles.
//   * warp 0 is the producer: one lane streams, per z step, the input plane of the tile (rows y0-6 .. y0+TY+5), the
//     matching Veff plane and the Prev plane of the output that completes at this step into a shared-memory ring
//     with TMA (cp.async.bulk.tensor over the (x, y, z, column) tensors); out-of-range rows / planes are
//     zero-filled by TMA = Dirichlet; periodic y / z by wrapping the box coordinate.  Periodic x needs no halo
//     columns at all: consumers address their x neighbours through per-thread precomputed (wrapped) offsets.
//   * the other warps are consumers.  Each thread owns 2 (x) x AY (y) points of the tile and keeps the 13 partial
//     z-sums of each of them in registers ("register-blocked z-column", accumulate form): an arriving plane adds
//     its centre/x/y taps to the output plane it is the centre of and one z tap to each of the 12 neighbouring
//     output planes; the output plane that just received its last tap gets + beta*Prev and is stored with a
//     16-byte coalesced store.  Shared-memory traffic is 13 doubles per output; coefficients sit in the constant bank.
#include <cuda.h>

#include <algorithm>

#include "internal.h"
#include "sm100_ptx.cuh"

namespace {

constexpr int R = 6;             // stencil radius of the tuned path (FD order 12)
constexpr int NSLOT = 2 * R + 1; // 13 partial sums per point
constexpr int BOX_ROWS = 6;      // TMA box height of the input plane (= halo height)
constexpr int MAX_THREADS_AY2 = 384;   // 168 registers / thread
constexpr int MAX_THREADS_AY1 = 320;   // two CTAs of this size per SM -> 102 registers / thread
constexpr int MAX_STAGES = 8;

struct TmaParams {
    double cx[R + 1], cy[R + 1], cz[R + 1];   // alpha * (-1/2 w_p / h^2)
    double c0a;                                // alpha * (c0 + shift)
    double alpha, beta;
    double *out;
    int64_t ldo;
    int nx, ny, nz;
    int W;            // smem row pitch of the input plane in doubles (multiple of 8)
    int x_start;      // first x coordinate of the input box: 0 (periodic x) or -6 (Dirichlet x)
    int TY;           // tile rows
    int ntx;          // nx / 2 consumer threads along x
    int n_consumers;  // ntx * (TY / AY)
    int nstage;
    int ytiles, zchunks, zchunk_len;
    int per_x, per_y, per_z;
    uint32_t psi_bytes, tile_bytes, stage_bytes;   // input plane, Veff / Prev tile, whole stage (128-B multiples)
};

using namespace sm100;


// AY: rows per consumer thread (2: 4 points / 168 registers, 1: 2 points / ~100 registers, twice the warps);
// CW, CNX: compile-time smem pitches (doubles) of the input plane and of the Veff / Prev tiles, 0 = run time (P.W, P.nx).
template <int AY, int CW, int CNX, bool HAS_PREV>
__global__ void __launch_bounds__(AY == 1 ? MAX_THREADS_AY1 : MAX_THREADS_AY2, AY == 1 ? 2 : 1)
stencil_tma_kernel(const __grid_constant__ CUtensorMap tmap_x, const __grid_constant__ CUtensorMap tmap_v,
                   const __grid_constant__ CUtensorMap tmap_p, const __grid_constant__ TmaParams P)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    // barriers first, stages after them at the next 128-byte boundary (TMA destination alignment)
    uint64_t *bar_full = reinterpret_cast<uint64_t *>(smem_raw);    // [MAX_STAGES] TMA landed
    uint64_t *bar_empty = bar_full + MAX_STAGES;                    // [MAX_STAGES] consumers done
    const uint32_t stage0 = (smem_u32(smem_raw) + 2 * MAX_STAGES * 8 + 127u) & ~127u;

    const int tid = threadIdx.x;
    const int n_cwarps = (P.n_consumers + 31) >> 5;
    if (tid == 0) {
        for (int s = 0; s < P.nstage; ++s) {
            mbar_init(&bar_full[s], 1);
            mbar_init(&bar_empty[s], (uint32_t)n_cwarps);
        }
        mbar_fence_init();
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
    const int W = CW ? CW : P.W;
    const int NX = CNX ? CNX : P.nx;

    if (tid < 32) {
        // ================================ producer warp (one lane) =======================================
        if (tid != 0) return;
        prefetch_tmap(&tmap_x);
        prefetch_tmap(&tmap_v);
        if (HAS_PREV) prefetch_tmap(&tmap_p);
        const int nboxes = (P.TY + 2 * R) / BOX_ROWS;
        const uint32_t box_bytes = (uint32_t)(BOX_ROWS * W * 8);
        const uint32_t tile_tx = (uint32_t)(P.TY * NX * 8);
        int stage = 0;
        uint32_t phase = 0;
        for (int s = 0; s < nsteps; ++s) {
            if (s >= P.nstage) {
                while (!mbar_try_wait(&bar_empty[stage], phase ^ 1u)) __nanosleep(40);   // do not steal issue slots
            }
            const bool do_xy = (s >= R) && (s < R + nzc);
            const bool do_prev = HAS_PREV && (s >= 2 * R);
            int zin = z0 - R + s;
            if (P.per_z) { if (zin < 0) zin += P.nz; else if (zin >= P.nz) zin -= P.nz; }
            const uint32_t dst = stage0 + (uint32_t)stage * P.stage_bytes;
            mbar_arrive_expect_tx(&bar_full[stage], P.psi_bytes + (do_xy ? tile_tx : 0u) + (do_prev ? tile_tx : 0u));
            for (int b = 0; b < nboxes; ++b) {
                int y = y0 - R + b * BOX_ROWS;
                if (P.per_y) { if (y < 0) y += P.ny; else if (y >= P.ny) y -= P.ny; }
                tma_load_4d(dst + (uint32_t)b * box_bytes, &tmap_x, &bar_full[stage], P.x_start, y, zin, col);
            }
            if (do_xy) tma_load_3d(dst + P.psi_bytes, &tmap_v, &bar_full[stage], 0, y0, z0 - R + s);
            if (do_prev) tma_load_4d(dst + P.psi_bytes + P.tile_bytes, &tmap_p, &bar_full[stage], 0, y0, z0 - 2 * R + s, col);
            if (++stage == P.nstage) { stage = 0; phase ^= 1u; }
        }
        return;
    }

    // ==================================== consumer warps ====================================================
    const int ct = tid - 32;
    const bool active = ct < P.n_consumers;
    const int cta = active ? ct : 0;                 // inactive lanes shadow thread 0 and never store
    const int ty = cta / P.ntx, tx = cta - ty * P.ntx;
    const int lane = tid & 31;
    const uint32_t pitchB = (uint32_t)W * 8u;
    const uint32_t tile_pitchB = (uint32_t)NX * 8u;
    // shared-memory byte addresses (relative to the stage) of the x-neighbour pairs tx-3 .. tx+3 in the first own
    // row; a periodic x axis wraps the pair index instead of storing halo columns
    uint32_t xo[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) {
        int p = tx + k - 3;
        if (P.per_x) { if (p < 0) p += P.ntx; else if (p >= P.ntx) p -= P.ntx; }
        else p += 3;
        xo[k] = (uint32_t)(ty * AY + R) * pitchB + (uint32_t)p * 16u;
    }
    const uint32_t tile_off = P.psi_bytes + (uint32_t)((ty * AY * NX + 2 * tx) * 8);   // own pair inside the Veff tile
    const int64_t plane = (int64_t)P.nx * P.ny;
    // running output pointer: plane z0 - 12 at step 0, advanced by one plane per step
    double *out_z = P.out + (int64_t)col * P.ldo + (int64_t)(y0 + ty * AY) * P.nx + 2 * tx + (int64_t)(z0 - 2 * R) * plane;

    double acc[NSLOT][AY][2];
#pragma unroll
    for (int s = 0; s < NSLOT; ++s)
#pragma unroll
        for (int a = 0; a < AY; ++a) acc[s][a][0] = acc[s][a][1] = 0.0;

    int s = 0, stage = 0;
    uint32_t phase = 0;
    for (int sb = 0; sb < nsteps; sb += NSLOT) {
#pragma unroll
        for (int ph = 0; ph < NSLOT; ++ph) {
            if (s >= nsteps) break;
            const bool do_xy = (s >= R) && (s < R + nzc);
            const bool do_store = (s >= 2 * R);
            const uint32_t st = stage0 + (uint32_t)stage * P.stage_bytes;

            mbar_wait(&bar_full[stage], phase);
            double2 own[AY];
#pragma unroll
            for (int a = 0; a < AY; ++a) own[a] = lds2(st + xo[3] + a * pitchB);

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
                    const double2 vf = lds2(st + tile_off + a * tile_pitchB);
                    const double2 m3 = lds2(st + xo[0] + a * pitchB), m2 = lds2(st + xo[1] + a * pitchB);
                    const double2 m1 = lds2(st + xo[2] + a * pitchB), p1 = lds2(st + xo[4] + a * pitchB);
                    const double2 p2 = lds2(st + xo[5] + a * pitchB), p3 = lds2(st + xo[6] + a * pitchB);
                    // left and right halves are separate dependency chains
                    double l0 = fma(P.alpha, vf.x, P.c0a) * own[a].x;
                    double l1 = fma(P.alpha, vf.y, P.c0a) * own[a].y;
                    double r0 = P.cx[1] * own[a].y, r1 = P.cx[1] * own[a].x;   // x+1 of point 0, x-1 of point 1
                    l0 = fma(P.cx[1], m1.y, l0); l0 = fma(P.cx[2], m1.x, l0); l0 = fma(P.cx[3], m2.y, l0);
                    l0 = fma(P.cx[4], m2.x, l0); l0 = fma(P.cx[5], m3.y, l0); l0 = fma(P.cx[6], m3.x, l0);
                    r0 = fma(P.cx[2], p1.x, r0); r0 = fma(P.cx[3], p1.y, r0); r0 = fma(P.cx[4], p2.x, r0);
                    r0 = fma(P.cx[5], p2.y, r0); r0 = fma(P.cx[6], p3.x, r0);
                    r1 = fma(P.cx[2], m1.y, r1); r1 = fma(P.cx[3], m1.x, r1); r1 = fma(P.cx[4], m2.y, r1);
                    r1 = fma(P.cx[5], m2.x, r1); r1 = fma(P.cx[6], m3.y, r1);
                    l1 = fma(P.cx[1], p1.x, l1); l1 = fma(P.cx[2], p1.y, l1); l1 = fma(P.cx[3], p2.x, l1);
                    l1 = fma(P.cx[4], p2.y, l1); l1 = fma(P.cx[5], p3.x, l1); l1 = fma(P.cx[6], p3.y, l1);
                    acc[ph][a][0] += l0 + r0;
                    acc[ph][a][1] += l1 + r1;
                }
                double ys[AY][2];
#pragma unroll
                for (int a = 0; a < AY; ++a) ys[a][0] = ys[a][1] = 0.0;
#pragma unroll
                for (int rr = -R; rr < AY + R; ++rr) {
                    const double2 yv = (rr >= 0 && rr < AY) ? own[rr >= 0 && rr < AY ? rr : 0]
                                                            : lds2(st + xo[3] + rr * (int)pitchB);
#pragma unroll
                    for (int a = 0; a < AY; ++a) {
                        const int dist = rr > a ? rr - a : a - rr;
                        if (dist >= 1 && dist <= R) {
                            if (rr < a) {      // lower rows go to the side chain, upper rows to the accumulator
                                ys[a][0] = fma(P.cy[dist], yv.x, ys[a][0]);
                                ys[a][1] = fma(P.cy[dist], yv.y, ys[a][1]);
                            } else {
                                acc[ph][a][0] = fma(P.cy[dist], yv.x, acc[ph][a][0]);
                                acc[ph][a][1] = fma(P.cy[dist], yv.y, acc[ph][a][1]);
                            }
                        }
                    }
                }
#pragma unroll
                for (int a = 0; a < AY; ++a) { acc[ph][a][0] += ys[a][0]; acc[ph][a][1] += ys[a][1]; }
            }
            double2 pv[AY];
            if (HAS_PREV && do_store) {
#pragma unroll
                for (int a = 0; a < AY; ++a) pv[a] = lds2(st + tile_off + P.tile_bytes + a * tile_pitchB);
            }
            // ---- this stage is free again ---------------------------------------------------------------------
            __syncwarp();
            if (lane == 0) mbar_arrive(&bar_empty[stage]);
            if (++stage == P.nstage) { stage = 0; phase ^= 1u; }

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
                        *reinterpret_cast<double2 *>(out_z + a * NX) = o;
                    }
                }
            }
            out_z += plane;
            ++s;
        }
    }
}

typedef StencilTileChoice TileChoice;

constexpr int SMEM_PER_SM = 227 * 1024;

typedef void (*StencilKernel)(const CUtensorMap, const CUtensorMap, const CUtensorMap, const TmaParams);

// compile-time pitch variants: (input-plane pitch W, tile pitch nx); variant 0 is the run-time-pitch kernel
constexpr int N_VARIANTS = 4;
constexpr int VAR_W[N_VARIANTS] = {0, 48, 64, 96};
constexpr int VAR_NX[N_VARIANTS] = {0, 48, 60, 96};

template <int AYV, bool HP>
StencilKernel pick_variant(int v)
{
    switch (v) {
    case 1: return stencil_tma_kernel<AYV, VAR_W[1], VAR_NX[1], HP>;
    case 2: return stencil_tma_kernel<AYV, VAR_W[2], VAR_NX[2], HP>;
    case 3: return stencil_tma_kernel<AYV, VAR_W[3], VAR_NX[3], HP>;
    default: return stencil_tma_kernel<AYV, 0, 0, HP>;
    }
}

StencilKernel pick_kernel(int ay, int variant, bool has_prev)
{
    if (ay == 1) return has_prev ? pick_variant<1, true>(variant) : pick_variant<1, false>(variant);
    return has_prev ? pick_variant<2, true>(variant) : pick_variant<2, false>(variant);
}

// Tile rows TY: a multiple of 6 (TMA box rows) and of AY dividing ny.  Preference: the tallest tile whose CTA still
// fits at least twice on an SM (the kernels are register-limited), else the smallest valid tile.  The ring depth is
// whatever the per-CTA share of shared memory allows.
bool compute_tile(const sparc_gpu_ctx *ctx, TileChoice *tc)
{
    const int nx = ctx->n[0], ny = ctx->n[1];
    const int ntx = nx / 2;
    const bool per_x = ctx->bc[0] == 0;
    const int ay = ctx->opt_stencil_ay == 1 ? 1 : 2;
    const int max_threads = ay == 1 ? MAX_THREADS_AY1 : MAX_THREADS_AY2;
    const int max_warps_sm = ay == 1 ? 21 : 12;                       // 65536 / (regs per thread * 32)
    // candidates: maximise the consumer threads resident per SM; among near-ties take the smallest tile with a halo
    // factor (TY + 12) / TY <= 2 (more CTAs per SM, shorter tail), else the tallest (measured, profiles/)
    int ty = 0, best_useful = 0;
    for (int pass = 0; pass < 2; ++pass) {
        int pick_small = 0, pick_large = 0;
        for (int t = BOX_ROWS; t <= ny; t += BOX_ROWS) {
            if (ny % t || t % ay) continue;
            if (ctx->opt_stencil_ty > 0 && t != ctx->opt_stencil_ty) continue;
            const int cons = ntx * (t / ay);
            const int threads = 32 + (cons + 31) / 32 * 32;
            if (threads > max_threads) continue;
            const int useful = std::max(1, max_warps_sm / (threads / 32)) * cons;
            if (pass == 0) { best_useful = std::max(best_useful, useful); continue; }
            if (useful * 20 < best_useful * 19) continue;
            if (t >= 2 * R && !pick_small) pick_small = t;
            pick_large = t;
        }
        if (pass == 1) ty = pick_small ? pick_small : pick_large;
    }
    if (!ty) return false;
    tc->AY = ay;
    tc->TY = ty;
    tc->threads = 32 + (ntx * (ty / ay) + 31) / 32 * 32;
    tc->W = (int)round_up_i64(per_x ? nx : nx + 2 * R, 8);
    tc->variant = 0;
    for (int v = 1; v < N_VARIANTS; ++v)
        if (VAR_W[v] == tc->W && VAR_NX[v] == nx) tc->variant = v;
    tc->psi_bytes = (uint32_t)(tc->W * (ty + 2 * R) * 8);
    tc->tile_bytes = (uint32_t)round_up_i64((int64_t)ty * nx * 8, 128);
    tc->stage_bytes = tc->psi_bytes + 2 * tc->tile_bytes;
    StencilKernel kern = pick_kernel(ay, tc->variant, true);
    for (int ctas = 5; ctas >= 1; --ctas) {
        const int64_t budget = SMEM_PER_SM / ctas - 1024 - 512;
        int nstage = (int)std::min<int64_t>(MAX_STAGES, budget / tc->stage_bytes);
        nstage = std::min(nstage, ctx->opt_stencil_stages > 0 ? ctx->opt_stencil_stages : 3);   // deeper rings measured slower
        if (nstage < 2 || (nstage < 3 && ctas > 1)) continue;
        const size_t smem = 512 + (size_t)nstage * tc->stage_bytes;
        int occ = 0;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, tc->threads, smem) != cudaSuccess) {
            (void)cudaGetLastError();
            continue;
        }
        if (occ < ctas && ctas > 1) continue;
        if (occ < 1) continue;
        tc->nstage = nstage;
        tc->ctas_per_sm = std::min(occ, ctas);
        tc->smem = smem;
        return true;
    }
    return false;
}

// the choice depends only on the grid, the boundary flags and the stencil_* options: computed once per context
// (sparc_gpu_set_option invalidates it), so a degree step costs no occupancy queries
bool choose_tile(const sparc_gpu_ctx *ctx, TileChoice *tc)
{
    if (ctx->tma_choice.valid == 0) {
        TileChoice t;
        t.valid = compute_tile(ctx, &t) ? 1 : -1;
        ctx->tma_choice = t;
    }
    *tc = ctx->tma_choice;
    return tc->valid == 1;
}

bool a16(const void *p) { return ((uintptr_t)p & 15) == 0; }

// (x, y, z[, column]) tensor map over an N_d x ncols column-major block; box = bx x by x 1 [x 1]
bool encode_map(const sparc_gpu_ctx *ctx, CUtensorMap *tm, const void *base, int rank, int64_t ncols, int64_t ld, int bx,
                int by)
{
    return encode_grid_map(ctx->fn_encode_tiled, tm, base, ctx->n, rank, ncols, ld, bx, by);
}

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
    return choose_tile(ctx, &tc);
}

int launch_stencil_tma(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, double *Out, int64_t ldo, const double *Prev,
                       int64_t ldp, int64_t ncols, double alpha, double shift, double beta, cudaStream_t st)
{
    const bool has_prev = (beta != 0.0) && Prev;
    if (!stencil_tma_supported(ctx, X, ldx, Out, ldo, has_prev ? Prev : nullptr, ldp)) return SPARC_GPU_UNSUPPORTED;
    const int nx = ctx->n[0], ny = ctx->n[1], nz = ctx->n[2];
    TileChoice tc;
    choose_tile(ctx, &tc);

    TmaParams P;
    for (int p = 0; p <= R; ++p) { P.cx[p] = alpha * ctx->coef.cx[p]; P.cy[p] = alpha * ctx->coef.cy[p]; P.cz[p] = alpha * ctx->coef.cz[p]; }
    P.c0a = alpha * (ctx->coef.c0 + shift);
    P.alpha = alpha; P.beta = beta;
    P.ldo = ldo;
    P.nx = nx; P.ny = ny; P.nz = nz;
    P.per_x = ctx->bc[0] == 0; P.per_y = ctx->bc[1] == 0; P.per_z = ctx->bc[2] == 0;
    P.W = tc.W;
    P.x_start = P.per_x ? 0 : -R;
    P.TY = tc.TY;
    P.ntx = nx / 2;
    P.n_consumers = P.ntx * (tc.TY / tc.AY);
    P.nstage = tc.nstage;
    P.ytiles = ny / tc.TY;
    P.psi_bytes = tc.psi_bytes; P.tile_bytes = tc.tile_bytes; P.stage_bytes = tc.stage_bytes;

    CUtensorMap tmap_v;
    if (!encode_map(ctx, &tmap_v, ctx->d_veff, 3, 1, ctx->nd, nx, tc.TY)) return SPARC_GPU_CUDA_ERROR;
    StencilKernel kern = pick_kernel(tc.AY, tc.variant, has_prev);
    SPARC_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tc.smem));

    const int64_t max_cols_per_launch = std::max<int64_t>(1, (int64_t)INT32_MAX / ((int64_t)P.ytiles * nz));
    for (int64_t j0 = 0; j0 < ncols; j0 += max_cols_per_launch) {
        const int64_t nb = std::min<int64_t>(max_cols_per_launch, ncols - j0);
        // z chunks: split the march only as far as needed to give the chip about two waves of CTAs
        int zchunks = 1;
        const int64_t base = nb * P.ytiles;
        const int64_t want = 2LL * ctx->sm_count * tc.ctas_per_sm;
        if (base < want) zchunks = (int)std::min<int64_t>((want + base - 1) / base, std::max(1, nz / 12));
        if (ctx->opt_stencil_zchunks > 0) zchunks = std::min(ctx->opt_stencil_zchunks, nz);
        P.zchunk_len = (nz + zchunks - 1) / zchunks;
        P.zchunks = (nz + P.zchunk_len - 1) / P.zchunk_len;
        P.out = Out + j0 * ldo;

        CUtensorMap tmap_x, tmap_p;
        if (!encode_map(ctx, &tmap_x, X + j0 * ldx, 4, nb, ldx, tc.W, BOX_ROWS)) return SPARC_GPU_CUDA_ERROR;
        if (!encode_map(ctx, &tmap_p, has_prev ? Prev + j0 * ldp : X + j0 * ldx, 4, nb, has_prev ? ldp : ldx, nx, tc.TY))
            return SPARC_GPU_CUDA_ERROR;

        const unsigned grid = (unsigned)(nb * P.ytiles * P.zchunks);
        prof_begin(ctx, KK_STENCIL_TMA, st);
        kern<<<grid, tc.threads, tc.smem, st>>>(tmap_x, tmap_v, tmap_p, P);
        prof_end(ctx, KK_STENCIL_TMA, st);
    }
    SPARC_CUDA_TRY(cudaGetLastError());
    return SPARC_GPU_SUCCESS;
}
