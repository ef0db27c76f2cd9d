// stencil_dmma.cu -- hybrid fused local pass: the in-plane (x, y) taps of the radius-6 stencil on the FP64 tensor pipe,
// the z taps and the pointwise terms on the FP64 FMA pipe.
//     Out = alpha (H_loc X + shift X) + beta Prev,   H_loc = -1/2 Laplacian(radius 6) + Veff
//
// Same data path as stencil_tma.cu (producer warp, TMA ring of input planes + Veff / Prev tiles, z march with 13 partial
// sums per point in registers).  What changes is the in-plane part: a warp owns an 8 (y) x 8 (x) block of outputs and
// evaluates
//     y taps:  C[y_out, x] += T_y[y_out, y_in] . In[y_in, x]        (A = 8 x 20 banded Toeplitz constants, B = data)
//     x taps:  C[y, x_out] += In[y, x_in] . T_x[x_in, x_out]        (A = data, B = 20 x 8 banded Toeplitz constants)
// as 5 + 5 DMMA.8x8x4 with the partial z-sum of the centre plane as accumulator.  Both products leave lane (r, c) of
// the warp with row y0 + r, columns x0 + 2c, x0 + 2c + 1 -- the two points whose z-sums that lane keeps.  The band is
// 13 / 20 dense, so the tensor pipe does 1.5 x the arithmetic, but one instruction replaces 8 DFMA-pairs and 8 shared-
// memory loads per point pair become 10 LDS.64 per 64 points: the DFMA version is bound by instruction latency at 10-11
// warps per SM (168 registers), not by either pipe (profiles/r01b_ncu_kernels_cfg1.md).
// Shared-memory row pitch W = 4 or 12 mod 16 doubles: the x-tap fragments (8 rows x 4 consecutive x) are conflict-free,
// the y-tap fragments (4 rows x 8 consecutive x) 2-way.
#include <cuda.h>

#include <algorithm>

#include "internal.h"
#include "sm100_ptx.cuh"

namespace {

constexpr int R = 6;
constexpr int NSLOT = 2 * R + 1;
constexpr int TB = 8;              // rows of one DMMA m-tile; a CTA tile has TYB of them (TY = 8 TYB rows)
constexpr int KS = 5;              // k-steps of 4 over the 20-wide input window
constexpr int MAX_STAGES = 8;

struct DmParams {
    double cx[R + 1], cy[R + 1], cz[R + 1];   // alpha * (-1/2 w_p / h^2)
    double c0a;                                // alpha * (c0 + shift)
    double rxy;                                // cx[p] / cy[p] = (h_y / h_x)^2: one Toeplitz fragment set serves both axes
    double alpha, beta;
    double *out;
    int64_t ldo;
    int nx, ny, nz;
    int W;            // smem row pitch in doubles (all three tiles)
    int x_start;      // first x coordinate of the boxes: 0 (periodic x) or -6 (Dirichlet x)
    int nwarps;       // consumer warps = TYB * nxb
    int nxb;          // x blocks = ceil(nx / 8): the last one may overhang the grid (its extra columns are not stored)
    int nstage;
    int ytiles, zchunks, zchunk_len;
    int per_x, per_y, per_z;
    uint32_t psi_bytes, tile_bytes, stage_bytes;
    // x tiling (grids wider than 96 points): nxt tiles of xt columns (a multiple of 8; the last may overhang); every tile then
    // stores 6 halo columns on either side (x_start = tile start - 6); on a periodic x axis the first / last tile gets the
    // wrapped columns as two extra 8-column boxes behind the Veff / Prev tiles
    int nxt, xt;
    uint32_t halo_bytes;      // one 8-column x TY-row halo box
};

using namespace sm100;


template <bool HAS_PREV, int TYB, int MINB>
__global__ void __launch_bounds__(MINB == 1 ? 13 * 32 : 7 * 32, MINB)
stencil_dmma_kernel(const __grid_constant__ CUtensorMap tmap_x8,
                    const __grid_constant__ CUtensorMap tmap_v, const __grid_constant__ CUtensorMap tmap_p,
                    const __grid_constant__ CUtensorMap tmap_h, const __grid_constant__ DmParams P)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t *bar_full = reinterpret_cast<uint64_t *>(smem_raw);    // [MAX_STAGES] TMA landed
    uint64_t *bar_empty = bar_full + MAX_STAGES;                    // [MAX_STAGES] consumers done
    const uint32_t stage0 = (smem_u32(smem_raw) + 2 * MAX_STAGES * 8 + 127u) & ~127u;

    constexpr int TY = TB * TYB;
    const int tid = threadIdx.x;
    if (tid == 0) {
        for (int s = 0; s < P.nstage; ++s) {
            mbar_init(&bar_full[s], 1);
            mbar_init(&bar_empty[s], (uint32_t)P.nwarps);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const int per_col = P.ytiles * P.zchunks * P.nxt;
    const int col = blockIdx.x / per_col;
    int rem = blockIdx.x - col * per_col;
    const int xtile = rem % P.nxt;               // x tiles of one (column, y tile, z chunk) are neighbours in the grid
    rem /= P.nxt;
    const int ytile = rem / P.zchunks;
    const int zc = rem - ytile * P.zchunks;
    const bool tiled = P.nxt > 1;
    const int xt0 = xtile * P.xt;
    const bool halo_l = tiled && P.per_x && xtile == 0, halo_r = tiled && P.per_x && xtile == P.nxt - 1;
    const uint32_t halo_off = P.psi_bytes + 2 * P.tile_bytes;     // left box, then right box
    const int y0 = ytile * TY;
    const int z0 = zc * P.zchunk_len;
    const int z1 = min(z0 + P.zchunk_len, P.nz);
    const int nzc = z1 - z0;
    const int nsteps = nzc + 2 * R;          // input planes z0-6 .. z1+5
    const int W = P.W;

    if (tid < 32) {
        // ================================ producer warp (one lane) =======================================
        if (tid != 0) return;
        prefetch_tmap(&tmap_x8);
        prefetch_tmap(&tmap_v);
        if (HAS_PREV) prefetch_tmap(&tmap_p);
        const int xs = tiled ? xt0 - R : P.x_start, xv = tiled ? xt0 : 0;
        const uint32_t row_bytes = (uint32_t)(W * 8);
        const uint32_t tile_tx = (uint32_t)(TY * W * 8);
        // TYB + 2 boxes of 8 rows (128-byte aligned destinations): rows y0-8 .. y0-1 (6 used), the tile, y0+TY ..
        // y0+TY+7 (6 used); the halo boxes wrap as a whole on a periodic y axis, rows outside a Dirichlet face are
        // zero-filled
        int yt = y0 - TB, yb = y0 + TY;
        if (P.per_y) { if (yt < 0) yt += P.ny; if (yb >= P.ny) yb -= P.ny; }
        int stage = 0;
        uint32_t phase = 0;
        for (int s = 0; s < nsteps; ++s) {
            if (s >= P.nstage) {
                while (!mbar_try_wait(&bar_empty[stage], phase ^ 1u)) __nanosleep(40);
            }
            const bool do_xy = (s >= R) && (s < R + nzc);
            const bool do_prev = HAS_PREV && (s >= 2 * R);
            int zin = z0 - R + s;
            if (P.per_z) { if (zin < 0) zin += P.nz; else if (zin >= P.nz) zin -= P.nz; }
            const uint32_t dst = stage0 + (uint32_t)stage * P.stage_bytes;
            mbar_arrive_expect_tx(&bar_full[stage], P.psi_bytes + (do_xy ? tile_tx : 0u) + (do_prev ? tile_tx : 0u) +
                                                        ((do_xy && halo_l) ? P.halo_bytes : 0u) + ((do_xy && halo_r) ? P.halo_bytes : 0u));
            tma_load_4d(dst, &tmap_x8, &bar_full[stage], xs, yt, zin, col);
#pragma unroll
            for (int j = 0; j < TYB; ++j)
                tma_load_4d(dst + (1 + j) * TB * row_bytes, &tmap_x8, &bar_full[stage], xs, y0 + TB * j, zin, col);
            tma_load_4d(dst + (1 + TYB) * TB * row_bytes, &tmap_x8, &bar_full[stage], xs, yb, zin, col);
            if (do_xy) tma_load_3d(dst + P.psi_bytes, &tmap_v, &bar_full[stage], xv, y0, z0 - R + s);
            if (do_prev) tma_load_4d(dst + P.psi_bytes + P.tile_bytes, &tmap_p, &bar_full[stage], xv, y0, z0 - 2 * R + s, col);
            // wrapped x halo of the centre plane's tile rows: columns nx-8 .. nx-1 (left), 0 .. 7 (right)
            if (do_xy && halo_l) tma_load_4d(dst + halo_off, &tmap_h, &bar_full[stage], P.nx - 8, y0, zin, col);
            if (do_xy && halo_r) tma_load_4d(dst + halo_off + P.halo_bytes, &tmap_h, &bar_full[stage], 0, y0, zin, col);
            if (++stage == P.nstage) { stage = 0; phase ^= 1u; }
        }
        return;
    }

    // ==================================== consumer warps ====================================================
    const int cw = (tid >> 5) - 1;             // (row block, 8-wide x block) of this warp
    if (cw >= P.nwarps) return;
    const int lane = tid & 31, lq = lane & 3, lr = lane >> 2;
    const int rb = cw / P.nxb;                  // 8-row block of the tile
    const int x0 = 8 * (cw - rb * P.nxb);
    const int ry = TB * rb;
    const bool xvalid = xt0 + x0 + 2 * (lane & 3) < P.nx;       // n_x is even: a lane's pair is inside or outside as a whole
    const int xoff = (P.per_x && !tiled) ? 0 : R;    // halo columns are stored for a Dirichlet x axis and for x tiles
    // Toeplitz fragments: tap distance d = (k - 6) - (output index), k = 4 s + lq; the centre tap is pointwise
    double ay[KS];                              // (the x fragments are rxy times the same numbers)
    uint32_t xa[KS];                            // byte offsets of the x-tap data fragments (row y0 + lr, wrapped column)
#pragma unroll
    for (int s = 0; s < KS; ++s) {
        const int d = 4 * s + lq - R - lr;
        const int ad = d < 0 ? -d : d;
        ay[s] = (ad >= 1 && ad <= R) ? P.cy[ad] : 0.0;
        int xc = x0 - R + 4 * s + lq;
        if (!tiled) {
            if (P.per_x) { if (xc < 0) xc += P.nx; else if (xc >= P.nx) xc -= P.nx; }
            else xc += R;
            xa[s] = (uint32_t)(((TB + ry + lr) * W + xc) * 8);
        } else {
            const int xg = xt0 + xc;                                        // global column of this fragment element
            if (halo_l && xg < 0) xa[s] = halo_off + (uint32_t)(((ry + lr) * 8 + xg + 8) * 8);
            else if (halo_r && xg >= P.nx && xg < P.nx + 8) xa[s] = halo_off + P.halo_bytes + (uint32_t)(((ry + lr) * 8 + xg - P.nx) * 8);
            else xa[s] = (uint32_t)(((TB + ry + lr) * W + xc + R) * 8);    // inside the box (zero-filled outside a Dirichlet face)
        }
    }
    const uint32_t ya0 = (uint32_t)(((TB - R + ry + lq) * W + x0 + lr + xoff) * 8);      // row y0 + ry - 6 + lq, + s * 4 rows
    const uint32_t ystep = (uint32_t)(4 * W * 8);
    const uint32_t own_off = (uint32_t)(((TB + ry + lr) * W + x0 + 2 * lq + xoff) * 8);
    const uint32_t tile_off = P.psi_bytes + (uint32_t)(((ry + lr) * W + x0 + 2 * lq) * 8);
    const int64_t plane = (int64_t)P.nx * P.ny;
    double *out_z = P.out + (int64_t)col * P.ldo + (int64_t)(y0 + ry + lr) * P.nx + xt0 + x0 + 2 * lq + (int64_t)(z0 - 2 * R) * plane;

    double acc[NSLOT][2];
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) acc[s][0] = acc[s][1] = 0.0;

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
            const double2 own = lds2(st + own_off);
            // ---- in-plane taps of the plane this one is the centre of: 5 + 5 DMMA into its partial z-sum ------
            if (do_xy) {
                double fy[KS], fx[KS];
#pragma unroll
                for (int k = 0; k < KS; ++k) {
                    fy[k] = lds1(st + ya0 + k * ystep);
                    fx[k] = lds1(st + xa[k]);
                }
                const double2 vf = lds2(st + tile_off);
                // this plane's own slot was opened by the plane six steps back (or is the first use in the chunk)
                double c0 = acc[ph][0], c1 = acc[ph][1], e0 = 0.0, e1 = 0.0;
#pragma unroll
                for (int k = 0; k < KS; ++k) {
                    dmma884(c0, c1, ay[k], fy[k]);        // y taps: constants x data
                    dmma884(e0, e1, fx[k], ay[k]);        // x taps: data x constants (second chain), scaled below
                }
                acc[ph][0] = c0 + fma(P.rxy, e0, fma(P.alpha, vf.x, P.c0a) * own.x);
                acc[ph][1] = c1 + fma(P.rxy, e1, fma(P.alpha, vf.y, P.c0a) * own.y);
            }
            // ---- z taps: this plane feeds the 12 neighbouring output planes --------------------------------------
#pragma unroll
            for (int d = -R; d <= R; ++d) {
                if (d == 0) continue;
                const int slot = (ph - d + NSLOT) % NSLOT;
                const double c = P.cz[d < 0 ? -d : d];
                if (d == -R) {            // first contribution to output plane zin + 6: opens the slot
                    acc[slot][0] = c * own.x;
                    acc[slot][1] = c * own.y;
                } else {
                    acc[slot][0] = fma(c, own.x, acc[slot][0]);
                    acc[slot][1] = fma(c, own.y, acc[slot][1]);
                }
            }
            double2 pv = make_double2(0.0, 0.0);
            if (HAS_PREV && do_store) pv = lds2(st + tile_off + P.tile_bytes);
            __syncwarp();
            if (lane == 0) mbar_arrive(&bar_empty[stage]);
            if (++stage == P.nstage) { stage = 0; phase ^= 1u; }

            // ---- output plane zin - 6 has all 37 taps: recurrence axpy + store ---------------------------------
            if (do_store) {
                const int cs = (ph + R + 1) % NSLOT;
                double2 o;
                o.x = HAS_PREV ? fma(P.beta, pv.x, acc[cs][0]) : acc[cs][0];
                o.y = HAS_PREV ? fma(P.beta, pv.y, acc[cs][1]) : acc[cs][1];
                if (xvalid) *reinterpret_cast<double2 *>(out_z) = o;
            }
            out_z += plane;
            ++s;
        }
    }
}

// (x, y, z[, column]) tensor map over an N_d x ncols column-major block; box = bx x by x 1 [x 1]
bool encode_map(const sparc_gpu_ctx *ctx, CUtensorMap *tm, const void *base, int rank, int64_t ncols, int64_t ld, int bx,
                int by)
{
    return encode_grid_map(ctx->fn_encode_tiled, tm, base, ctx->n, rank, ncols, ld, bx, by);
}

// smallest pitch >= need with pitch mod 16 in {4, 12}: 8 rows x 4 consecutive doubles then tile all 32 banks
int pick_pitch(int need)
{
    int w = need;
    while (!((w % 16) == 4 || (w % 16) == 12)) ++w;
    return w;
}

bool a16(const void *p) { return ((uintptr_t)p & 15) == 0; }

}  // namespace

bool stencil_dmma_supported(const sparc_gpu_ctx *ctx, const double *X, int64_t ldx, const double *Out, int64_t ldo,
                            const double *Prev, int64_t ldp)
{
    if (!ctx->fn_encode_tiled || ctx->radius != R) return false;
    const int nx = ctx->n[0], ny = ctx->n[1];
    if (nx % 2 || nx < 16) return false;                     // wider than 96 points: x tiles
    if (ny % TB || ny < 2 * TB) return false;
    if (nx <= 96 && pick_pitch((nx + 7) / 8 * 8 + (ctx->bc[0] == 0 ? 0 : 2 * R)) > 256) return false;
    if (!a16(X) || !a16(Out) || (Prev && !a16(Prev)) || (ldx & 1) || (ldo & 1) || (Prev && (ldp & 1))) return false;
    return true;
}

int launch_stencil_dmma(sparc_gpu_ctx *ctx, const double *X, int64_t ldx, double *Out, int64_t ldo, const double *Prev,
                        int64_t ldp, int64_t ncols, double alpha, double shift, double beta, cudaStream_t st)
{
    const bool has_prev = (beta != 0.0) && Prev;
    if (!stencil_dmma_supported(ctx, X, ldx, Out, ldo, has_prev ? Prev : nullptr, ldp)) return SPARC_GPU_UNSUPPORTED;
    const int nx = ctx->n[0], ny = ctx->n[1], nz = ctx->n[2];
    DmParams P;
    for (int p = 0; p <= R; ++p) { P.cx[p] = alpha * ctx->coef.cx[p]; P.cy[p] = alpha * ctx->coef.cy[p]; P.cz[p] = alpha * ctx->coef.cz[p]; }
    P.c0a = alpha * (ctx->coef.c0 + shift);
    P.rxy = (ctx->h[1] * ctx->h[1]) / (ctx->h[0] * ctx->h[0]);
    P.alpha = alpha; P.beta = beta;
    P.ldo = ldo;
    P.nx = nx; P.ny = ny; P.nz = nz;
    P.per_x = ctx->bc[0] == 0; P.per_y = ctx->bc[1] == 0; P.per_z = ctx->bc[2] == 0;
    // x tiling for grids wider than 96 points (12 consumer warps): tile width a multiple of 8.  Measured at n_x = 128 (config 5,
    // stencil only): 2 x 64 and 4 x 32 reach 3.7 TB/s, 3 x 48 (16 columns of overhang) 3.3, 2 x 96 (64 of overhang) 3.0 -- the
    // overhang of the last tile costs more than anything else, 8 resident consumer warps are enough, and every tile re-reads
    // 12 halo columns
    P.nxt = 1; P.xt = 8 * ((nx + 7) / 8);
    if (nx > 96) {
        double best = -1.0;
        for (int xt = 96; xt >= 32; xt -= 8) {
            const int nxt = (nx + xt - 1) / xt, warps = xt / 8;
            const double useful = nx / ((double)nxt * xt);
            const double score = std::min((warps <= 6 ? 2.0 : 1.0) * warps, 8.0) * useful * useful * useful * xt / (xt + R);
            if (score > best) { best = score; P.xt = xt; P.nxt = nxt; }
        }
        if (ctx->opt_stencil_xt >= 32 && ctx->opt_stencil_xt <= 96 && ctx->opt_stencil_xt % 8 == 0) {
            P.xt = ctx->opt_stencil_xt; P.nxt = (nx + P.xt - 1) / P.xt;
        }
    }
    const bool tiled = P.nxt > 1;
    P.W = pick_pitch(P.xt + ((P.per_x && !tiled) ? 0 : 2 * R));
    P.x_start = (P.per_x && !tiled) ? 0 : -R;
    // 16-row tiles (a third less halo traffic) when 2 nx / 8 consumer warps still fit the 12-warp kernel
    const int nxb = P.xt / 8;
    const int tyb = (ctx->opt_stencil_ty == 16 && ny % (2 * TB) == 0 && 2 * nxb <= 12) ? 2 : 1;
    const int TY = TB * tyb;
    P.nxb = nxb;
    P.nwarps = tyb * P.nxb;
    P.ytiles = ny / TY;
    P.psi_bytes = (uint32_t)((tyb + 2) * TB * P.W * 8);
    P.tile_bytes = (uint32_t)(TY * P.W * 8);
    P.halo_bytes = (uint32_t)(8 * TY * 8);
    P.stage_bytes = P.psi_bytes + 2 * P.tile_bytes + ((tiled && P.per_x) ? 2 * P.halo_bytes : 0u);
    const int threads = (P.nwarps + 1) * 32;
    // one 8-row block and up to 6 consumer warps: two CTAs per SM (128 registers; a third would need <= 80 and spills the
    // z-sums); otherwise one CTA of up to 12 consumer warps.  The kernel's TYB must be the one the parameters (boxes per
    // stage, y tiles, warps) were built for, so it is chosen from tyb first.
    const bool small = tyb == 1 && P.nwarps <= 6;
    typedef void (*Kern)(const CUtensorMap, const CUtensorMap, const CUtensorMap, const CUtensorMap, const DmParams);
    Kern kern = tyb == 2 ? (has_prev ? (Kern)stencil_dmma_kernel<true, 2, 1> : (Kern)stencil_dmma_kernel<false, 2, 1>)
                : small  ? (has_prev ? (Kern)stencil_dmma_kernel<true, 1, 2> : (Kern)stencil_dmma_kernel<false, 1, 2>)
                         : (has_prev ? (Kern)stencil_dmma_kernel<true, 1, 1> : (Kern)stencil_dmma_kernel<false, 1, 1>);
    // ring depth: as deep as shared memory allows (one or two CTAs per SM by registers); the kernel waits on TMA data
    // more than on anything else
    const int ctas = small ? 2 : 1;
    int nstage = (int)std::min<int64_t>(ctx->opt_stencil_stages > 0 ? ctx->opt_stencil_stages : 6,
                                        (227 * 1024 / ctas - 2048) / P.stage_bytes);
    nstage = std::min(nstage, MAX_STAGES);
    if (nstage < 2) return SPARC_GPU_UNSUPPORTED;
    P.nstage = nstage;
    const size_t smem = 512 + (size_t)nstage * P.stage_bytes;
    // once per context and kernel variant (the attribute is per device and function; the maximum any launch may ask for)
    const int vbit = 20 + (tyb == 2 ? 0 : small ? 2 : 4) + (has_prev ? 1 : 0);
    if (!(ctx->func_attr_done & (1ull << vbit))) {
        SPARC_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        ctx->func_attr_done |= 1ull << vbit;
    }

    CUtensorMap tmap_v;
    if (!encode_map(ctx, &tmap_v, ctx->d_veff, 3, 1, ctx->nd, P.W, TY)) return SPARC_GPU_CUDA_ERROR;   // whole tile
    const int64_t max_cols_per_launch = std::max<int64_t>(1, (int64_t)INT32_MAX / ((int64_t)P.ytiles * nz * P.nxt));
    for (int64_t j0 = 0; j0 < ncols; j0 += max_cols_per_launch) {
        const int64_t nb = std::min<int64_t>(max_cols_per_launch, ncols - j0);
        int zchunks = 1;
        const int64_t base = nb * P.ytiles * P.nxt;
        const int64_t want = 2LL * ctx->sm_count * ctas;
        if (base < want) zchunks = (int)std::min<int64_t>((want + base - 1) / base, std::max(1, nz / 12));
        if (ctx->opt_stencil_zchunks > 0) zchunks = std::min(ctx->opt_stencil_zchunks, nz);
        P.zchunk_len = (nz + zchunks - 1) / zchunks;
        P.zchunks = (nz + P.zchunk_len - 1) / P.zchunk_len;
        P.out = Out + j0 * ldo;
        CUtensorMap tmap_x, tmap_p, tmap_h;
        if (!encode_map(ctx, &tmap_x, X + j0 * ldx, 4, nb, ldx, P.W, TB)) return SPARC_GPU_CUDA_ERROR;
        if (!encode_map(ctx, &tmap_h, X + j0 * ldx, 4, nb, ldx, 8, TY)) return SPARC_GPU_CUDA_ERROR;
        if (!encode_map(ctx, &tmap_p, has_prev ? Prev + j0 * ldp : X + j0 * ldx, 4, nb, has_prev ? ldp : ldx, P.W, TY))
            return SPARC_GPU_CUDA_ERROR;
        const unsigned grid = (unsigned)(nb * P.ytiles * P.zchunks * P.nxt);
        prof_begin(ctx, KK_STENCIL_TMA, st);
        kern<<<grid, threads, smem, st>>>(tmap_x, tmap_v, tmap_p, tmap_h, P);
        prof_end(ctx, KK_STENCIL_TMA, st);
    }
    SPARC_CUDA_TRY(cudaGetLastError());
    return SPARC_GPU_SUCCESS;
}
