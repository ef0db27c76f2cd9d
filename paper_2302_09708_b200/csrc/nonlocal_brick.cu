// nonlocal_brick.cu -- brick-tiled Kleinman-Bylander nonlocal term on the FP64 tensor pipe (default nonlocal path).
//
//   V_nl X = sum_J S_J^T chi_J diag(gamma_J) chi_J^T S_J X
//
// The per-atom formulation gathers X at each atom's support and scatter-adds with atomics: 8c + 16c bytes and one
// atomic per (support row, column) (c = coverage, 4-5 at configs 3-4).  Here the grid is cut into bricks of 128
// points (BX x BY x BZ, x fastest) and one CTA owns (brick, NC columns): it reads the 128 x NC tile of Out once into
// tensor-core accumulator fragments, adds the contribution of EVERY atom whose support meets the brick
// ("pull": Out^T[col, pt] += D_J^T[col, q] chi_J^T[q, pt], DMMA m8n8k4), writes the tile back once, and -- the tile
// now being the final Psi_{k+1} -- contracts it with the same chi blocks for the NEXT degree step
// ("project": C_J[q, col] += chi_J^T[q, pt] Out[pt, col]), so that the nonlocal term costs one 16 B read-modify-write
// of Out per degree step.  The accumulator fragment of the pull is, register for register, the B operand of the
// projection (k index = point pair), so no layout change is needed.
//
// Work decomposition inside a CTA (round 2): the brick is 16 "octets" of 2 x 2 x 2 points (cubes follow the spherical
// supports more closely than 8-point rods: 0.83 instead of 0.69 of the DMMA columns carry a support point at config 3);
// a consumer warp owns one HALF of the brick (8 octets) times 16 columns, i.e. two independent 8-column DMMA chains per
// chi block: every chi fragment read from shared memory feeds two DMMAs, and a warp always has two (pull) or four
// (project) accumulator chains in flight.
//
// Tables built at create (host): for every (brick, atom) pair a 16-bit mask of the octets the atom touches, and per
// touched octet a dense block of chi values already permuted into DMMA fragment order (zeros where the atom does not
// cover a point; gamma folded into the pull blocks).  Blocks of one (brick, atom) pair are contiguous; a producer warp
// streams them (and the NC-column slice of C_J) into a shared-memory byte ring with cp.async.bulk, ahead of the consumer
// warps (full / empty mbarriers per job slot).  The tile itself is staged by one TMA box copy each way.
//
// The 9th projector of an s+p+d atom is applied as a rank-1 FMA update beside the two k-steps of DMMA (a third
// k-step would be 3/4 padding).
#include <cuda.h>

#include <math.h>
#include <string.h>

#include <algorithm>
#include <unordered_map>
#include <vector>

#include "internal.h"
#include "sm100_ptx.cuh"

namespace {

using namespace sm100;

constexpr int NB_PTS = 128;        // points per brick
constexpr int NB_OCT = 16;         // octets (2 x 2 x 2 cubes) per brick = width of the job masks
constexpr int NB_HOCT = 8;         // octets per half brick = octets per consumer warp
constexpr int NLB_MAXJ = 32;       // (brick, atom) jobs per load round (one mbarrier each)
constexpr int NLB_WARPS = 8;       // warps per CTA: (half brick) x (4 pairs of 8-column slices) = 64 columns
constexpr int NLB_COLS = 64;

struct BrickJob {                  // one (brick, atom) pair
    int32_t atom;
    uint32_t mask;                 // bits 0-15: octets of the brick this atom touches; bits 16-24: sign bits of gamma_q
    int64_t blk0;                  // index of its first chi block
    int32_t po;                    // offset of the atom's first projector (prefix sum of P_J)
    int32_t pj;                    // P_J
};

struct BrickParams {
    const int32_t *brick_org;      // [n_active][4] origin (x0, y0, z0), union mask
    const int32_t *job_ptr;        // [n_active + 1]
    const BrickJob *jobs;
    const double *blk;             // [n_blocks][BLK] chi sqrt|gamma| in the shared fragment layout
    double *tile;                  // X (project only) or Out: N_d x ncols, ld
    int64_t ld;
    // C buffers hold D = scale sign(gamma) (chi sqrt|gamma|)_J^T Psi, one slab of SLAB doubles per (atom, 16-column group) at
    // (atom * ngroups16 + group) * SLAB, in the order of the pull's A fragments (CLayout below): the pull reads its operands
    // with two vector loads and no arithmetic
    const double *c_in;            // of the previous pass (pull)
    double *c_out;                 // accumulated by this pass (project), zeroed by the caller
    int64_t ncp;                   // padded column count of the C buffers (multiple of 64)
    int32_t ngroups16;             // ncp / 16
    int32_t ncols;
    int32_t ncolgroups;
    int32_t nx, ny, nz;
    int32_t bx, by;                // brick extent in x and y (bz = 128 / (bx by)); all even
    int32_t lhx, lhy;              // log2 of the cube counts along x and y (bx / 2, by / 2)
    int32_t cap_blocks;            // chi blocks the CTA's shared memory holds
    int32_t toct[NB_OCT];          // persistent kernel: byte offset of cube o inside a staged half tile (lane part excluded)
    double scale;                  // factor folded into c_out by the projection (the alpha of the degree step that will pull it)
    int32_t dbg;                   // timing experiments only (option "nlb_dbg"): 1 no atomics, 2 no pull math, 4 no project math
};

// One chi block = the 8 points of an octet x the projectors of one atom, stored ONCE and read as both DMMA operand
// kinds: the pull's B fragment (k = projector, n = point) and the projection's A fragment (m = projector, k = point).
//   P <= 9 class (BLK = 72): element (pt, q < 8) at rowpos(pt) * 8 + (q ^ 4 (pt & 1)), rowpos = pt with bits 0 and 1
//     swapped; element (pt, 8) at 64 + pt.  Both fragment reads (8 points x 4 projectors; 4 points of one parity x 8
//     projectors) then touch every shared-memory bank exactly twice: conflict-free 64-bit loads.
//   P <= 4 class (BLK = 32): element (pt, q) at 4 pt + q.
// Values are chi[pt, q] sqrt|gamma_q|; the sign of gamma_q travels in the job descriptor and is applied to the pull's A
// operand, so that pull(project(X)) = chi gamma chi^T X with one copy of the table.
template <bool P9> struct BlkLayout {
    static constexpr int BLK = P9 ? 72 : 32;
    __host__ __device__ static int at(int pt, int q)
    {
        if (!P9) return 4 * pt + q;
        if (q == 8) return 64 + pt;
        const int rowpos = ((pt >> 1) & 1) | ((pt & 1) << 1) | (pt & 4);
        return rowpos * 8 + (q ^ (4 * (pt & 1)));
    }
};

// Slab of the C buffers: the sums of one atom for one 16-column group, in pull-fragment order.  Slice s = columns 8 s .. 8 s + 7.
//   P <= 9 class (SLAB = 144): (q < 8, column c, slice s) at 64 s + 2 (4 c + (q & 3)) + (q >> 2): lane (lr = c, lq) of the pull
//     reads its two k-step operands (q = lq, 4 + lq) as one 16-byte vector; (q = 8, c, s) at 128 + 8 s + c.
//   P <= 4 class (SLAB = 64): (q, c, s) at 32 s + 4 c + q.
template <bool P9> struct CLayout {
    static constexpr int SLAB = P9 ? 144 : 64;
    __host__ __device__ static int at(int q, int c, int s)
    {
        if (!P9) return 32 * s + 4 * c + q;
        if (q == 8) return 128 + 8 * s + c;
        return 64 * s + 2 * (4 * c + (q & 3)) + (q >> 2);
    }
};

// Per-lane constants of a consumer warp.  A warp owns one HALF of the brick (8 cubes) times 16 columns: two 8-column
// slices, i.e. two independent DMMA chains per chi fragment read.
template <bool P9> struct WarpCtx {
    int lq, lr, half;
    uint32_t kA, kB0, kB1, kX;     // byte offsets of the lane's fragment elements inside a block
    bool bval;                     // P <= 4: projection rows 4-7 are padding
    int colw;                      // first global column of the warp
    bool cv0, cv1;                 // the lane's column of slice 0 / 1 exists
    __device__ __forceinline__ void init(int lane, int half_, int colw_, int ncols)
    {
        typedef BlkLayout<P9> L;
        lq = lane & 3; lr = lane >> 2; half = half_;
        kA = (uint32_t)L::at(lr, lq) * 8u;                    // pull B fragment, k-step 0 (k-step 1: kA ^ 32)
        const int qq = lr < (P9 ? 8 : 4) ? lr : 0;
        kB0 = (uint32_t)L::at(2 * lq, qq) * 8u; kB1 = (uint32_t)L::at(2 * lq + 1, qq) * 8u;
        kX = (uint32_t)(64 + 2 * lq) * 8u;                    // the pair of the 9th projector row
        bval = P9 || lr < 4;
        set_cols(colw_, ncols);
    }
    __device__ __forceinline__ void set_cols(int colw_, int ncols)
    {
        colw = colw_;
        cv0 = colw + lr < ncols; cv1 = colw + 8 + lr < ncols;
    }
};

// One phase (PULL: Out^T += D^T chi^T; else: C += chi^T Out) of the jobs r0 .. r1 - 1 of a brick on the warp's register
// tile c.  jobinfo[j - jbase] = (block offset in the store, octet mask | gamma signs << 16, P_J, projector offset);
// `store` is the shared-memory byte address of the block store (a multiple of 64, like the block size: the second k-step's
// fragment is then at address ^ 32); wait_full: the blocks of job j have landed when full[j - jbase] completes `parity`.
// stage != 0: the projection's 16 x P_J partial sums leave through that per-warp shared-memory slab and one bulk
// reduce-add (UBLKRED.ADD.F64) onto the atom's contiguous C slab instead of 2-3 atomics per lane.
template <bool P9, bool PULL>
__device__ __forceinline__ void run_jobs(double2 (&c)[2][NB_HOCT], const WarpCtx<P9> &w, const BrickParams &p, uint32_t store,
                                         const int4 *jobinfo, uint64_t *full, int jbase, int r0, int r1, bool wait_full,
                                         uint32_t parity, uint32_t stage = 0u)
{
    constexpr uint32_t BLKB = BlkLayout<P9>::BLK * 8;
    constexpr int KP = P9 ? 2 : 1;
    const int lq = w.lq, lr = w.lr;
    // A operands of the pull, fetched one job ahead: D_J^T[col, q], stored ready-made (scaled, signed, fragment order)
    double nA[2][KP], n8[2];
    const int64_t gslab = (int64_t)(w.colw >> 4) * CLayout<P9>::SLAB;
    auto fetch_a = [&](int j) {
        const int4 info = jobinfo[j - jbase];
        const double *cs = p.c_in + (int64_t)info.w * p.ngroups16 * CLayout<P9>::SLAB + gslab;
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            if (P9) {
                const double2 v = *reinterpret_cast<const double2 *>(cs + 64 * s + 2 * (4 * lr + lq));
                nA[s][0] = v.x; nA[s][KP - 1] = v.y;
                n8[s] = cs[128 + 8 * s + lr];
            } else {
                nA[s][0] = cs[32 * s + 4 * lr + lq];
                n8[s] = 0.0;
            }
        }
    };
    if (PULL && r0 < r1) fetch_a(r0);

#pragma unroll 1
    for (int j = r0; j < r1; ++j) {
        if (wait_full) mbar_wait(&full[j - jbase], parity);
        const int4 info = jobinfo[j - jbase];
        const uint32_t mask_all = (uint32_t)info.y & 0xffffu;
        // (the OR over the warp of a warp-uniform value: tells the compiler that the octet branches below are uniform)
        const uint32_t mask = __reduce_or_sync(0xffffffffu, (mask_all >> (NB_HOCT * w.half)) & 0xffu);
        const int PJ = info.z;
        const uint32_t blk0 = store + (uint32_t)(info.x + (w.half ? __popc(mask_all & 0xffu) : 0)) * BLKB;   // the other half's blocks come first

        if (PULL) {
            double dA[2][KP], d8[2];
#pragma unroll
            for (int ks = 0; ks < KP; ++ks) { dA[0][ks] = nA[0][ks]; dA[1][ks] = nA[1][ks]; }
            d8[0] = n8[0]; d8[1] = n8[1];
            if (j + 1 < r1) fetch_a(j + 1);
            if (mask && !(p.dbg & 2)) {
                // operands of the next block are fetched while the current block's DMMAs issue (reading one block
                // past the job's last stays inside the store + its slack)
                uint32_t aA = blk0 + w.kA, aX = blk0 + w.kX;
                double nb0 = lds1(aA), nb1 = 0.0;
                if (KP > 1) nb1 = lds1(aA ^ 32u);
                double2 nx8 = make_double2(0.0, 0.0);
                if (P9) nx8 = lds2(aX);
#pragma unroll
                for (int o = 0; o < NB_HOCT; ++o) {
                    if (mask & (1u << o)) {
                        const double b0 = nb0, b1 = nb1;
                        const double2 x8 = nx8;
                        aA += BLKB; aX += BLKB;
                        nb0 = lds1(aA);
                        if (KP > 1) nb1 = lds1(aA ^ 32u);
                        if (P9) nx8 = lds2(aX);
                        // the rank-1 update of projector 8 goes FIRST: a DFMA behind the DMMAs of the same accumulator would
                        // wait out their 26-cycle latency with the (in-order) warp unable to issue the next octet
                        if (P9) {
                            c[0][o].x = fma(d8[0], x8.x, c[0][o].x);
                            c[0][o].y = fma(d8[0], x8.y, c[0][o].y);
                            c[1][o].x = fma(d8[1], x8.x, c[1][o].x);
                            c[1][o].y = fma(d8[1], x8.y, c[1][o].y);
                        }
                        dmma884(c[0][o].x, c[0][o].y, dA[0][0], b0);
                        dmma884(c[1][o].x, c[1][o].y, dA[1][0], b0);
                        if (KP > 1) {
                            dmma884(c[0][o].x, c[0][o].y, dA[0][KP - 1], b1);
                            dmma884(c[1][o].x, c[1][o].y, dA[1][KP - 1], b1);
                        }
                    }
                }
            }
        } else if (mask && !(p.dbg & 4)) {
            // C_J[q, col] += sum_pt chi_J[pt, q] Out[pt, col]; per column slice two accumulator sets (cube parity)
            double acc[2][2][2], p8[2][2];
#pragma unroll
            for (int s = 0; s < 2; ++s)
#pragma unroll
                for (int e = 0; e < 2; ++e) { acc[s][e][0] = acc[s][e][1] = 0.0; p8[s][e] = 0.0; }
            uint32_t aB0 = blk0 + w.kB0, aB1 = blk0 + w.kB1, aX = blk0 + w.kX;
            double na0 = w.bval ? lds1(aB0) : 0.0, na1 = w.bval ? lds1(aB1) : 0.0;
            double2 nx8 = make_double2(0.0, 0.0);
            if (P9) nx8 = lds2(aX);
#pragma unroll
            for (int o = 0; o < NB_HOCT; ++o) {
                if (mask & (1u << o)) {
                    const double a0 = na0, a1 = na1;
                    const double2 x8 = nx8;
                    aB0 += BLKB; aB1 += BLKB; aX += BLKB;
                    if (w.bval) { na0 = lds1(aB0); na1 = lds1(aB1); }
                    if (P9) nx8 = lds2(aX);
                    dmma884(acc[0][o & 1][0], acc[0][o & 1][1], a0, c[0][o].x);
                    dmma884(acc[1][o & 1][0], acc[1][o & 1][1], a0, c[1][o].x);
                    dmma884(acc[0][o & 1][0], acc[0][o & 1][1], a1, c[0][o].y);
                    dmma884(acc[1][o & 1][0], acc[1][o & 1][1], a1, c[1][o].y);
                    if (P9) {
                        p8[0][o & 1] = fma(x8.x, c[0][o].x, p8[0][o & 1]);
                        p8[0][o & 1] = fma(x8.y, c[0][o].y, p8[0][o & 1]);
                        p8[1][o & 1] = fma(x8.x, c[1][o].x, p8[1][o & 1]);
                        p8[1][o & 1] = fma(x8.y, c[1][o].y, p8[1][o & 1]);
                    }
                }
            }
            // the lane holds rows q = lr of C_J for columns 2 lq, 2 lq + 1 of each slice; they leave as D = +- scale C in the slab
            // order of CLayout (rows q >= P_J are exact zeros: the blocks carry zeros there)
            const uint32_t sg = (uint32_t)info.y >> 16;
            const double sc = ((sg >> lr) & 1u) ? -p.scale : p.scale;
            const double sc8 = ((sg >> 8) & 1u) ? -p.scale : p.scale;
            const int64_t slab_g = ((int64_t)info.w * p.ngroups16 + (w.colw >> 4)) * CLayout<P9>::SLAB;
            double v8[2] = {0.0, 0.0};
            if (P9) {
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    double v = p8[s][0] + p8[s][1];
                    v += __shfl_xor_sync(0xffffffffu, v, 1);
                    v += __shfl_xor_sync(0xffffffffu, v, 2);
                    v8[s] = sc8 * v;                                              // lanes lq == 0 .. 3 all hold column lr
                }
            }
            if (stage) {
                // staged in shared memory and added to the atom's slab with one bulk reduction (UBLKRED.ADD.F64)
                if (w.lq == 0 && w.lr == 0) tma_store_wait_read_all();           // the previous job's copy has read the slab
                __syncwarp();
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    if (w.bval) {
                        sts1(stage + (uint32_t)(CLayout<P9>::at(lr, 2 * lq, s) * 8), sc * (acc[s][0][0] + acc[s][1][0]));
                        sts1(stage + (uint32_t)(CLayout<P9>::at(lr, 2 * lq + 1, s) * 8), sc * (acc[s][0][1] + acc[s][1][1]));
                    }
                    if (P9 && lq == 0) sts1(stage + (uint32_t)(CLayout<P9>::at(8, lr, s) * 8), v8[s]);
                }
                fence_async_smem();
                __syncwarp();
                if (w.lq == 0 && w.lr == 0 && !(p.dbg & 1))
                    bulk_reduce_add_f64(p.c_out + slab_g, stage, (uint32_t)(CLayout<P9>::SLAB * 8));
            } else if (!(p.dbg & 1)) {
                double *cout = p.c_out + slab_g;
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    if (w.bval) {
                        atomicAdd(cout + CLayout<P9>::at(lr, 2 * lq, s), sc * (acc[s][0][0] + acc[s][1][0]));
                        atomicAdd(cout + CLayout<P9>::at(lr, 2 * lq + 1, s), sc * (acc[s][0][1] + acc[s][1][1]));
                    }
                    if (P9 && lq == 0) atomicAdd(cout + CLayout<P9>::at(8, lr, s), v8[s]);
                }
            }
        }
    }
}

// Warp 0 cuts the longest range of jobs r0 .. that fits the block store (at most NLB_MAXJ jobs), writes their records and
// requests their blocks (one cp.async.bulk and one mbarrier per job); returns the end of the range in round_end[0].
template <bool P9>
__device__ __forceinline__ void load_round(const BrickParams &p, int j0, int na, int r0, int lane, double *store,
                                           int4 *jobinfo, uint64_t *full, int32_t *round_end)
{
    constexpr int BLK = BlkLayout<P9>::BLK;
    const int jm = r0 + lane;
    BrickJob job = {0, 0u, 0, 0, 0};
    if (jm < na) job = p.jobs[j0 + jm];
    const int nb = __popc(job.mask & 0xffffu);
    int incl = nb;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += v;
    }
    const bool take = jm < na && incl <= p.cap_blocks;
    const int cnt = __popc(__ballot_sync(0xffffffffu, take));      // a prefix: incl is non-decreasing
    if (take) {
        jobinfo[lane] = make_int4(incl - nb, (int)job.mask, job.pj, job.atom);
        if (p.dbg & 16) mbar_arrive(&full[lane]);
        else {
            mbar_arrive_expect_tx(&full[lane], (uint32_t)(nb * BLK * 8));
            bulk_g2s(store + (incl - nb) * BLK, p.blk + job.blk0 * BLK, (uint32_t)(nb * BLK * 8), &full[lane]);
        }
    } else {
        mbar_arrive(&full[lane]);             // keeps every barrier on the round's phase
    }
    if (lane == 0) round_end[0] = r0 + cnt;
}

// ---- general kernel: one CTA per (brick, 64 columns); tile by direct global loads / stores; load rounds when a brick has
// more chi blocks than the store holds.  P9: projector class (true: up to 9 projectors = two DMMA k-steps + a rank-1 FMA
// update for projector 8; false: up to 4 = one k-step).  DO_PULL / DO_PROJ select the three variants: project only (C_0 of
// a filter call, first half of H X), pull only (last degree step, second half of H X), both.
template <bool P9, bool DO_PULL, bool DO_PROJ>
__global__ void __launch_bounds__(NLB_WARPS * 32, 2)
nl_brick_kernel(const BrickParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw);                          // [NLB_MAXJ]
    int4 *jobinfo = reinterpret_cast<int4 *>(full + NLB_MAXJ);                        // [NLB_MAXJ]
    int32_t *round_end = reinterpret_cast<int32_t *>(jobinfo + NLB_MAXJ);             // [4]
    double *store = reinterpret_cast<double *>(smem_raw + 1024);                      // [cap_blocks][BLK] (+ 1 KB read slack)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int brick = blockIdx.x / p.ncolgroups;
    const int cg = blockIdx.x - brick * p.ncolgroups;
    if (tid == 0) {
        for (int s = 0; s < NLB_MAXJ; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    const int j0 = p.job_ptr[brick];
    const int na = p.job_ptr[brick + 1] - j0;

    // ---- the warp's 64 points x 16 columns of the tile, straight into accumulator-fragment registers -------------------
    // c[s][o]: lane (lr, lq) holds, for column slice s, column colw + 8 s + lr and the x pair (py, pz) = (lq & 1, lq >> 1)
    // of cube o of its half brick.
    WarpCtx<P9> w;
    w.init(lane, warp & 1, cg * NLB_COLS + (warp >> 1) * 16, p.ncols);
    double *t0 = p.tile + (int64_t)(w.colw + w.lr) * p.ld;
    double *t1 = t0 + 8 * p.ld;
    const int x0 = p.brick_org[4 * brick], y0 = p.brick_org[4 * brick + 1], z0 = p.brick_org[4 * brick + 2];
    auto row_off = [&](int o) -> int {                        // grid index of the lane's pair of cube o, -1 outside the grid
        const int og = o + NB_HOCT * w.half;
        const int cx = og & ((1 << p.lhx) - 1), cy = (og >> p.lhx) & ((1 << p.lhy) - 1), cz = og >> (p.lhx + p.lhy);
        const int y = y0 + 2 * cy + (w.lq & 1), z = z0 + 2 * cz + (w.lq >> 1);
        return (y < p.ny && z < p.nz) ? x0 + 2 * cx + p.nx * (y + p.ny * z) : -1;
    };
    double2 c[2][NB_HOCT];
#pragma unroll
    for (int o = 0; o < NB_HOCT; ++o) {
        const int ro = row_off(o);
        c[0][o] = (w.cv0 && ro >= 0 && !(p.dbg & 8)) ? *reinterpret_cast<const double2 *>(t0 + ro) : make_double2(0.0, 0.0);
        c[1][o] = (w.cv1 && ro >= 0 && !(p.dbg & 8)) ? *reinterpret_cast<const double2 *>(t1 + ro) : make_double2(0.0, 0.0);
    }
    __syncthreads();                                          // barriers initialised

    const uint32_t store_a = smem_u32(store);
    int rounds = 0;
    bool resident = false;                                    // the store holds the brick's ONLY round
#pragma unroll 1
    for (int ph = DO_PULL ? 0 : 1; ph < (DO_PROJ ? 2 : 1); ++ph) {
        const bool pull = ph == 0;
#pragma unroll 1
        for (int r0 = 0; r0 < na;) {
            bool wait_full = false;
            if (!(resident && !pull)) {
                if (rounds > 0) __syncthreads();              // every warp is done reading the previous round
                if (warp == 0) load_round<P9>(p, j0, na, r0, lane, store, jobinfo, full, round_end);
                __syncthreads();
                wait_full = true;
                ++rounds;
            }
            const int r1 = round_end[0];
            if (pull && DO_PROJ && r0 == 0 && r1 == na) resident = true;
            const uint32_t parity = (uint32_t)((rounds - 1) & 1);
            if (pull) run_jobs<P9, true>(c, w, p, store_a, jobinfo, full, r0, r0, r1, wait_full, parity);
            else run_jobs<P9, false>(c, w, p, store_a, jobinfo, full, r0, r0, r1, wait_full, parity);
            r0 = r1;
        }
        if (pull) {                                           // all atoms pulled: the registers hold the final Out
#pragma unroll
            for (int o = 0; o < NB_HOCT; ++o) {
                const int ro = row_off(o);
                if (w.cv0 && ro >= 0 && !(p.dbg & 8)) *reinterpret_cast<double2 *>(t0 + ro) = c[0][o];
                if (w.cv1 && ro >= 0 && !(p.dbg & 8)) *reinterpret_cast<double2 *>(t1 + ro) = c[1][o];
            }
        }
    }
}

// ---- persistent kernel (the one the benchmark shapes take): one CTA per SM walks over "units" = (brick, chunk of 16-column
// groups).  The brick's chi blocks are loaded ONCE per unit and stay in shared memory while the CTA's sixteen warps stream
// the unit's column groups through them: warp w owns half (w & 1) of the brick and takes the groups w / 2, w / 2 + 8, ...
// Every warp is its own pipeline: it owns an 8 KB tile buffer (half brick x 16 columns) filled by a TMA box copy (dimensions
// x, column, y, z) and an mbarrier; the tile goes to registers, the pull runs, the result returns through the same buffer
// and one TMA box store, and the copy of the warp's NEXT item is issued one projection job later (when the store has read
// the buffer), so that it overlaps the rest of the projection.  No barrier couples the warps inside a unit.  Concurrent CTAs
// work on x-adjacent bricks and the same column groups, which keeps the 64-byte x runs of a brick row on the same DRAM pages.
constexpr int NLP_WARPS = 16;
constexpr int NLP_COLS = 16;                                  // columns per item
constexpr int NLP_GSTEP = NLP_WARPS / 2;                      // column groups in flight per half
constexpr int NLP_TILE_BYTES = (NB_PTS / 2) * NLP_COLS * 8;   // 8 KB
constexpr int NLP_SLAB_BYTES = CLayout<true>::SLAB * 8;         // one slab: 16 columns x 9 sums of one job

template <bool P9, bool DO_PULL, bool DO_PROJ>
__global__ void __launch_bounds__(NLP_WARPS * 32, 1)
nl_brick_persist_kernel(const __grid_constant__ CUtensorMap tmap, const BrickParams p, int nunits, int nchunks, int chunk_len)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw);                          // [NLB_MAXJ] chi blocks of job j landed
    uint64_t *tile_full = full + NLB_MAXJ;                                            // [NLP_WARPS] tile of the warp landed
    int4 *jobinfo = reinterpret_cast<int4 *>(tile_full + NLP_WARPS);                  // [NLB_MAXJ]
    int32_t *round_end = reinterpret_cast<int32_t *>(jobinfo + NLB_MAXJ);             // [4]
    unsigned char *tiles = smem_raw + 1024;                                           // [NLP_WARPS][NLP_TILE_BYTES]
    unsigned char *slabs = tiles + NLP_WARPS * NLP_TILE_BYTES;                       // [NLP_WARPS][NLP_SLAB_BYTES] projection results
    double *store = reinterpret_cast<double *>(slabs + NLP_WARPS * NLP_SLAB_BYTES);   // [cap_blocks][BLK] (+ 1 KB read slack)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < NLB_MAXJ; ++s) mbar_init(&full[s], 1);
        for (int s = 0; s < NLP_WARPS; ++s) mbar_init(&tile_full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();

    WarpCtx<P9> w;
    w.init(lane, warp & 1, 0, p.ncols);
    const int gsel = warp >> 1;
    const uint32_t tbuf = smem_u32(tiles + warp * NLP_TILE_BYTES);
    uint64_t *tbar = &tile_full[warp];
    const uint32_t store_a = smem_u32(store);
    const uint32_t slab = smem_u32(slabs + warp * NLP_SLAB_BYTES);
    const int bzh = (NB_PTS / (p.bx * p.by)) / 2;             // z planes of a half brick
    // byte address of the lane's pair of cube o inside the staged half tile [z][y][column][x]: tlane + p.toct[cube]
    const uint32_t tlane = tbuf + (uint32_t)(((((w.lq >> 1) * p.by + (w.lq & 1)) * NLP_COLS + w.lr) * p.bx) * 8);
    const int32_t *toct = p.toct + NB_HOCT * w.half;
    const uint32_t tslice = (uint32_t)(8 * p.bx * 8);         // eight columns further
    auto unit_range = [&](int unit, int *brick, int *g0, int *g1) {
        *brick = unit / nchunks;
        *g0 = (unit - *brick * nchunks) * chunk_len;
        *g1 = min(*g0 + chunk_len, p.ncolgroups);
    };
    auto issue_tile = [&](int brick, int g) {
        mbar_arrive_expect_tx(tbar, (uint32_t)NLP_TILE_BYTES);
        tma_load_4d(tbuf, &tmap, tbar, p.brick_org[4 * brick], g * NLP_COLS, p.brick_org[4 * brick + 1],
                    p.brick_org[4 * brick + 2] + w.half * bzh);
    };
    // the warp's first item: the first unit of this CTA that has a column group for it
    if (lane == 0 && !(p.dbg & (8 | 128))) {
        for (int u = blockIdx.x; u < nunits; u += gridDim.x) {
            int b, g0, g1;
            unit_range(u, &b, &g0, &g1);
            if (g0 + gsel < g1) { issue_tile(b, g0 + gsel); break; }
        }
    }
    uint32_t tpar = 0;                                        // phase of the warp's tile barrier
    int units_done = 0;
#pragma unroll 1
    for (int unit = blockIdx.x; unit < nunits; unit += gridDim.x, ++units_done) {
        int brick, g0, g1;
        unit_range(unit, &brick, &g0, &g1);
        const int j0 = p.job_ptr[brick];
        const int na = p.job_ptr[brick + 1] - j0;
        if (units_done > 0) __syncthreads();                  // every warp is done with the previous unit's chi blocks
        if (warp == 0) load_round<P9>(p, j0, na, 0, lane, store, jobinfo, full, round_end);   // single round by construction
        __syncthreads();
        const uint32_t cpar = (uint32_t)(units_done & 1);
        const int x0 = p.brick_org[4 * brick], y0 = p.brick_org[4 * brick + 1], z0 = p.brick_org[4 * brick + 2] + w.half * bzh;
        bool first = true;
#pragma unroll 1
        for (int g = g0 + gsel; g < g1; g += NLP_GSTEP) {
            w.set_cols(g * NLP_COLS, p.ncols);
            double2 c[2][NB_HOCT];
            if (!(p.dbg & (8 | 128))) { mbar_wait(tbar, tpar); tpar ^= 1u; }
#pragma unroll
            for (int o = 0; o < NB_HOCT; ++o) {
                c[0][o] = lds2(tlane + toct[o]);
                c[1][o] = lds2(tlane + toct[o] + tslice);
            }
            auto next_tile = [&]() {                           // lane 0: request the warp's next item (the buffer is free)
                if (g + NLP_GSTEP < g1) issue_tile(brick, g + NLP_GSTEP);
                else {
                    for (int u = unit + gridDim.x; u < nunits; u += gridDim.x) {
                        int b, h0, h1;
                        unit_range(u, &b, &h0, &h1);
                        if (h0 + gsel < h1) { issue_tile(b, h0 + gsel); break; }
                    }
                }
            };
            if (DO_PULL) {
                run_jobs<P9, true>(c, w, p, store_a, jobinfo, full, 0, 0, na, first, cpar);
                // all atoms pulled: the registers hold the final Out; it leaves through the warp's tile buffer and one TMA
                // box store
#pragma unroll
                for (int o = 0; o < NB_HOCT; ++o) {
                    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(tlane + toct[o]), "d"(c[0][o].x), "d"(c[0][o].y) : "memory");
                    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(tlane + toct[o] + tslice), "d"(c[1][o].x), "d"(c[1][o].y) : "memory");
                }
                fence_async_smem();                                                // generic writes -> async proxy
                __syncwarp();
                if (lane == 0 && !(p.dbg & (8 | 64))) tma_store_4d(&tmap, tbuf, x0, g * NLP_COLS, y0, z0);
                if (DO_PROJ) {
                    // the next tile is requested one projection job later: by then the store has read the buffer
                    run_jobs<P9, false>(c, w, p, store_a, jobinfo, full, 0, 0, min(1, na), false, cpar, slab);
                    if (lane == 0 && !(p.dbg & (8 | 128))) { tma_store_wait_read_all(); next_tile(); }
                    run_jobs<P9, false>(c, w, p, store_a, jobinfo, full, 0, min(1, na), na, false, cpar, slab);
                } else if (lane == 0 && !(p.dbg & (8 | 128))) {
                    tma_store_wait_read_all();
                    next_tile();
                }
            } else {
                __syncwarp();                                  // the whole warp holds the tile in registers
                if (lane == 0 && !(p.dbg & (8 | 128))) next_tile();
                run_jobs<P9, false>(c, w, p, store_a, jobinfo, full, 0, 0, na, first, cpar, slab);
            }
            first = false;
        }
    }
    if (lane == 0) tma_store_wait_all();                      // the warp's last stores / reductions have left shared memory
}

template <typename T>
int upload_vec(T **dst, const std::vector<T> &v)
{
    *dst = nullptr;
    if (v.empty()) return SPARC_GPU_SUCCESS;
    SPARC_CUDA_TRY(cudaMalloc((void **)dst, v.size() * sizeof(T)));
    SPARC_CUDA_TRY(cudaMemcpy(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice));
    return SPARC_GPU_SUCCESS;
}

int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }

}  // namespace

// Build the brick tables from the descriptor (host pointers, already validated).  Leaves ctx->nlb.ok = 0 when the
// grid does not meet the preconditions (even nx with a brick width dividing it); the per-atom kernels then serve.
int nlb_build(sparc_gpu_ctx *ctx, const sparc_gpu_desc *d)
{
    NlBrick &B = ctx->nlb;
    B.ok = 0;
    const int nx = ctx->n[0], ny = ctx->n[1], nz = ctx->n[2];
    if (ctx->n_atoms == 0 || ctx->n_proj_total == 0 || ctx->supp_total == 0) return SPARC_GPU_SUCCESS;
    if (ctx->max_proj > 9) return SPARC_GPU_SUCCESS;      // l <= 2 (s+p+d); larger sets use the per-atom kernels
    if (nx % 8 == 0) { B.bx = 8; B.by = 4; B.bz = 4; }
    else if (nx % 4 == 0) { B.bx = 4; B.by = 8; B.bz = 4; }
    else if (nx % 2 == 0) { B.bx = 2; B.by = 8; B.bz = 8; }
    else return SPARC_GPU_SUCCESS;
    B.pclass = ctx->max_proj <= 4 ? 4 : 9;
    const bool p9 = B.pclass == 9;
    const int blk_sz = p9 ? BlkLayout<true>::BLK : BlkLayout<false>::BLK;
    const int nbx = nx / B.bx, nby = (ny + B.by - 1) / B.by, nbz = (nz + B.bz - 1) / B.bz;
    const int64_t nbricks = (int64_t)nbx * nby * nbz;
    if (nbricks >= (int64_t)INT32_MAX) return SPARC_GPU_SUCCESS;
    const int hx = B.bx / 2, hy = B.by / 2;               // cubes per brick along x and y

    struct Pair { int32_t brick, atom; uint32_t mask; };
    std::vector<Pair> pairs;
    // grid index -> brick, octet (2 x 2 x 2 cube, x fastest over the cubes) and point inside the octet (x fastest)
    auto locate = [&](int32_t i, int32_t *brick, int *oct, int *pt) {
        const int x = i % nx, y = (i / nx) % ny, z = i / (nx * ny);
        const int bx = x / B.bx, by = y / B.by, bz = z / B.bz;
        *brick = bx + nbx * (by + nby * bz);
        const int lx = x - bx * B.bx, ly = y - by * B.by, lz = z - bz * B.bz;
        *oct = (lx >> 1) + hx * ((ly >> 1) + hy * (lz >> 1));
        *pt = (lx & 1) + 2 * (ly & 1) + 4 * (lz & 1);
    };
    // pass 1: octet masks per (brick, atom)
    for (int J = 0; J < ctx->n_atoms; ++J) {
        if (d->n_proj[J] <= 0) continue;
        std::unordered_map<int32_t, uint32_t> m;
        for (int64_t t = d->supp_ptr[J]; t < d->supp_ptr[J + 1]; ++t) {
            int32_t brick; int o, r;
            locate(d->supp_idx[t], &brick, &o, &r);
            m[brick] |= 1u << o;
        }
        for (auto &kv : m) pairs.push_back({kv.first, J, kv.second});
    }
    if (pairs.empty()) return SPARC_GPU_SUCCESS;
    std::sort(pairs.begin(), pairs.end(), [](const Pair &a, const Pair &b) {
        return a.brick != b.brick ? a.brick < b.brick : a.atom < b.atom;
    });
    std::vector<int32_t> pofs((size_t)ctx->n_atoms + 1, 0);
    for (int J = 0; J < ctx->n_atoms; ++J) pofs[(size_t)J + 1] = pofs[(size_t)J] + d->n_proj[J];
    std::vector<int32_t> org, job_ptr;
    std::vector<BrickJob> jobs(pairs.size());
    int64_t nblocks = 0, in_brick = 0, jobs_in_brick = 0;
    B.max_blocks = 0; B.max_jobs = 0;
    for (size_t k = 0; k < pairs.size(); ++k) {
        if (k == 0 || pairs[k].brick != pairs[k - 1].brick) {
            const int32_t b = pairs[k].brick;
            const int bx = b % nbx, by = (b / nbx) % nby, bz = b / (nbx * nby);
            org.push_back(bx * B.bx); org.push_back(by * B.by); org.push_back(bz * B.bz); org.push_back(0);
            job_ptr.push_back((int32_t)k);
            in_brick = 0; jobs_in_brick = 0;
        }
        org[org.size() - 1] |= (int32_t)pairs[k].mask;
        const int J = pairs[k].atom;
        uint32_t signs = 0;                                // gamma_q < 0: the pull negates its A operand (blocks carry sqrt|gamma|)
        for (int q = 0; q < d->n_proj[J]; ++q)
            if (d->gamma[pofs[(size_t)J] + q] < 0.0) signs |= 1u << q;
        jobs[k] = {J, pairs[k].mask | (signs << 16), nblocks, pofs[(size_t)J], d->n_proj[J]};
        const int nb = __builtin_popcount(pairs[k].mask);
        nblocks += nb;
        in_brick += nb;
        B.max_blocks = std::max<int64_t>(B.max_blocks, in_brick);
        B.max_jobs = std::max<int64_t>(B.max_jobs, ++jobs_in_brick);
    }
    job_ptr.push_back((int32_t)pairs.size());
    B.n_active = (int32_t)(job_ptr.size() - 1);
    B.n_blocks = nblocks;

    // pass 2: chi sqrt|gamma| blocks in the shared fragment layout
    std::vector<double> blk((size_t)nblocks * blk_sz, 0.0);
    std::vector<std::unordered_map<int32_t, int64_t>> jobof((size_t)ctx->n_atoms);     // per atom: brick -> job index
    for (size_t k = 0; k < pairs.size(); ++k) jobof[(size_t)pairs[k].atom][pairs[k].brick] = (int64_t)k;
    for (int J = 0; J < ctx->n_atoms; ++J) {
        const int P = d->n_proj[J];
        if (P <= 0) continue;
        const int64_t s0 = d->supp_ptr[J], nJ = d->supp_ptr[J + 1] - s0;
        const double *chi = d->chi + d->chi_ptr[J];
        double sg[SPARC_MAX_PROJ];
        for (int q = 0; q < P; ++q) sg[q] = sqrt(fabs(d->gamma[pofs[(size_t)J] + q]));
        for (int64_t t = 0; t < nJ; ++t) {
            int32_t brick; int o, r;
            locate(d->supp_idx[s0 + t], &brick, &o, &r);
            const BrickJob &job = jobs[(size_t)jobof[(size_t)J][brick]];
            const int64_t b = job.blk0 + __builtin_popcount(job.mask & 0xffffu & ((1u << o) - 1u));
            double *bp = blk.data() + b * blk_sz;
            for (int q = 0; q < P; ++q)
                bp[p9 ? BlkLayout<true>::at(r, q) : BlkLayout<false>::at(r, q)] = chi[t + (int64_t)q * nJ] * sg[q];
        }
    }
    int st;
    if ((st = upload_vec(&B.d_org, org))) return st;
    if ((st = upload_vec(&B.d_job_ptr, job_ptr))) return st;
    {
        B.d_jobs = nullptr;
        SPARC_CUDA_TRY(cudaMalloc(&B.d_jobs, jobs.size() * sizeof(BrickJob)));
        SPARC_CUDA_TRY(cudaMemcpy(B.d_jobs, jobs.data(), jobs.size() * sizeof(BrickJob), cudaMemcpyHostToDevice));
    }
    if ((st = upload_vec(&B.d_blk, blk))) return st;
    B.ok = 1;
    return SPARC_GPU_SUCCESS;
}

void nlb_free(sparc_gpu_ctx *ctx)
{
    NlBrick &B = ctx->nlb;
    cudaFree(B.d_org); cudaFree(B.d_job_ptr); cudaFree(B.d_jobs); cudaFree(B.d_blk);
    B = NlBrick();
}

bool nlb_supported(const sparc_gpu_ctx *ctx, const double *X, int64_t ld)
{
    return ctx->nlb.ok && (((uintptr_t)X & 15) == 0) && (ld % 2 == 0);
}

namespace {

constexpr int NLB_SMEM_MAX = 110 * 1024;       // general kernel: two CTAs per SM
constexpr int NLP_SMEM_MAX = 227 * 1024;       // persistent kernel: one CTA per SM

// (x, column, y, z) tensor map over the N_d x ncols block with a bx x 16 x by x bz/2 box: half a brick x 16 columns; the
// box lands as [z][y][column][x]
bool encode_tile_map(const sparc_gpu_ctx *ctx, CUtensorMap *tm, const double *base, int64_t ld, int64_t ncols)
{
    const NlBrick &B = ctx->nlb;
    const int nx = ctx->n[0], ny = ctx->n[1], nz = ctx->n[2];
    const cuuint64_t gdim[4] = {(cuuint64_t)nx, (cuuint64_t)ncols, (cuuint64_t)ny, (cuuint64_t)nz};
    const cuuint64_t gstr[3] = {(cuuint64_t)ld * 8, (cuuint64_t)nx * 8, (cuuint64_t)nx * ny * 8};
    const cuuint32_t box[4] = {(cuuint32_t)B.bx, (cuuint32_t)NLP_COLS, (cuuint32_t)B.by, (cuuint32_t)(B.bz / 2)};
    return encode_f64_map(ctx->fn_encode_tiled, tm, base, 4, gdim, gstr, box);
}

template <bool P9>
int launch_general(sparc_gpu_ctx *ctx, int mode, BrickParams &P, cudaStream_t st)
{
    constexpr int BLK = BlkLayout<P9>::BLK;
    const int64_t ngroups = (P.ncols + NLB_COLS - 1) / NLB_COLS;
    if ((int64_t)ctx->nlb.n_active * ngroups >= (int64_t)INT32_MAX) return SPARC_GPU_UNSUPPORTED;
    P.ncolgroups = (int32_t)ngroups;
    // shared memory: 1 KB of barriers and job records, the block store, 1 KB of read slack.  The store holds the largest
    // brick of this context when that fits two CTAs per SM (every brick then loads its chi blocks once); otherwise the
    // kernel works in rounds.
    const int64_t want = std::max<int64_t>(ctx->nlb.max_blocks, NB_OCT);
    int cap = (int)std::min<int64_t>(want, (NLB_SMEM_MAX - 2048) / (BLK * 8));
    if (ctx->opt_nlb_cap > 0) cap = std::max(NB_OCT, std::min(cap, ctx->opt_nlb_cap));       // test knob: forces rounds
    const size_t smem = 2048 + (size_t)cap * BLK * 8;
    P.cap_blocks = cap;
    void (*kern)(const BrickParams) = mode == 1 ? nl_brick_kernel<P9, false, true>
                                      : mode == 2 ? nl_brick_kernel<P9, true, false>
                                                  : nl_brick_kernel<P9, true, true>;
    // once per context and kernel variant (the attribute is per device and function)
    const int bit = (P9 ? 4 : 0) + mode;
    if (!(ctx->func_attr_done & (1ull << bit))) {
        SPARC_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, NLB_SMEM_MAX));
        ctx->func_attr_done |= 1ull << bit;
    }
    const unsigned grid = (unsigned)((int64_t)ctx->nlb.n_active * ngroups);
    prof_begin(ctx, KK_NL_BRICK, st);
    kern<<<grid, NLB_WARPS * 32, smem, st>>>(P);
    prof_end(ctx, KK_NL_BRICK, st);
    SPARC_CUDA_TRY(cudaGetLastError());
    return SPARC_GPU_SUCCESS;
}

// chi blocks the persistent kernel's store holds next to its four tile buffers
template <bool P9> constexpr int persist_cap() { return (NLP_SMEM_MAX - 2048 - NLP_WARPS * (NLP_TILE_BYTES + NLP_SLAB_BYTES)) / (BlkLayout<P9>::BLK * 8); }

template <bool P9>
int launch_persist(sparc_gpu_ctx *ctx, int mode, BrickParams &P, const CUtensorMap &tmap, cudaStream_t st)
{
    constexpr int BLK = BlkLayout<P9>::BLK;
    const NlBrick &B = ctx->nlb;
    const int ngroups = (int)((P.ncols + NLP_COLS - 1) / NLP_COLS);
    P.ncolgroups = ngroups;
    const int cap = (int)std::max<int64_t>(B.max_blocks, NB_OCT);
    P.cap_blocks = cap;
    const size_t smem = 2048 + (size_t)NLP_WARPS * (NLP_TILE_BYTES + NLP_SLAB_BYTES) + (size_t)cap * BLK * 8;
    // units = (brick, chunk of column groups): whole bricks when there are enough of them to balance the SMs (three units per
    // SM: measured at config 1, 80 us with 582 whole-brick units against 87 us with 1164 half units -- a longer unit amortises
    // its chi-block load and keeps the warps' tile prefetch running), else chunks of at least one group per warp
    int chunk_len = ngroups;
    while ((int64_t)B.n_active * ((ngroups + chunk_len - 1) / chunk_len) < 3LL * ctx->sm_count && chunk_len > NLP_GSTEP)
        chunk_len = std::max(NLP_GSTEP, (chunk_len / 2 + NLP_GSTEP - 1) / NLP_GSTEP * NLP_GSTEP);
    const int nchunks = (ngroups + chunk_len - 1) / chunk_len;
    const int64_t nunits = (int64_t)B.n_active * nchunks;
    if (nunits >= (int64_t)INT32_MAX) return SPARC_GPU_UNSUPPORTED;
    void (*kern)(const CUtensorMap, const BrickParams, int, int, int) =
        mode == 1 ? nl_brick_persist_kernel<P9, false, true>
        : mode == 2 ? nl_brick_persist_kernel<P9, true, false> : nl_brick_persist_kernel<P9, true, true>;
    const int bit = 8 + (P9 ? 4 : 0) + mode;
    if (!(ctx->func_attr_done & (1ull << bit))) {
        SPARC_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, NLP_SMEM_MAX));
        ctx->func_attr_done |= 1ull << bit;
    }
    const unsigned grid = (unsigned)std::min<int64_t>(nunits, ctx->sm_count);
    prof_begin(ctx, KK_NL_BRICK, st);
    kern<<<grid, NLP_WARPS * 32, smem, st>>>(tmap, P, (int)nunits, nchunks, chunk_len);
    prof_end(ctx, KK_NL_BRICK, st);
    SPARC_CUDA_TRY(cudaGetLastError());
    return SPARC_GPU_SUCCESS;
}

}  // namespace

int launch_nl_brick(sparc_gpu_ctx *ctx, int mode, double *XorOut, int64_t ld, int64_t ncols, double scale,
                    const double *c_in, double *c_out, cudaStream_t st)
{
    const NlBrick &B = ctx->nlb;
    if (!nlb_supported(ctx, XorOut, ld) || mode < 1 || mode > 3) return SPARC_GPU_UNSUPPORTED;
    if (ncols <= 0 || B.n_active == 0) return SPARC_GPU_SUCCESS;
    BrickParams P;
    P.brick_org = B.d_org; P.job_ptr = B.d_job_ptr; P.jobs = (const BrickJob *)B.d_jobs;
    P.blk = B.d_blk;
    P.tile = XorOut; P.ld = ld;
    P.c_in = c_in; P.c_out = c_out;
    P.ncp = nlb_c_cols(ncols);
    P.ngroups16 = (int32_t)(P.ncp / 16);
    P.ncols = (int32_t)ncols;
    P.nx = ctx->n[0]; P.ny = ctx->n[1]; P.nz = ctx->n[2];
    P.bx = B.bx; P.by = B.by;
    P.lhx = ilog2(B.bx / 2); P.lhy = ilog2(B.by / 2);
    P.scale = scale;
    P.dbg = ctx->opt_nlb_dbg;
    for (int og = 0; og < NB_OCT; ++og) {       // staged half tile [z][y][16 columns][x], z relative to the half's first plane
        const int hx = B.bx / 2, hy = B.by / 2, bzh = B.bz / 2;
        const int cx = og % hx, cy = (og / hx) % hy, cz = og / (hx * hy);
        const int zrel = 2 * cz - (og / NB_HOCT) * bzh;
        P.toct[og] = ((zrel * B.by + 2 * cy) * 16 * B.bx + 2 * cx) * 8;
    }
    // the persistent kernel needs every brick's chi blocks to fit its store in one round and the TMA entry point; option
    // "nlb_kernel": 0 auto, 1 general kernel, 2 persistent kernel or UNSUPPORTED
    const bool p9 = B.pclass == 9;
    const bool fits = ctx->fn_encode_tiled && B.max_jobs <= NLB_MAXJ &&
                      B.max_blocks <= (p9 ? persist_cap<true>() : persist_cap<false>()) && ctx->opt_nlb_cap == 0;
    if (ctx->opt_nlb_kernel == 2 && !fits) return SPARC_GPU_UNSUPPORTED;
    if (fits && ctx->opt_nlb_kernel != 1) {
        CUtensorMap tmap;
        if (!encode_tile_map(ctx, &tmap, XorOut, ld, ncols)) return SPARC_GPU_CUDA_ERROR;
        return p9 ? launch_persist<true>(ctx, mode, P, tmap, st) : launch_persist<false>(ctx, mode, P, tmap, st);
    }
    return p9 ? launch_general<true>(ctx, mode, P, st) : launch_general<false>(ctx, mode, P, st);
}
