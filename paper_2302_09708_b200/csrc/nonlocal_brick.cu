// nonlocal_brick.cu -- brick-tiled Kleinman-Bylander nonlocal term on the FP64 tensor pipe (default nonlocal path).
//
//   V_nl X = sum_J S_J^T chi_J diag(gamma_J) chi_J^T S_J X
//
// The per-atom formulation gathers X at each atom's support and scatter-adds with atomics: 8c + 16c bytes and one
// atomic per (support row, column) (c = coverage, 4-5 at configs 3-4).  Here the grid is cut into bricks of 128
// points (BX x BY x BZ, x fastest) and one CTA owns (brick, 64 columns): it reads the 128 x 64 tile of Out once into
// tensor-core accumulator fragments, adds the contribution of EVERY atom whose support meets the brick
// ("pull": Out^T[col, pt] += D_J^T[col, q] chi_J^T[q, pt], DMMA m8n8k4), writes the tile back once, and -- the tile
// now being the final Psi_{k+1} -- contracts it with the same chi blocks for the NEXT degree step
// ("project": C_J[q, col] += chi_J^T[q, pt] Out[pt, col]), so that the nonlocal term costs one 16 B read-modify-write
// of Out per degree step and one atomic per (brick, atom, projector, column).  The accumulator fragment of the pull
// is, register for register, the B operand of the projection (k index = point pair), so no layout change is needed.
//
// Tables built at create (host): for every (brick, atom) pair a 16-bit mask of the brick's 8-point octets the atom
// touches, and per touched octet a dense block of chi values already permuted into DMMA fragment order (zeros where
// the atom does not cover a point; gamma folded into the pull blocks).  Blocks of one (brick, atom) pair are
// contiguous; a producer warp streams them (and the 64-column slice of C_J) into a shared-memory byte ring with
// cp.async.bulk, up to 16 (brick, atom) jobs ahead of the eight consumer warps; two CTAs share an SM (full / empty mbarriers).
//
// The 9th projector of an s+p+d atom is applied as a rank-1 FMA update beside the two k-steps of DMMA (a third
// k-step would be 3/4 padding).
#include <cuda.h>

#include <string.h>

#include <algorithm>
#include <unordered_map>
#include <vector>

#include "internal.h"

namespace {

constexpr int NB_PTS = 128;        // points per brick
constexpr int NB_HOCT = 16;        // octets per brick (bit mask width): one consumer warp holds all of them
constexpr int NLB_WARPS = 8;       // consumer warps: 8 column slices of 8 columns
constexpr int NLB_COLS = 64;       // columns per CTA: 8 per warp

struct BrickJob {                  // one (brick, atom) pair
    int32_t atom;
    uint32_t mask;                 // octets of the brick this atom touches
    int64_t blk0;                  // index of its first chi block
    int32_t po;                    // offset of the atom's first projector (prefix sum of P_J)
    int32_t pj;                    // P_J
};

struct BrickParams {
    const int32_t *brick_org;      // [n_active][3] origin (x0, y0, z0)
    const int32_t *job_ptr;        // [n_active + 1]
    const BrickJob *jobs;
    const double *blk_pull;        // [n_blocks][PULL_SZ]
    const double *blk_proj;        // [n_blocks][PROJ_SZ]
    const double *src;             // X (project-only) or Out (pull): N_d x ncols, ld
    double *dst;                   // Out (pull variants)
    int64_t ld;
    // C buffers hold the raw sums chi_J^T Psi atom-major: element (J, q, col) at po_J * ncp + col * P_J + q
    const double *c_in;            // chi^T Psi_k of the previous pass (pull)
    double *c_out;                 // accumulated chi^T Psi_{k+1} (project), zeroed by the caller
    int64_t ncp;                   // padded column count of the C buffers (multiple of 64)
    int32_t ncols;
    int32_t ncolgroups;
    int32_t nx, ny, nz;
    int32_t bx, by, bz;
    double scale;
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
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
        "NLB_WAIT:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra NLB_DONE;\n\t"
        "bra NLB_WAIT;\n\t"
        "NLB_DONE:\n\t"
        "}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}


__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void tma_load_tile(void *dst, const CUtensorMap *tmap, uint64_t *bar, int x, int c, int y, int z)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(
            smem_u32(dst)),
        "l"(tmap), "r"(x), "r"(c), "r"(y), "r"(z), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void tma_store_tile(const CUtensorMap *tmap, const void *src, int x, int c, int y, int z)
{
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%1, %2, %3, %4}], [%5];" ::"l"(tmap), "r"(x),
                 "r"(c), "r"(y), "r"(z), "r"(smem_u32(src))
                 : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}

constexpr int NLB_SLOTS = 16;                 // jobs in flight (mbarrier pairs)
constexpr int NLB_TILE_BYTES = NB_PTS * NLB_COLS * 8;   // the 128 x 64 tile staged by TMA: [x-run][column][points of the run]
constexpr int NLB_RING_TMA = 40 * 1024;       // ring size next to the staged tile (two CTAs per SM)
constexpr int NLB_RING_BYTES = 72 * 1024;     // byte ring the producer warp streams chi blocks (+ C slices) through

// KP: DMMA k-steps of the pull (projectors 0 .. 4 KP - 1); MT: 8-projector m-tiles of the projection; R1: projector
// number 8 applied as a rank-1 FMA update (s+p+d atoms: P = 9).  DO_PULL / DO_PROJ select the three variants:
// project only (C_0 of a filter call, first half of H X), pull only (last degree step, second half of H X), both.
// Warps 0-7 are consumers (8 columns each, the whole 128-point brick), warp 8 is the producer (two CTAs share an SM, so one
// CTA's tile load / store overlaps the other's DMMAs): it walks the brick's job list ahead of the
// consumers and streams, per (brick, atom) job, the chi blocks (and for a pull job the 64-column slice of C_J) into a
// byte ring with cp.async.bulk; full/empty mbarriers per slot.
// TMA_IO: the tile is loaded (and, after the pull, stored) by one TMA box copy through shared memory instead of 16
// predicated 16-byte global accesses per lane: the tensor map orders the dimensions (x, column, y, z), so the box lands
// as [x-run][column][points of the run] -- a warp's fragment read is then 512 contiguous bytes.
template <int KP, int MT, bool R1, bool DO_PULL, bool DO_PROJ, bool TMA_IO>
__global__ void __launch_bounds__((NLB_WARPS + 1) * 32, 2)
nl_brick_kernel(const __grid_constant__ CUtensorMap tmap, const BrickParams p)
{
    constexpr int PULL_SZ = KP * 32 + (R1 ? 8 : 0);
    constexpr int PROJ_SZ = MT * 64 + (R1 ? 8 : 0);
    constexpr int RING_BYTES = TMA_IO ? NLB_RING_TMA : NLB_RING_BYTES;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    unsigned char *tile = smem_raw;                                                   // [NLB_TILE_BYTES] (TMA_IO only)
    unsigned char *ring = smem_raw + (TMA_IO ? NLB_TILE_BYTES : 0);                   // [RING_BYTES]
    int32_t *pt_off = reinterpret_cast<int32_t *>(ring + RING_BYTES);                 // [NB_PTS] grid index, -1 outside
    uint64_t *full = reinterpret_cast<uint64_t *>(pt_off + NB_PTS);                   // [NLB_SLOTS]
    uint64_t *empty = full + NLB_SLOTS;                                               // [NLB_SLOTS]
    int4 *slot_info = reinterpret_cast<int4 *>(empty + NLB_SLOTS);                    // [NLB_SLOTS] offset, mask, P_J, po
    int32_t *slot_size = reinterpret_cast<int32_t *>(slot_info + NLB_SLOTS);          // [NLB_SLOTS] ring bytes (producer only)
    uint64_t *tile_bar = reinterpret_cast<uint64_t *>(slot_size + NLB_SLOTS);         // tile landed (TMA_IO only)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int lq = lane & 3, lr = lane >> 2;
    const int brick = blockIdx.x / p.ncolgroups;
    const int cg = blockIdx.x - brick * p.ncolgroups;
    const int x0 = p.brick_org[4 * brick], y0 = p.brick_org[4 * brick + 1], z0 = p.brick_org[4 * brick + 2];
    const uint32_t umask = (uint32_t)p.brick_org[4 * brick + 3];
    if (!TMA_IO && tid < NB_PTS) {
        const int lx = tid % p.bx, ly = (tid / p.bx) % p.by, lz = tid / (p.bx * p.by);
        const int x = x0 + lx, y = y0 + ly, z = z0 + lz;
        pt_off[tid] = (y < p.ny && z < p.nz) ? x + p.nx * (y + p.ny * z) : -1;
    }
    if (tid == 0) {
        for (int s = 0; s < NLB_SLOTS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NLB_WARPS); }
        if (TMA_IO) mbar_init(tile_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int j0 = p.job_ptr[brick];
    const int na = p.job_ptr[brick + 1] - j0;
    const int njobs = (DO_PULL ? na : 0) + (DO_PROJ ? na : 0);

    if (warp == NLB_WARPS) {
        // ================================ producer warp ==========================================================
        // lanes fetch 32 job descriptors at a time; lane 0 allocates ring space in order and issues the copies
        if (TMA_IO && lane == 0) {
            mbar_expect_tx(tile_bar, (uint32_t)NLB_TILE_BYTES);
            tma_load_tile(tile, &tmap, tile_bar, x0, cg * NLB_COLS, y0, z0);
        }
        int head = 0, used = 0, freed = 0;
        for (int jb = 0; jb < njobs; jb += 32) {
            const int jmine = jb + lane;
            BrickJob job = {0, 0u, 0, 0, 0};
            if (jmine < njobs) job = p.jobs[j0 + (jmine < na ? jmine : jmine - na)];
            const int cnt = min(32, njobs - jb);
            for (int i = 0; i < cnt; ++i) {
                const int jj = jb + i;
                const uint32_t mask = __shfl_sync(0xffffffffu, job.mask, i);
                const int pj = __shfl_sync(0xffffffffu, job.pj, i);
                const int po = __shfl_sync(0xffffffffu, job.po, i);
                const long long blk0 = __shfl_sync(0xffffffffu, (long long)job.blk0, i);
                if (lane != 0) continue;
                const bool pull = DO_PULL && jj < na;
                const uint32_t blk_bytes = (uint32_t)__popc(mask) * (uint32_t)(pull ? PULL_SZ : PROJ_SZ) * 8u;
                const uint32_t c_bytes = pull ? (uint32_t)(NLB_COLS * pj * 8) : 0u;
                int need = (int)((blk_bytes + c_bytes + 127u) & ~127u);
                const bool wrap = head + need > RING_BYTES;                       // no job straddles the ring end
                const int skip = wrap ? RING_BYTES - head : 0;
                while (jj - freed >= NLB_SLOTS || used + need + skip > RING_BYTES) {
                    const int fs = freed % NLB_SLOTS;
                    mbar_wait(&empty[fs], (uint32_t)((freed / NLB_SLOTS) & 1));
                    used -= slot_size[fs];
                    ++freed;
                }
                if (wrap) head = 0;
                const int slot = jj % NLB_SLOTS;
                slot_size[slot] = need + skip;
                used += need + skip;
                slot_info[slot] = make_int4(head, (int)mask, pj, po);
                mbar_expect_tx(&full[slot], blk_bytes + c_bytes);
                const double *src = pull ? p.blk_pull + blk0 * PULL_SZ : p.blk_proj + blk0 * PROJ_SZ;
                bulk_g2s(ring + head, src, blk_bytes, &full[slot]);
                if (pull)
                    bulk_g2s(ring + head + blk_bytes, p.c_in + (int64_t)po * p.ncp + (int64_t)cg * NLB_COLS * pj, c_bytes,
                             &full[slot]);
                head += need;
            }
        }
        return;
    }

    // ==================================== consumer warps ============================================================
    // the 128 x 8 tile of this warp, in accumulator-fragment order: lane (lr, lq)
    // holds column colw + lr, points 2 lq and 2 lq + 1 of every octet
    const int colw = cg * NLB_COLS + (warp & 7) * 8;
    const int col = colw + lr;
    const bool colv = col < p.ncols;
    const uint32_t umask_h = umask & 0xffffu;
    const int32_t *pt_h = pt_off + 2 * lq;
    const double *srcc = p.src + (int64_t)(colv ? col : 0) * p.ld;
    double2 c[NB_HOCT];
    // byte offset of this lane's pair of octet 0 inside the staged tile: [x-run][column][points of the run]
    const int colL = (warp & 7) * 8 + lr;
    // (an octet is 8 consecutive brick-local points = 8 / bx x-runs: octets are 8 x 64 x 8 = 4096 bytes apart)
    const uint32_t toff0 = (uint32_t)(((((2 * lq) / p.bx) * NLB_COLS + colL) * p.bx + ((2 * lq) % p.bx)) * 8);
    if (TMA_IO) {
        mbar_wait(tile_bar, 0u);
#pragma unroll
        for (int o = 0; o < NB_HOCT; ++o) c[o] = *reinterpret_cast<const double2 *>(tile + toff0 + 4096 * o);
    } else {
        // all offsets first, then branch-free loads: an untouched octet reads the column's first pair (a cached dummy)
        int off[NB_HOCT];
#pragma unroll
        for (int o = 0; o < NB_HOCT; ++o) off[o] = pt_h[8 * o];
#pragma unroll
        for (int o = 0; o < NB_HOCT; ++o) {
            const bool ok = ((umask_h >> o) & 1u) && off[o] >= 0 && colv;
            const double2 v = *reinterpret_cast<const double2 *>(srcc + (ok ? off[o] : 0));
            c[o] = ok ? v : make_double2(0.0, 0.0);
        }
    }

    for (int jj = 0; jj < njobs; ++jj) {
        const int slot = jj % NLB_SLOTS;
        const bool pull = DO_PULL && jj < na;
        mbar_wait(&full[slot], (uint32_t)((jj / NLB_SLOTS) & 1));
        const int4 info = slot_info[slot];                 // ring offset, octet mask, P_J, projector offset
        const uint32_t mask_all = (uint32_t)info.y;
        const uint32_t mask = mask_all & 0xffffu;
        const int PJ = info.z, po = info.w;
        const double *base = reinterpret_cast<const double *>(ring + info.x);

        if (pull) {
            // A operand: D_J^T[col, q] = scale (chi_J^T Psi_k)[q, col]   (gamma_q is folded into the pull blocks)
            const double *cs = base + __popc(mask_all) * PULL_SZ + ((warp & 7) * 8 + lr) * PJ;
            double dA[KP], d8 = 0.0;
#pragma unroll
            for (int ks = 0; ks < KP; ++ks) {
                const int q = 4 * ks + lq;
                dA[ks] = (q < PJ && (!R1 || q < 8)) ? p.scale * cs[q] : 0.0;
            }
            if (R1) d8 = (8 < PJ) ? p.scale * cs[8] : 0.0;
            // operands of the next block are fetched while the current block's DMMAs issue (reading one block past
            // the job's last stays inside the ring / the C slice)
            const double *bp = base;
            double nb[KP];
            double2 nx8 = make_double2(0.0, 0.0);
#pragma unroll
            for (int ks = 0; ks < KP; ++ks) nb[ks] = bp[ks * 32 + lane];
            if (R1) nx8 = *reinterpret_cast<const double2 *>(bp + KP * 32 + 2 * lq);
#pragma unroll
            for (int o = 0; o < NB_HOCT; ++o) {
                if (mask & (1u << o)) {
                    double b[KP];
#pragma unroll
                    for (int ks = 0; ks < KP; ++ks) b[ks] = nb[ks];
                    const double2 x8 = nx8;
                    bp += PULL_SZ;
#pragma unroll
                    for (int ks = 0; ks < KP; ++ks) nb[ks] = bp[ks * 32 + lane];
                    if (R1) nx8 = *reinterpret_cast<const double2 *>(bp + KP * 32 + 2 * lq);
#pragma unroll
                    for (int ks = 0; ks < KP; ++ks) dmma884(c[o].x, c[o].y, dA[ks], b[ks]);
                    if (R1) {
                        c[o].x = fma(d8, x8.x, c[o].x);
                        c[o].y = fma(d8, x8.y, c[o].y);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[slot]);
            if (jj == na - 1) {                            // all atoms pulled: the tile is the final Out
                if (TMA_IO) {
#pragma unroll
                    for (int o = 0; o < NB_HOCT; ++o) *reinterpret_cast<double2 *>(tile + toff0 + 4096 * o) = c[o];
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // generic writes -> async proxy
                    asm volatile("bar.sync 1, %0;" ::"n"(NLB_WARPS * 32) : "memory");  // the eight consumer warps
                    if (tid == 0) tma_store_tile(&tmap, tile, x0, cg * NLB_COLS, y0, z0);
                } else {
                    double *dstc = p.dst + (int64_t)(colv ? col : 0) * p.ld;
                    int off[NB_HOCT];
#pragma unroll
                    for (int o = 0; o < NB_HOCT; ++o) off[o] = pt_h[8 * o];
#pragma unroll
                    for (int o = 0; o < NB_HOCT; ++o) {
                        const bool ok = ((umask_h >> o) & 1u) && off[o] >= 0 && colv;
                        if (ok) *reinterpret_cast<double2 *>(dstc + off[o]) = c[o];
                    }
                }
            }
        } else {
            // C_J[q, col] += sum_pt chi_J[pt, q] Out[pt, col]; two independent accumulator sets shorten the DMMA chains
            double acc[2][MT][2], p8[2];
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                p8[s] = 0.0;
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) acc[s][mt][0] = acc[s][mt][1] = 0.0;
            }
            const double *bp = base;
            double nb[2 * MT];
            double2 nx8 = make_double2(0.0, 0.0);
#pragma unroll
            for (int k = 0; k < 2 * MT; ++k) nb[k] = bp[k * 32 + lane];
            if (R1) nx8 = *reinterpret_cast<const double2 *>(bp + MT * 64 + 2 * lq);
#pragma unroll
            for (int o = 0; o < NB_HOCT; ++o) {
                if (mask & (1u << o)) {
                    double b[2 * MT];
#pragma unroll
                    for (int k = 0; k < 2 * MT; ++k) b[k] = nb[k];
                    const double2 x8 = nx8;
                    bp += PROJ_SZ;
#pragma unroll
                    for (int k = 0; k < 2 * MT; ++k) nb[k] = bp[k * 32 + lane];
                    if (R1) nx8 = *reinterpret_cast<const double2 *>(bp + MT * 64 + 2 * lq);
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) {
                        dmma884(acc[o & 1][mt][0], acc[o & 1][mt][1], b[2 * mt], c[o].x);
                        dmma884(acc[o & 1][mt][0], acc[o & 1][mt][1], b[2 * mt + 1], c[o].y);
                    }
                    if (R1) {
                        p8[o & 1] = fma(x8.x, c[o].x, p8[o & 1]);
                        p8[o & 1] = fma(x8.y, c[o].y, p8[o & 1]);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[slot]);
            double *cout = p.c_out + (int64_t)po * p.ncp;
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const double v0 = acc[0][mt][0] + acc[1][mt][0];
                const double v1 = acc[0][mt][1] + acc[1][mt][1];
                const int q = mt * 8 + lr;
                const int ca = colw + 2 * lq;
                if (q < PJ && (!R1 || q < 8)) {
                    if (ca < p.ncols) atomicAdd(cout + (int64_t)ca * PJ + q, v0);
                    if (ca + 1 < p.ncols) atomicAdd(cout + (int64_t)(ca + 1) * PJ + q, v1);
                }
            }
            if (R1) {
                double v = p8[0] + p8[1];
                v += __shfl_xor_sync(0xffffffffu, v, 1);
                v += __shfl_xor_sync(0xffffffffu, v, 2);
                if (lq == 0 && colv && 8 < PJ) atomicAdd(cout + (int64_t)col * PJ + 8, v);
            }
        }
    }
    // the bulk store reads the staged tile asynchronously: it must be done before the CTA (and its shared memory) goes
    if (TMA_IO && DO_PULL && tid == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

struct ClassInfo { int kp, mt, r1, pull_sz, proj_sz; };

ClassInfo class_info(int pclass)
{
    if (pclass == 4) return {1, 1, 0, 32, 64};
    return {2, 1, 1, 72, 72};
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
    const ClassInfo ci = class_info(B.pclass);
    const int nbx = nx / B.bx, nby = (ny + B.by - 1) / B.by, nbz = (nz + B.bz - 1) / B.bz;
    const int64_t nbricks = (int64_t)nbx * nby * nbz;
    if (nbricks >= (int64_t)INT32_MAX) return SPARC_GPU_SUCCESS;

    struct Pair { int32_t brick, atom; uint32_t mask; };
    std::vector<Pair> pairs;
    auto locate = [&](int32_t i, int32_t *brick, int *li) {
        const int x = i % nx, y = (i / nx) % ny, z = i / (nx * ny);
        const int bx = x / B.bx, by = y / B.by, bz = z / B.bz;
        *brick = bx + nbx * (by + nby * bz);
        *li = (x - bx * B.bx) + B.bx * ((y - by * B.by) + B.by * (z - bz * B.bz));
    };
    // pass 1: octet masks per (brick, atom)
    for (int J = 0; J < ctx->n_atoms; ++J) {
        if (d->n_proj[J] <= 0) continue;
        std::unordered_map<int32_t, uint32_t> m;
        for (int64_t t = d->supp_ptr[J]; t < d->supp_ptr[J + 1]; ++t) {
            int32_t brick; int li;
            locate(d->supp_idx[t], &brick, &li);
            m[brick] |= 1u << (li >> 3);
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
    int64_t nblocks = 0;
    for (size_t k = 0; k < pairs.size(); ++k) {
        if (k == 0 || pairs[k].brick != pairs[k - 1].brick) {
            const int32_t b = pairs[k].brick;
            const int bx = b % nbx, by = (b / nbx) % nby, bz = b / (nbx * nby);
            org.push_back(bx * B.bx); org.push_back(by * B.by); org.push_back(bz * B.bz); org.push_back(0);
            job_ptr.push_back((int32_t)k);
        }
        org[org.size() - 1] |= (int32_t)pairs[k].mask;
        jobs[k] = {pairs[k].atom, pairs[k].mask, nblocks, pofs[(size_t)pairs[k].atom], d->n_proj[pairs[k].atom]};
        nblocks += __builtin_popcount(pairs[k].mask);
    }
    job_ptr.push_back((int32_t)pairs.size());
    B.n_active = (int32_t)(job_ptr.size() - 1);
    B.n_blocks = nblocks;

    // pass 2: chi blocks in fragment order
    std::vector<double> pull((size_t)nblocks * ci.pull_sz, 0.0), proj((size_t)nblocks * ci.proj_sz, 0.0);
    // per atom: brick -> job index
    std::vector<std::unordered_map<int32_t, int64_t>> jobof((size_t)ctx->n_atoms);
    for (size_t k = 0; k < pairs.size(); ++k) jobof[(size_t)pairs[k].atom][pairs[k].brick] = (int64_t)k;
    for (int J = 0; J < ctx->n_atoms; ++J) {
        const int P = d->n_proj[J];
        if (P <= 0) continue;
        const int64_t s0 = d->supp_ptr[J], nJ = d->supp_ptr[J + 1] - s0;
        const double *chi = d->chi + d->chi_ptr[J];
        for (int64_t t = 0; t < nJ; ++t) {
            int32_t brick; int li;
            locate(d->supp_idx[s0 + t], &brick, &li);
            const BrickJob &job = jobs[(size_t)jobof[(size_t)J][brick]];
            const int o = li >> 3, r = li & 7;
            const int64_t blk = job.blk0 + __builtin_popcount(job.mask & ((1u << o) - 1u));
            double *bp = pull.data() + blk * ci.pull_sz;
            double *bj = proj.data() + blk * ci.proj_sz;
            for (int q = 0; q < P; ++q) {
                const double v = chi[t + (int64_t)q * nJ];
                const double vg = v * d->gamma[pofs[(size_t)J] + q];       // pull blocks carry chi * gamma
                if (ci.r1 && q == 8) {
                    bp[ci.kp * 32 + r] = vg;
                    bj[ci.mt * 64 + r] = v;
                    continue;
                }
                // pull B fragment of k-step q/4: lane = 4 * point + q % 4
                bp[(q >> 2) * 32 + r * 4 + (q & 3)] = vg;
                // projection A fragment (m-tile q/8, k-step r%2): lane = 4 * (q % 8) + r / 2
                bj[(2 * (q >> 3) + (r & 1)) * 32 + (q & 7) * 4 + (r >> 1)] = v;
            }
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
    if ((st = upload_vec(&B.d_pull, pull))) return st;
    if ((st = upload_vec(&B.d_proj, proj))) return st;
    B.ok = 1;
    return SPARC_GPU_SUCCESS;
}

void nlb_free(sparc_gpu_ctx *ctx)
{
    NlBrick &B = ctx->nlb;
    cudaFree(B.d_org); cudaFree(B.d_job_ptr); cudaFree(B.d_jobs); cudaFree(B.d_pull); cudaFree(B.d_proj);
    B = NlBrick();
}

bool nlb_supported(const sparc_gpu_ctx *ctx, const double *X, int64_t ld)
{
    return ctx->nlb.ok && (((uintptr_t)X & 15) == 0) && (ld % 2 == 0);
}

namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// (x, column, y, z) tensor map over the N_d x ncols block with a bx x 64 x by x bz box: one brick x 64 columns
bool encode_tile_map(const sparc_gpu_ctx *ctx, CUtensorMap *tm, const double *base, int64_t ld, int64_t ncols)
{
    const NlBrick &B = ctx->nlb;
    const int nx = ctx->n[0], ny = ctx->n[1], nz = ctx->n[2];
    const cuuint64_t gdim[4] = {(cuuint64_t)nx, (cuuint64_t)ncols, (cuuint64_t)ny, (cuuint64_t)nz};
    const cuuint64_t gstr[3] = {(cuuint64_t)ld * 8, (cuuint64_t)nx * 8, (cuuint64_t)nx * ny * 8};
    const cuuint32_t box[4] = {(cuuint32_t)B.bx, (cuuint32_t)NLB_COLS, (cuuint32_t)B.by, (cuuint32_t)B.bz};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult cr = ((EncodeTiledFn)ctx->fn_encode_tiled)(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void *)base, gdim, gstr, box,
                                                        estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                                        CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return cr == CUDA_SUCCESS;
}

template <int KP, int MT, bool R1, bool TMA_IO>
int launch_class(sparc_gpu_ctx *ctx, int mode, const CUtensorMap &tmap, const BrickParams &P, unsigned grid, cudaStream_t st)
{
    constexpr size_t SMEM = (size_t)(TMA_IO ? NLB_TILE_BYTES + NLB_RING_TMA : NLB_RING_BYTES) + NB_PTS * 4 +
                            NLB_SLOTS * (8 + 8 + 5 * 4) + 16;
    void (*kern)(const CUtensorMap, const BrickParams) = mode == 1 ? nl_brick_kernel<KP, MT, R1, false, true, TMA_IO>
                                                         : mode == 2 ? nl_brick_kernel<KP, MT, R1, true, false, TMA_IO>
                                                                     : nl_brick_kernel<KP, MT, R1, true, true, TMA_IO>;
    SPARC_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM));
    prof_begin(ctx, KK_NL_BRICK, st);
    kern<<<grid, (NLB_WARPS + 1) * 32, SMEM, st>>>(tmap, P);
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
    const int64_t ngroups = (ncols + NLB_COLS - 1) / NLB_COLS;
    if ((int64_t)B.n_active * ngroups >= (int64_t)INT32_MAX) return SPARC_GPU_UNSUPPORTED;
    BrickParams P;
    P.brick_org = B.d_org; P.job_ptr = B.d_job_ptr; P.jobs = (const BrickJob *)B.d_jobs;
    P.blk_pull = B.d_pull; P.blk_proj = B.d_proj;
    P.src = XorOut; P.dst = XorOut; P.ld = ld;
    P.c_in = c_in; P.c_out = c_out;
    P.ncp = nlb_c_cols(ncols);
    P.ncols = (int32_t)ncols;
    P.ncolgroups = (int32_t)ngroups;
    P.nx = ctx->n[0]; P.ny = ctx->n[1]; P.nz = ctx->n[2];
    P.bx = B.bx; P.by = B.by; P.bz = B.bz;
    P.scale = scale;
    const unsigned grid = (unsigned)((int64_t)B.n_active * ngroups);
    // tile staged by TMA when the driver entry point is there (option "nlb_tma" = 1 turns it off)
    CUtensorMap tmap;
    const bool tma = ctx->fn_encode_tiled && ctx->opt_nlb_tma != 1 && encode_tile_map(ctx, &tmap, XorOut, ld, ncols);
    if (!tma) memset(&tmap, 0, sizeof(tmap));
    if (B.pclass == 4) {
        if (tma) SPARC_TRY((launch_class<1, 1, false, true>(ctx, mode, tmap, P, grid, st)));
        else SPARC_TRY((launch_class<1, 1, false, false>(ctx, mode, tmap, P, grid, st)));
    } else {
        if (tma) SPARC_TRY((launch_class<2, 1, true, true>(ctx, mode, tmap, P, grid, st)));
        else SPARC_TRY((launch_class<2, 1, true, false>(ctx, mode, tmap, P, grid, st)));
    }
    return SPARC_GPU_SUCCESS;
}
