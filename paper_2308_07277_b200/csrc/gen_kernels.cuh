// The unfused xy passes (sm_100a): what the library runs when the fused plane kernel (fft_kernels.cuh k_plane) cannot
// take a box -- n1 != n2 (the fused kernel uses one line factorisation for x and y), an axis longer than 144, or a plane
// array X * n2 that does not fit one SM's shared memory (GSpace takes any lattice and cut-off; 1490, 1666:
// the 432- and 1024-atom runs).  Same mathematics, same phase functions (fft_phases.cuh), same transposed labels, so the z
// kernels, the V / box layouts and every entry point stay as they are; the difference is that the half-transformed data
// of a z-plane goes through HBM as a "slab" instead of staying in shared memory (design D1):
//   slab[bp][r][c]   bp = band * n3 + p (p = transposed z label),  r = plane row (occupied i1),  c = transposed y label
//   k_gen_y<CY, true>   sticks of a row (W) -> backward y transform -> slab row            (one team per row)
//   k_gen_x<CX, MODE>   slab column tile -> shared memory -> the x round trip of MODE (fft_kernels.cuh) -> slab
//   k_gen_y<CY, false>  slab row -> forward y transform -> occupied sticks (W)
// Each pass is HBM-bound by construction: 16 B read + 16 B written per slab element.
#pragma once
#include <cuda_runtime.h>
#include "fft_phases.cuh"
#include "async_copy.cuh"
#include "qm_plan.h"

#ifndef QM_GEN_X_MINB
#define QM_GEN_X_MINB 4      /* resident CTAs per SM the x pass is compiled for (168 registers: 4 x 3 warps per SM; measured
                               -23 % x-pass time against the uncapped 176-254 registers and 2 CTAs) */
#endif
#ifndef QM_GEN_XG
#define QM_GEN_XG 1          /* 96-thread groups per CTA of the x pass: 1 = independent groups, several resident CTAs per SM */
#endif
constexpr int GEN_GROUP = 96;                   // threads per CTA of the y pass = one group of GEN_GROUP / TT teams
template <class C> struct GenGeom {
    static constexpr int TPG = GEN_GROUP / C::TT;              // teams (lines) per 96 threads
    static constexpr int LP = C::L | 1;                        // line pitch in shared memory
    static constexpr int XG = QM_GEN_XG;                       // groups per CTA of the x pass
    static constexpr int TC = XG * TPG;                        // columns per x tile
    static constexpr int TCP = TC | 1;                         // tile row pitch (odd)
    static __host__ __device__ size_t y_smem() { return 2 * (size_t)TPG * LP * sizeof(c128); }
    static __host__ __device__ size_t x_smem(int X) { return (2 * (size_t)X * TCP + (size_t)TC * LP) * sizeof(c128); }
};

// 16-byte asynchronous global -> shared copy (LDGSTS); src_bytes = 0 zero-fills the destination
__device__ __forceinline__ void gen_cp_async16(void *smem_dst, const void *gsrc, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gsrc), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void gen_cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void gen_cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Persistent: a CTA walks chunks of TPG rows gridDim.x apart (twiddle row loaded once).  The slab side is moved by the
// whole CTA with consecutive lanes on consecutive elements of a row (a thread's own R2 outputs are 16 B pieces 16 R2 B
// apart: one wavefront per lane, measured 2.4 x slower): backward, the finished lines are copied out of shared memory;
// forward, the rows of the NEXT chunk land asynchronously in a second set of lines while this chunk is transformed.
template <class C, bool BACK>
__global__ void __launch_bounds__(GEN_GROUP, QM_GEN_X_MINB)
k_gen_y(QmKPlanDev kp, const c128 *__restrict__ tw, c128 *__restrict__ W, c128 *__restrict__ slab, int n3, int bp0, int nbp,
        int quarter, size_t wband)
{
    extern __shared__ __align__(16) unsigned char gen_smem[];
    using GG = GenGeom<C>;
    constexpr int TPG = GG::TPG, LP = GG::LP;
    const int tid = threadIdx.x, team = tid / C::TT, u = tid % C::TT;
    const int X = kp.nx;
    c128 *lines = reinterpret_cast<c128 *>(gen_smem);                  // [TPG][LP] (forward: two sets)
    TwRow<BACK ? C::R1 : C::R2> twr;
    load_twrow(twr, tw, u, BACK ? C::R2 : C::R1);
    pdl_launch_dependents();
    pdl_wait();                 // W and the slab come from the previous kernels
    const int items = nbp * X, nchunks = (items + TPG - 1) / TPG;            // 32-bit: a launch holds < 2^31 rows (host checks)
    // rows of a chunk are consecutive slab rows: row (chunk * TPG + t) of the launch at slab + that * N
    auto rows_in = [&](int chunk) { return max(0, min(TPG, items - chunk * TPG)); };
    auto stage_rows = [&](int chunk, c128 *set) {      // forward: asynchronous copy of the chunk's rows into padded lines
        const c128 *src = slab + (size_t)chunk * TPG * C::N;
        const int n = rows_in(chunk) * C::N;
        for (int i = tid; i < n; i += blockDim.x) {
            const int t = i / C::N, l = i % C::N;
            gen_cp_async16(set + t * LP + C::pos(l), src + i, 16);
        }
    };
    struct Item { bool ok; Pruned pr; WView Wp; };
    auto item_of = [&](int chunk) {          // this team's row of a chunk: its sticks in W and their hoisted addressing
        const int item = chunk * TPG + team;
        Item it;
        it.ok = team < TPG && chunk < nchunks && item < items;
        const int bpl = it.ok ? item / X : 0, r = it.ok ? item - bpl * X : 0;      // plane within this launch, row
        const int bp = bp0 + bpl, band = bp / n3, p = bp - band * n3;
        const int4 q = kp.row_info[r];
        it.pr = make_pruned_packed<C>(q.x, q.y, u, 1);
        if (!it.ok) it.pr.m1 = it.pr.m2 = 0u;
        it.Wp = qm_wview(W + (size_t)band * wband, p, n3) + q.z;
        return it;
    };
    int cur = 0;
    Item itc = item_of(blockIdx.x);
    c128 pre[2 * Quarter<C>::Q];
    if constexpr (BACK) {
        if (quarter) prefetch_quarter<C>(itc.Wp, C::R2, itc.pr, pre);
    } else {
        if ((int)blockIdx.x < nchunks) stage_rows(blockIdx.x, lines);
        gen_cp_async_commit();
    }
    for (int chunk = blockIdx.x; chunk < nchunks; chunk += gridDim.x) {       // same trip count for the whole CTA
        const Item itn = item_of(chunk + gridDim.x);
        if constexpr (BACK) {
            const SLine line = qm_sline(lines + (size_t)(team < TPG ? team : 0) * LP);
            if (itc.ok) {
                if (quarter) prunedA_step1_pre<C>(pre, line, u, twr);
                else prunedA_step1<C>(itc.Wp, C::R2, itc.pr, line, u, twr);
            }
            if (quarter) prefetch_quarter<C>(itn.Wp, C::R2, itn.pr, pre);          // the next chunk's sticks, masked off past the end
            __syncthreads();
            if (itc.ok) lineA_step2<C>(line, u);
            __syncthreads();
            c128 *dst = slab + (size_t)chunk * TPG * C::N;
            const int n = rows_in(chunk) * C::N;
            for (int i = tid; i < n; i += blockDim.x) dst[i] = lines[(i / C::N) * LP + C::pos(i % C::N)];
        } else {
            c128 *set = lines + (size_t)cur * TPG * LP;
            if (chunk + (int)gridDim.x < nchunks) stage_rows(chunk + gridDim.x, lines + (size_t)(cur ^ 1) * TPG * LP);
            gen_cp_async_commit();
            gen_cp_async_wait<1>();
            __syncthreads();
            const SLine line = qm_sline(set + (size_t)(team < TPG ? team : 0) * LP);
            if (itc.ok) lineB_step1<C>(line, u, twr);
            __syncthreads();
            if (itc.ok) {
                if (quarter) prunedB_step2_quarter<C>(line, itc.Wp, C::R2, itc.pr, u);
                else prunedB_step2<C>(line, itc.Wp, C::R2, itc.pr, u);
            }
            cur ^= 1;
        }
        __syncthreads();       // the lines are free for the next chunk
        itc = itn;
    }
    if constexpr (!BACK) gen_cp_async_wait<0>();
}

// x pass.  A CTA takes one tile of TC adjacent columns (transposed y labels) of one slab plane: rows r, columns
// c0 .. c0 + TC - 1, staged in shared memory (coalesced row segments), one team per column.
// MODE as in the fused kernel: 0 apply (x V), 1 g2r (write transposed boxes), 2 r2g (read transposed boxes, optionally
// times the conjugate of a second one), 3 density, 4 apply with a complex field.  In MODE 3 a CTA owns its tile for ALL
// bands of the launch and walks them in order, so every point of rho is summed by one thread in band order.
template <class C, int MODE>
__global__ void __launch_bounds__(GenGeom<C>::XG * GEN_GROUP, QM_GEN_X_MINB)
k_gen_x(QmKPlanDev kp, const c128 *__restrict__ tw, const double *__restrict__ vt, c128 *__restrict__ slab,
        c128 *__restrict__ box, const c128 *__restrict__ box2, int npair2, double scale, int n2, int n3, int bp0, int nbp,
        int quarter, const double *__restrict__ occ, double *__restrict__ rhot)
{
    extern __shared__ __align__(16) unsigned char gen_smem[];
    using GG = GenGeom<C>;
    constexpr int TC = GG::TC, TCP = GG::TCP, LP = GG::LP;
    constexpr bool LOADS = MODE != 2, STORES = MODE != 1 && MODE != 3;
    const int X = kp.nx;
    c128 *tiles = reinterpret_cast<c128 *>(gen_smem);                  // two buffers [X][TCP]: the next tile lands while this one is worked on
    c128 *scr = tiles + 2 * (size_t)X * TCP;                           // [TC][LP]
    const int tid = threadIdx.x, grp = tid / GEN_GROUP, gl = tid % GEN_GROUP;
    const int team = gl / C::TT, u = gl % C::TT;
    const bool team_ok = team < GG::TPG;
    const int tcol = grp * GG::TPG + team;                              // column of the tile this team owns
    const int nchunk = (n2 + TC - 1) / TC;
    const bool xq = (quarter & 2) != 0;
    TwRow<C::R1> twa;
    load_twrow(twa, tw, u, C::R2);
    TwRow<C::R2> twb;
    load_twrow(twb, tw, u, C::R1);
    const Pruned px = make_pruned<C>(kp.x_iv.x, kp.x_iv.y, kp.x_iv.z, kp.x_iv.w, u, TCP);
    const SLine myscr = qm_sline(scr + (size_t)(team_ok ? tcol : 0) * LP);
    // The work list of this CTA: tiles tl = blockIdx.x, + gridDim.x, ...; MODE 3 walks each tile (p, chunk) over the
    // nbp / n3 bands of the launch in order (one CTA sums a point of rho, in band order), the others have one plane per tile.
    const int nloop = MODE == 3 ? nbp / n3 : 1;
    const long long ntiles = (long long)(MODE == 3 ? n3 : nbp) * nchunk;
    auto plane_of = [&](long long tl, int lb) { return MODE == 3 ? lb * n3 + (int)(tl / nchunk) : (int)(tl / nchunk); };
    auto stage = [&](long long tl, int lb, c128 *buf) {       // asynchronous copy of a tile: rows are contiguous in the slab
        const c128 *plane = slab + (size_t)plane_of(tl, lb) * X * n2;
        const int c0 = (int)(tl % nchunk) * TC;
        for (int i = tid; i < X * TC; i += blockDim.x) {
            const int r = i / TC, cc = i % TC;
            const bool in = c0 + cc < n2;
            gen_cp_async16(buf + r * TCP + cc, plane + (size_t)r * n2 + (in ? c0 + cc : 0), in ? 16 : 0);
        }
    };
    pdl_launch_dependents();
    pdl_wait();                 // the slab (and the boxes) come from the previous kernels
    int cur = 0;
    if constexpr (LOADS) {
        if ((long long)blockIdx.x < ntiles) stage(blockIdx.x, 0, tiles);
        gen_cp_async_commit();
    }
    for (long long tl = blockIdx.x; tl < ntiles; tl += gridDim.x)
    for (int lb = 0; lb < nloop; ++lb) {
        const int chunk = (int)(tl % nchunk);
        const int bpl = plane_of(tl, lb);
        const int bp = bp0 + bpl, band = bp / n3, p = bp - band * n3;
        const int c0 = chunk * TC, col = c0 + tcol;
        const bool ok = team_ok && col < n2;
        c128 *tile = tiles + (size_t)cur * X * TCP;
        const SLine Acol = qm_sline(tile + (team_ok ? tcol : 0));
        VRow<C::R2> vr;
        if constexpr (MODE == 0) { if (ok) load_vrow<C>(vr, vt + ((size_t)p * n2 + col) * VLayout<C>::COL, u); }
        if constexpr (LOADS) {
            // next tile of this CTA into the other buffer (its last readers passed the barrier that ended their iteration)
            const bool more_lb = lb + 1 < nloop;
            const long long ntl = more_lb ? tl : tl + gridDim.x;
            if (ntl < ntiles) stage(ntl, more_lb ? lb + 1 : 0, tiles + (size_t)(cur ^ 1) * X * TCP);
            gen_cp_async_commit();
            gen_cp_async_wait<1>();            // this tile has landed (this thread's copies; the barrier covers the others')
            __syncthreads();
            if (ok) {
                if (xq) prunedA_step1_quarter<C>(Acol, C::R2 * TCP, px, myscr, u, twa);
                else prunedA_step1<C>(Acol, C::R2 * TCP, px, myscr, u, twa);
            }
            __syncthreads();
        }
        if constexpr (MODE == 3) {
            if (ok) xcol_density<C>(myscr, u, rhot + ((size_t)p * n2 + col) * VLayout<C>::COL, scale * occ[band]);
        } else {
            c128 *bx = nullptr;
            const c128 *bx2 = nullptr;
            const size_t coloff = ((size_t)p * n2 + (ok ? col : 0)) * C::N, boxsz = (size_t)C::N * n2 * n3;
            if constexpr (MODE == 1) bx = box + (size_t)band * boxsz + coloff;
            if constexpr (MODE == 2) {
                bx = box + (size_t)(npair2 > 0 ? band / npair2 : band) * boxsz + coloff;
                if (npair2 > 0) bx2 = box2 + (size_t)(band % npair2) * boxsz + coloff;
            }
            if constexpr (MODE == 4) bx2 = box2 + coloff;
            if (ok) xcol_step2<C, MODE>(myscr, u, twb, vr, bx, bx2, scale);
        }
        if constexpr (STORES) {
            __syncthreads();
            if (ok) {
                if (xq) prunedB_step2_quarter<C>(myscr, Acol, C::R2 * TCP, px, u);
                else prunedB_step2<C>(myscr, Acol, C::R2 * TCP, px, u);
            }
            __syncthreads();
            c128 *plane = slab + (size_t)bpl * X * n2;
            for (int i = tid; i < X * TC; i += blockDim.x) {
                const int r = i / TC, cc = i % TC;
                if (c0 + cc < n2) plane[(size_t)r * n2 + c0 + cc] = tile[r * TCP + cc];
            }
        }
        __syncthreads();
        if constexpr (LOADS) cur ^= 1;
    }
    if constexpr (LOADS) gen_cp_async_wait<0>();
}
