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
#include "qm_plan.h"

constexpr int GEN_GROUP = 96;                   // threads per CTA of the y pass = one group of GEN_GROUP / TT teams
template <class C> struct GenGeom {
    static constexpr int TPG = GEN_GROUP / C::TT;              // teams (lines) per 96 threads
    static constexpr int LP = C::L | 1;                        // line pitch in shared memory
    static constexpr int XG = 2;                               // groups per CTA of the x pass
    static constexpr int TC = XG * TPG;                        // columns per x tile
    static constexpr int TCP = TC | 1;                         // tile row pitch (odd)
    static __host__ __device__ size_t y_smem() { return (size_t)TPG * LP * sizeof(c128); }
    static __host__ __device__ size_t x_smem(int X) { return ((size_t)X * TCP + (size_t)TC * LP) * sizeof(c128); }
};

// second backward pass of a line, written to a global row in label order (label = k1 * R2 + k2)
template <class C, class L> QM_HD void lineA_step2_to_row(const L line, int u, c128 *row) {
    if (u >= C::R1) return;
    c128 t[C::R2];
    static_for<C::R2>([&](auto I) { constexpr int n2 = decltype(I)::value; t[n2] = line[u * C::R2P + n2]; });
    Dft<C::R2, +1>::run(t);
    static_for<C::R2>([&](auto I) { constexpr int k2 = decltype(I)::value; row[u * C::R2 + k2] = t[k2]; });
}
// first forward pass of a line, read from a global row in label order
template <class C, class L, class TW> QM_HD void lineB_step1_from_row(const c128 *row, const L line, int u, const TW &tw) {
    if (u >= C::R1) return;
    c128 t[C::R2];
    static_for<C::R2>([&](auto I) { constexpr int b = decltype(I)::value; t[b] = row[u * C::R2 + b]; });
    Dft<C::R2, -1>::run(t);
    stepB1_tail<C>(t, line, u, tw);
}

template <class C, bool BACK>
__global__ void __launch_bounds__(GEN_GROUP)
k_gen_y(QmKPlanDev kp, const c128 *__restrict__ tw, c128 *__restrict__ W, c128 *__restrict__ slab, int n3, int bp0, int nbp,
        int quarter, size_t wband)
{
    extern __shared__ __align__(16) unsigned char gen_smem[];
    using GG = GenGeom<C>;
    const int tid = threadIdx.x, team = tid / C::TT, u = tid % C::TT;
    const int X = kp.nx;
    const long long item = (long long)blockIdx.x * GG::TPG + team;
    const bool ok = team < GG::TPG && item < (long long)nbp * X;
    const int bpl = ok ? (int)(item / X) : 0, r = ok ? (int)(item % X) : 0;      // plane within this launch, row
    const int bp = bp0 + bpl, band = bp / n3, p = bp - band * n3;
    const SLine line = qm_sline(reinterpret_cast<c128 *>(gen_smem) + (size_t)(team < GG::TPG ? team : 0) * GG::LP);
    const int4 q = kp.row_info[r];
    const Pruned pr = make_pruned_packed<C>(q.x, q.y, u, 1);
    const WView Wp = qm_wview(W + (size_t)band * wband, p, n3) + q.z;
    c128 *row = slab + ((size_t)bpl * X + r) * C::N;
    if constexpr (BACK) {
        TwRow<C::R1> twa;
        load_twrow(twa, tw, u, C::R2);
        if (ok) {
            if (quarter) prunedA_step1_quarter<C>(Wp, C::R2, pr, line, u, twa);
            else prunedA_step1<C>(Wp, C::R2, pr, line, u, twa);
        }
        __syncthreads();
        if (ok) lineA_step2_to_row<C>(line, u, row);
    } else {
        TwRow<C::R2> twb;
        load_twrow(twb, tw, u, C::R1);
        if (ok) lineB_step1_from_row<C>(row, line, u, twb);
        __syncthreads();
        if (ok) {
            if (quarter) prunedB_step2_quarter<C>(line, Wp, C::R2, pr, u);
            else prunedB_step2<C>(line, Wp, C::R2, pr, u);
        }
    }
}

// x pass.  A CTA takes one tile of TC adjacent columns (transposed y labels) of one slab plane: rows r, columns
// c0 .. c0 + TC - 1, staged in shared memory (coalesced row segments), one team per column.
// MODE as in the fused kernel: 0 apply (x V), 1 g2r (write transposed boxes), 2 r2g (read transposed boxes, optionally
// times the conjugate of a second one), 3 density, 4 apply with a complex field.  In MODE 3 a CTA owns its tile for ALL
// bands of the launch and walks them in order, so every point of rho is summed by one thread in band order.
template <class C, int MODE>
__global__ void __launch_bounds__(GenGeom<C>::XG * GEN_GROUP)
k_gen_x(QmKPlanDev kp, const c128 *__restrict__ tw, const double *__restrict__ vt, c128 *__restrict__ slab,
        c128 *__restrict__ box, const c128 *__restrict__ box2, int npair2, double scale, int n2, int n3, int bp0, int nbp,
        int quarter, const double *__restrict__ occ, double *__restrict__ rhot)
{
    extern __shared__ __align__(16) unsigned char gen_smem[];
    using GG = GenGeom<C>;
    constexpr int TC = GG::TC, TCP = GG::TCP, LP = GG::LP;
    const int X = kp.nx;
    c128 *tile = reinterpret_cast<c128 *>(gen_smem);                   // [X][TCP]
    c128 *scr = tile + (size_t)X * TCP;                                // [TC][LP]
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
    const SLine Acol = qm_sline(tile + (team_ok ? tcol : 0));
    // MODE 3: blockIdx.x = (p, chunk), loop over the nbp / n3 bands; else blockIdx.x = (plane of the launch, chunk)
    const int nloop = MODE == 3 ? nbp / n3 : 1;
    for (int lb = 0; lb < nloop; ++lb) {
        const int chunk = (int)(blockIdx.x % nchunk);
        const int bpl = MODE == 3 ? lb * n3 + (int)(blockIdx.x / nchunk) : (int)(blockIdx.x / nchunk);
        const int bp = bp0 + bpl, band = bp / n3, p = bp - band * n3;
        const int c0 = chunk * TC, col = c0 + tcol;
        const bool ok = team_ok && col < n2;
        c128 *plane = slab + (size_t)bpl * X * n2;
        if constexpr (MODE != 2) {       // stage the tile: rows are contiguous in the slab
            for (int i = tid; i < X * TC; i += blockDim.x) {
                const int r = i / TC, cc = i % TC;
                tile[r * TCP + cc] = (c0 + cc < n2) ? plane[(size_t)r * n2 + c0 + cc] : c128{0.0, 0.0};
            }
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
            VRow<C::R2> vr;
            if constexpr (MODE == 0) { if (ok) load_vrow<C>(vr, vt + ((size_t)p * n2 + col) * VLayout<C>::COL, u); }
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
        if constexpr (MODE != 1 && MODE != 3) {
            __syncthreads();
            if (ok) {
                if (xq) prunedB_step2_quarter<C>(myscr, Acol, C::R2 * TCP, px, u);
                else prunedB_step2<C>(myscr, Acol, C::R2 * TCP, px, u);
            }
            __syncthreads();
            for (int i = tid; i < X * TC; i += blockDim.x) {
                const int r = i / TC, cc = i % TC;
                if (c0 + cc < n2) plane[(size_t)r * n2 + c0 + cc] = tile[r * TCP + cc];
            }
        }
        __syncthreads();
    }
}
