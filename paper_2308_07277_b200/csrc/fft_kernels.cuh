// CUDA kernels of the pruned 3-D FFT path (sm_100a).  DESIGN.md section 6.
//   k_zinv  : a1+a2(z)  scatter sphere -> z-sticks, backward z-FFT, write stick planes  W[band][p][S]
//   k_plane : a2(y,x)+a3+a4(x,y)  per (band, z-plane): y-FFT on X rows, x-FFT 'X->N1', V multiply,
//             x-FFT 'N1->X', y-FFT, all in shared memory; reads/writes only the S stick values
//   k_zfwd  : a4(z)+a5  forward z-FFT, gather to the sphere, + 1/2|k+G|^2 psi_in
#pragma once
#include <cuda_runtime.h>
#include "fft_phases.cuh"
#include "async_copy.cuh"
#include "qm_plan.h"

// z kernels.  A CTA owns tiles of QM_ZT adjacent sticks of one band (looping over tiles gridDim.x apart, so the
// per-thread twiddle row is loaded once).  The stick-plane workspace W is blocked by tile (WView): a tile's
// N3 x QM_ZT block is contiguous and moves with ONE bulk asynchronous copy (TMA engine) through a shared-memory
// staging buffer.  Sphere side: the G of a stick are two contiguous runs of psi (Pruned), loaded straight into
// registers one tile ahead (quarter rule), no zero fill, no table-driven scatter.  Thread mapping is (stick, u)
// with u fastest on the sphere side and (u, stick) with the stick fastest on the staging side.
template <class C> __host__ __device__ constexpr size_t qm_z_smem() {
    return ((size_t)QM_ZT * (C::L | 1) + (size_t)C::N * QM_ZT) * sizeof(c128) + 16;
}

// PH: multiply psi(G) by the per-G factor phase[g] as it is loaded (split-operator half-step, eq. 53).
template <class C, bool PH>
__global__ void __launch_bounds__(QM_ZT * C::TT, 2)
k_zinv(QmKPlanDev kp, const c128 *__restrict__ tw, const c128 *__restrict__ psi, const c128 *__restrict__ phase,
       c128 *__restrict__ W, int ntiles, int quarter)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int LP = C::L | 1;
    constexpr int NPRE = 2 * Quarter<C>::Q;
    c128 *stage = reinterpret_cast<c128 *>(smem_raw);                 // [N][QM_ZT], 128-byte aligned
    c128 *lines = stage + (size_t)C::N * QM_ZT;
    const int tid = threadIdx.x;
    const int S = kp.nsticks, band = blockIdx.y;
    const int t1 = tid / C::TT, u1 = tid % C::TT;      // pass 1: u fastest
    const int t2 = tid % QM_ZT, u2 = tid / QM_ZT;      // pass 2: stick fastest
    TwRow<C::R1> twa;
    load_twrow(twa, tw, u1, C::R2);
    const c128 *psib_raw = psi + (size_t)band * kp.ng;
    const auto psib = [&]() {
        if constexpr (PH) return PhasedPtr{psib_raw, phase}; else return psib_raw;
    }();
    c128 *Wb = W + (size_t)band * ntiles * C::N * QM_ZT;
    auto info = [&](int tile) {
        const int s = tile * QM_ZT + t1;
        return (tile < ntiles && s < S) ? kp.stick_info[s] : int4{1, 1, 0, 0};   // both intervals empty
    };
    auto pruned_of = [&](const int4 q) {
        return make_pruned<C>((int)(short)(q.x & 0xffff), q.x >> 16, (int)(short)(q.y & 0xffff), q.y >> 16, u1, 1);
    };
    int4 q = info(blockIdx.x), qn = info(blockIdx.x + gridDim.x);
    Pruned pr = pruned_of(q);
    c128 pre[NPRE];
    if (quarter) prefetch_quarter<C>(psib + q.z, C::R2, pr, pre);
    const SLine lines_s = qm_sline(lines), stage_s = qm_sline(stage);
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int ns = min(QM_ZT, S - tile * QM_ZT);
        if (t1 < ns) {
            if (quarter) prunedA_step1_pre<C>(pre, lines_s + t1 * LP, u1, twa);
            else prunedA_step1<C>(psib + q.z, C::R2, pr, lines_s + t1 * LP, u1, twa);
        }
        // advance the two-deep prefetch: data of the next tile, table entry of the one after
        q = qn; pr = pruned_of(q);
        if (quarter) prefetch_quarter<C>(psib + q.z, C::R2, pr, pre);
        qn = info(tile + 2 * gridDim.x);
        if (tid == 0) bulk_wait_read0();      // the previous tile's bulk store has read the staging buffer
        __syncthreads();
        if (t2 < ns) zinv_step2_store<C>(lines_s + t2 * LP, stage_s + t2, QM_ZT, u2);
        fence_async_smem();
        __syncthreads();
        if (tid == 0) { bulk_s2g(Wb + (size_t)tile * C::N * QM_ZT, stage, (uint32_t)(C::N * QM_ZT * sizeof(c128))); bulk_commit(); }
    }
    if (tid == 0) bulk_wait0();
}

// GM: what the gather stores (fft_phases.cuh GM_*).  aux: GM_KINETIC psi_in [nb][ng]; GM_PHASE per-G factors [ng].
template <class C, int GM>
__global__ void __launch_bounds__(QM_ZT * C::TT, 2)
k_zfwd(QmKPlanDev kp, const c128 *__restrict__ tw, const c128 *__restrict__ W,
       const c128 *__restrict__ aux, c128 *__restrict__ out, int ntiles, double scale, int quarter)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int LP = C::L | 1;
    constexpr int NPRE = 2 * Quarter<C>::Q;
    constexpr uint32_t TILE_BYTES = (uint32_t)(C::N * QM_ZT * sizeof(c128));
    c128 *stage = reinterpret_cast<c128 *>(smem_raw);                 // [N][QM_ZT]
    c128 *lines = stage + (size_t)C::N * QM_ZT;
    uint64_t *wbar = reinterpret_cast<uint64_t *>(lines + (size_t)QM_ZT * LP);
    const int tid = threadIdx.x;
    const int S = kp.nsticks, band = blockIdx.y;
    const int t1 = tid / C::TT, u1 = tid % C::TT;      // pass 2 (gather side): u fastest
    const int t2 = tid % QM_ZT, u2 = tid / QM_ZT;      // pass 1 (staging side): stick fastest
    const c128 *Wb = W + (size_t)band * ntiles * C::N * QM_ZT;
    if (tid == 0) {
        mbar_init(wbar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        mbar_expect_tx(wbar, TILE_BYTES);
        bulk_g2s(stage, Wb + (size_t)blockIdx.x * C::N * QM_ZT, TILE_BYTES, wbar);
    }
    TwRow<C::R2> twb;
    load_twrow(twb, tw, u2, C::R1);
    const size_t boff = (size_t)band * kp.ng;
    const c128 *auxb = GM == GM_KINETIC ? aux + boff : aux;
    __syncthreads();
    const SLine lines_s = qm_sline(lines), stage_s = qm_sline(stage);
    for (int tile = blockIdx.x, it = 0; tile < ntiles; tile += gridDim.x, ++it) {
        const int ns = min(QM_ZT, S - tile * QM_ZT);
        // gather-side inputs of this tile: in flight behind the wait and the first pass
        int4 q = int4{1, 1, 0, 0};             // both intervals empty
        if (t1 < ns) q = kp.stick_info[tile * QM_ZT + t1];
        const Pruned pr = make_pruned<C>((int)(short)(q.x & 0xffff), q.x >> 16, (int)(short)(q.y & 0xffff), q.y >> 16, u1, 1);
        c128 kin[NPRE];
        if (quarter) prefetch_kin<C, GM>(auxb + q.z, kp.g2 + q.z, pr, t1 < ns, kin);
        mbar_wait(wbar, (uint32_t)(it & 1));
        zfwd_step1_load<C>(stage_s + t2, QM_ZT, lines_s + t2 * LP, u2, twb);
        __syncthreads();                       // staging buffer consumed, lines complete
        if (tid == 0 && tile + (int)gridDim.x < ntiles) {
            fence_async_smem();
            mbar_expect_tx(wbar, TILE_BYTES);
            bulk_g2s(stage, Wb + (size_t)(tile + gridDim.x) * C::N * QM_ZT, TILE_BYTES, wbar);
        }
        if (t1 < ns) {
            if (quarter) zfwd_step2_gather_pre<C, GM>(lines_s + t1 * LP, out + boff + q.z, pr, u1, kin, scale);
            else zfwd_step2_gather<C, GM>(lines_s + t1 * LP, out + boff + q.z, auxb + q.z, kp.g2 + q.z, pr, u1, scale);
        }
        __syncthreads();
    }
}

// MODE 0 apply, 1 g2r (write a transposed box), 2 r2g (read a transposed box, optionally times the conjugate of a second
// one), 3 density (rho += w |psi(r)|^2), 4 apply with a complex field (split-operator middle factor); fft_phases.cuh
//
// One CTA per (band, z-plane).  The CTA is split into independent groups of G threads (G/TT teams of TT
// threads, one team per line); a group walks its own rows / columns and only synchronises with itself
// (named barrier, or __syncwarp when G == 32), so the groups hide each other's latencies.  CTA-wide
// barriers remain only between the phases (y backward | x round trip | y forward).
// All pruned-access masks and offsets are hoisted: per kernel for the x direction (Pruned px), per row for
// the y direction; the accesses themselves are predicated 16-byte loads/stores at base + immediate.
#ifndef QM_PLANE_MAX_THREADS
#define QM_PLANE_MAX_THREADS 384
#endif
#ifndef QM_PLANE_GROUP
#define QM_PLANE_GROUP 96
#endif
#ifndef QM_PLANE_YROWS
#define QM_PLANE_YROWS 1        /* plane rows a team works on between two group barriers of the y phase (2: spills, 343 vs 300 us) */
#endif
#ifndef QM_PLANE_XPREFETCH
#define QM_PLANE_XPREFETCH 0    /* x phase: fetch a column's step-1 inputs one column ahead (quarter rule) */
#endif
constexpr int QM_GROUP = QM_PLANE_GROUP;
// Scratch lines of neighbouring teams: with 12-thread teams a quarter-warp straddles two teams as 4+4
// threads, and their unit-stride 16-byte accesses are conflict free iff the pitch is 4 (mod 8); else odd.
__host__ __device__ constexpr int qm_scratch_pitch(int len, int tt) { return tt == 12 ? len + ((12 - len % 8) % 8) : (len | 1); }
// Which line of its group's chunk a team works on.  With 12-thread teams in 96-thread groups the quarter-warps
// that straddle two teams hold teams (0,1), (2,3), (4,5), (6,7): giving each pair lines 4 apart makes their
// 16-byte accesses to odd-pitch plane rows (pitch = 5 mod 8) and to columns 4 apart fall in disjoint banks.
template <int TT, int TPG> __host__ __device__ constexpr int qm_team_slot(int team) {
    return (TT == 12 && TPG == 8) ? ((team >> 1) + 4 * (team & 1)) : team;
}
template <int G> __device__ __forceinline__ void group_barrier(int grp) {
    if constexpr (G == 32) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "r"(G) : "memory");
}

// Persistent: a CTA walks the (band, z-plane) pairs pl = blockIdx.x, blockIdx.x + gridDim.x, ...  Between two x phases
// the y-forward pass of the plane just finished and the y-backward pass of the next plane run as ONE loop over
// row chunks (a row of the plane array is consumed and refilled by the same team), so there are two CTA-wide
// barriers per plane.  The next plane's stick values of a row are fetched into registers (quarter rule,
// prefetch_quarter) before the y-forward work of that row starts, which hides their latency.
// The two phases are separate (force-inlined) functions; making them __noinline__ to separate their register
// allocation was measured 25 % slower (the x loop then spills at the 168-register cap).
struct PlaneCtx {
    c128 *A, *scr;
    const int4 *rowinfo_s;
    int X, ngroups, n3, quarter;
    size_t wband;
};
template <class C> struct PlaneIds {
    static constexpr int G = QM_GROUP, TPG = G / C::TT;
    int grp, team, u, slot; bool team_ok;
    __device__ PlaneIds() {
        const int tid = threadIdx.x, gl = tid % G;
        grp = tid / G; team = gl / C::TT; u = gl % C::TT;
        team_ok = team < TPG;
        slot = qm_team_slot<C::TT, TPG>(team);
    }
};

template <class C, int MODE>
__device__ __forceinline__ void plane_y_phase(const PlaneCtx cx, c128 *__restrict__ W, int pl, int prev, bool have_cur,
                                              const TwRow<C::R1> &twa, const TwRow<C::R2> &twb)
{
    constexpr int G = QM_GROUP, TPG = G / C::TT, RP = C::L | 1, NPRE = 2 * Quarter<C>::Q;
    constexpr bool HAS_BACK = MODE != 2, HAS_FWD = MODE != 1 && MODE != 3;
    const PlaneIds<C> id;
    const int u = id.u, grp = id.grp, slot = id.slot, X = cx.X, n3 = cx.n3, quarter = cx.quarter & 1;
    const bool do_back = HAS_BACK && have_cur, do_fwd = HAS_FWD && prev >= 0;
    if (!(do_back || do_fwd)) return;
    const SLine As = qm_sline(cx.A);
    const int pc = have_cur ? pl : 0, pp = prev >= 0 ? prev : 0;
    const WView Wcur = qm_wview(W + (size_t)(pc / n3) * cx.wband, pc % n3, n3);
    const WView Wprev = qm_wview(W + (size_t)(pp / n3) * cx.wband, pp % n3, n3);
    // A team works on NR rows per round (rows r, r + rstride, ...): the same number of row steps with 1/NR of the
    // group barriers and NR independent load -> transform -> store chains between two barriers.
    constexpr int NR = QM_PLANE_YROWS;
    const int rstride = cx.ngroups * TPG;
    for (int r0 = grp * TPG + slot; r0 - slot < X; r0 += NR * rstride) {
        bool ok[NR];
        int sbase[NR];
        Pruned pr[NR];
        c128 pre[NR][NPRE];
#pragma unroll
        for (int i = 0; i < NR; ++i) {
            const int r = r0 + i * rstride;
            ok[i] = id.team_ok && r < X;
            sbase[i] = 0;
            pr[i] = Pruned{0u, 0u, 0, 0};
            if (ok[i]) {
                const int4 q = cx.rowinfo_s[r];
                sbase[i] = q.z;
                pr[i] = make_pruned_packed<C>(q.x, q.y, u, 1);
            }
            if (do_back && quarter && ok[i]) prefetch_quarter<C>(Wcur + sbase[i], C::R2, pr[i], pre[i]);
        }
        if (do_fwd) {
#pragma unroll
            for (int i = 0; i < NR; ++i)
                if (ok[i]) lineB_step1<C>(As + (r0 + i * rstride) * RP, u, twb);
            group_barrier<G>(grp);
        }
#pragma unroll
        for (int i = 0; i < NR; ++i) {
            const SLine Arow = As + (r0 + i * rstride) * RP;
            if (do_fwd && ok[i]) {
                if (quarter) prunedB_step2_quarter<C>(Arow, Wprev + sbase[i], C::R2, pr[i], u);
                else prunedB_step2<C>(Arow, Wprev + sbase[i], C::R2, pr[i], u);
            }
            // the team that read the row in the step above is the one that refills it: no barrier needed
            if (do_back && ok[i]) {
                if (quarter) prunedA_step1_pre<C>(pre[i], Arow, u, twa);
                else prunedA_step1<C>(Wcur + sbase[i], C::R2, pr[i], Arow, u, twa);
            }
        }
        if (do_back) {
            group_barrier<G>(grp);
#pragma unroll
            for (int i = 0; i < NR; ++i)
                if (ok[i]) lineA_step2<C>(As + (r0 + i * rstride) * RP, u);
        }
    }
}

template <class C, int MODE>
__device__ __forceinline__ void plane_x_phase(const PlaneCtx cx, const short4 x_iv, const double *__restrict__ vt,
                                           c128 *__restrict__ box, const c128 *__restrict__ box2, int npair2, int pl,
                                           double scale, int stagger_ns,
                                           double *__restrict__ rhot, const TwRow<C::R1> &twa, const TwRow<C::R2> &twb)
{
    constexpr int G = QM_GROUP, TPG = G / C::TT, RP = C::L | 1;
    constexpr int SL = qm_scratch_pitch(C::L, C::TT);    // scratch line pitch
    const PlaneIds<C> id;
    const int u = id.u, grp = id.grp, slot = id.slot, n3 = cx.n3, ngroups = cx.ngroups;
    const bool team_ok = id.team_ok;
    const bool xq = (cx.quarter & 2) != 0;               // quarter rule holds for the x rows: 2Q loads / stores per column
    const SLine As = qm_sline(cx.A);
    const Pruned px = make_pruned<C>(x_iv.x, x_iv.y, x_iv.z, x_iv.w, u, RP);
    const int band = pl / n3, p = pl - band * n3;
    const SLine myscr = qm_sline(cx.scr + (size_t)(grp * TPG + id.team) * SL);
    const double *vplane = vt + (size_t)p * C::N * VLayout<C>::COL;
    VRow<C::R2> vr;
    // De-phase the groups: they all do identical load -> FP64 -> store bursts, and when they run in
    // lock step the shared-memory pipe and the FP64 pipe are used alternately instead of together.
    if (stagger_ns > 0) __nanosleep((unsigned)(grp * stagger_ns));
    const int col0 = grp * TPG + slot;
    if constexpr (MODE == 0) {       // V of the first column: in flight while step 1 runs
        if (team_ok && col0 < C::N) load_vrow<C>(vr, vplane + (size_t)col0 * VLayout<C>::COL, u);
    }
    // Step-1 inputs of a column under the quarter rule: fetched one column ahead (before the barrier in front of the
    // previous column's step 3), so that their shared-memory latency hides behind that barrier and step 3.  Nobody else
    // touches a column of the plane array during the x phase: every column is owned by one team.
    constexpr bool XPRE = (MODE == 0 || MODE == 4) && QM_PLANE_XPREFETCH;
    c128 xpre[2 * Quarter<C>::Q];
    if constexpr (XPRE) {
        if (xq && team_ok && col0 < C::N) prefetch_quarter<C>(As + C::pos(col0), C::R2 * RP, px, xpre);
    }
    for (int col = col0; col - slot < C::N; col += ngroups * TPG) {
        const bool ok = team_ok && col < C::N;
        const SLine Acol = As + C::pos(col);
        if constexpr (MODE != 2) {
            if (ok) {
                if constexpr (XPRE) {
                    if (xq) prunedA_step1_pre<C>(xpre, myscr, u, twa);
                    else prunedA_step1<C>(Acol, C::R2 * RP, px, myscr, u, twa);
                } else {
                    if (xq) prunedA_step1_quarter<C>(Acol, C::R2 * RP, px, myscr, u, twa);
                    else prunedA_step1<C>(Acol, C::R2 * RP, px, myscr, u, twa);
                }
            }
            group_barrier<G>(grp);
        }
        if constexpr (MODE == 3) {
            // scale = weight * occupation of this band; rhot = running density of this plane in the V layout
            if (ok) xcol_density<C>(myscr, u, rhot + ((size_t)p * C::N + col) * VLayout<C>::COL, scale);
        } else if (ok) {
            // transposed boxes (fft_phases.cuh BoxT): column (p, col) of state `band`; with a second operand the plane
            // index counts pairs: band = a * npair2 + b, first operand state a, second operand state b (MODE 2)
            c128 *bx = nullptr;
            const c128 *bx2 = nullptr;
            const size_t coloff = ((size_t)p * C::N + col) * C::N, boxsz = (size_t)C::N * C::N * n3;
            if constexpr (MODE == 1) bx = box + (size_t)band * boxsz + coloff;
            if constexpr (MODE == 2) {
                bx = box + (size_t)(npair2 > 0 ? band / npair2 : band) * boxsz + coloff;
                if (npair2 > 0) bx2 = box2 + (size_t)(band % npair2) * boxsz + coloff;
            }
            if constexpr (MODE == 4) bx2 = box2 + coloff;
            xcol_step2<C, MODE>(myscr, u, twb, vr, bx, bx2, scale);
        }
        if constexpr (MODE == 0) {   // prefetch V of this team's next column behind steps 3 and 1
            const int ncol = col + ngroups * TPG;
            if (team_ok && ncol < C::N) load_vrow<C>(vr, vplane + (size_t)ncol * VLayout<C>::COL, u);
        }
        if constexpr (XPRE) {
            const int ncol = col + ngroups * TPG;
            if (xq && team_ok && ncol < C::N) prefetch_quarter<C>(As + C::pos(ncol), C::R2 * RP, px, xpre);
        }
        group_barrier<G>(grp);
        if constexpr (MODE != 1 && MODE != 3) {
            // no barrier after step 3: the scratch column a thread reads here is exactly the one it
            // overwrites in the next iteration's step 1 (MODE 2 has no step 1 and writes rows: barrier).
            if (ok) {
                if (xq) prunedB_step2_quarter<C>(myscr, Acol, C::R2 * RP, px, u);
                else prunedB_step2<C>(myscr, Acol, C::R2 * RP, px, u);
            }
            if constexpr (MODE == 2) group_barrier<G>(grp);
        }
    }
}

template <class C, int MODE>
__global__ void __launch_bounds__(QM_PLANE_MAX_THREADS)
k_plane(QmKPlanDev kp, QmGridDev gd, c128 *__restrict__ W, c128 *__restrict__ box, const c128 *__restrict__ box2,
        int npair2, int ngroups, double scale, int stagger_ns, int nplanes, int quarter, const double *__restrict__ occ,
        double *__restrict__ rhot)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int G = QM_GROUP;
    constexpr int SL = qm_scratch_pitch(C::L, C::TT);
    constexpr int TPG = G / C::TT;
    constexpr int RP = C::L | 1;                         // plane row pitch (== kp.rowpitch, host checks)
    PlaneCtx cx;
    cx.X = kp.nx; cx.ngroups = ngroups; cx.n3 = gd.ax[2].n; cx.quarter = quarter;
    cx.wband = (size_t)((kp.nsticks + QM_ZT - 1) / QM_ZT) * QM_ZT * gd.ax[2].n;   // W elements per band
    cx.A = reinterpret_cast<c128 *>(smem_raw);
    cx.scr = cx.A + (((size_t)cx.X * RP + 7) & ~(size_t)7);
    int4 *rowinfo_s = reinterpret_cast<int4 *>(cx.scr + (size_t)ngroups * TPG * SL);
    cx.rowinfo_s = rowinfo_s;
    for (int i = threadIdx.x; i < cx.X; i += blockDim.x) rowinfo_s[i] = kp.row_info[i];
    __syncthreads();
    // per-thread twiddle rows, loaded once (u is fixed for the whole kernel)
    const int u_tw = (int)(threadIdx.x % G) % C::TT;
    TwRow<C::R1> twa;
    load_twrow(twa, gd.tw[0], u_tw, C::R2);
    TwRow<C::R2> twb_store;
    if constexpr (C::R1 != C::R2) load_twrow(twb_store, gd.tw[0], u_tw, C::R1);
    const auto &twb = [&]() -> const TwRow<C::R2> & {
        if constexpr (C::R1 == C::R2) return twa; else return twb_store;
    }();
    const int n3 = cx.n3;
    // plane sequence of this CTA.  Apply / debug modes: pl = blockIdx.x, + gridDim.x, ... (pl = band * n3 + p).
    // Density mode: the CTA owns z-planes p = blockIdx.x, + gridDim.x, ... and walks ALL bands of a plane before
    // the next one, so every plane of rho is accumulated by one CTA in band order (deterministic, no atomics).
    const int nbands = nplanes / n3;
    auto plane_at = [&](int it) -> int {
        if constexpr (MODE == 3) {
            const int p = (int)blockIdx.x + (it / nbands) * (int)gridDim.x;
            return p < n3 ? (it % nbands) * n3 + p : nplanes;
        } else {
            const long long v = (long long)blockIdx.x + (long long)it * gridDim.x;
            return v < nplanes ? (int)v : nplanes;
        }
    };
    for (int it = 0, prev = -1;; ++it) {
        const int pl = plane_at(it);
        const bool have_cur = pl < nplanes;
        plane_y_phase<C, MODE>(cx, W, pl, prev, have_cur, twa, twb);
        if (!have_cur) break;
        __syncthreads();
        double sc = scale;
        if constexpr (MODE == 3) sc = scale * occ[pl / n3];
        plane_x_phase<C, MODE>(cx, kp.x_iv, gd.vt, box, box2, npair2, pl, sc, stagger_ns, rhot, twa, twb);
        __syncthreads();
        prev = pl;
    }
}
