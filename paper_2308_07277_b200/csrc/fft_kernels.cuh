// CUDA kernels of the pruned 3-D FFT path (sm_100a).  DESIGN.md section 6.
//   k_zinv  : a1+a2(z)  scatter sphere -> z-sticks, backward z-FFT, write stick planes  W[band][p][S]
//   k_plane : a2(y,x)+a3+a4(x,y)  per (band, z-plane): y-FFT on X rows, x-FFT 'X->N1', V multiply,
//             x-FFT 'N1->X', y-FFT, all in shared memory; reads/writes only the S stick values
//   k_zfwd  : a4(z)+a5  forward z-FFT, gather to the sphere, + 1/2|k+G|^2 psi_in
#pragma once
#include <cuda_runtime.h>
#include <cstdio>
#include "fft_phases.cuh"
#include "async_copy.cuh"
#include "qm_plan.h"

// z kernels.  A CTA owns tiles of QM_ZT adjacent sticks of one band (looping over tiles gridDim.x apart, so
// the per-thread twiddle row is loaded once).  Both kernels are global -> registers -> first radix pass ->
// shared memory -> second radix pass -> registers -> global: one shared-memory round trip, no zero fill, no
// table-driven scatter (the G of a stick are two contiguous index runs, Pruned).  Thread mapping is
// (stick, u) with u fastest where the sphere side is touched (contiguous psi runs) and (u, stick) with the
// stick fastest where the stick planes W[p][S] are touched (contiguous 256-byte segments).
constexpr int QM_ZT = 16;
template <class C> __host__ __device__ constexpr int qm_z_threads() { return QM_ZT * C::TT; }

template <class C>
__global__ void __launch_bounds__(QM_ZT * C::TT, 3)
k_zinv(QmKPlanDev kp, const c128 *__restrict__ tw, const c128 *__restrict__ psi, c128 *__restrict__ W, int ntiles)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int LP = C::L | 1;
    c128 *lines = reinterpret_cast<c128 *>(smem_raw);
    const int tid = threadIdx.x;
    const int S = kp.nsticks, band = blockIdx.y;
    const int t1 = tid / C::TT, u1 = tid % C::TT;      // pass 1: u fastest
    const int t2 = tid % QM_ZT, u2 = tid / QM_ZT;      // pass 2: stick fastest
    TwRow<C::R1> twa;
    load_twrow(twa, tw, u1, C::R2);
    const c128 *psib = psi + (size_t)band * kp.ng;
    c128 *Wb = W + (size_t)band * C::N * S;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int s0 = tile * QM_ZT;
        const int ns = min(QM_ZT, S - s0);
        if (t1 < ns) {
            const int4 q = kp.stick_info[s0 + t1];
            const Pruned pr = make_pruned<C>((int)(short)(q.x & 0xffff), q.x >> 16, (int)(short)(q.y & 0xffff), q.y >> 16, u1, 1);
            prunedA_step1<C>(SpaceGlobal{}, psib + q.z, C::R2, pr, lines + t1 * LP, u1, twa);
        }
        __syncthreads();
        if (t2 < ns) zinv_step2_store<C>(lines + t2 * LP, Wb + s0 + t2, S, u2);
        __syncthreads();
    }
}

template <class C>
__global__ void __launch_bounds__(QM_ZT * C::TT, 3)
k_zfwd(QmKPlanDev kp, const c128 *__restrict__ tw, const c128 *__restrict__ W,
       const c128 *__restrict__ psi_in, c128 *__restrict__ out, int ntiles, int kinetic)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int LP = C::L | 1;
    c128 *lines = reinterpret_cast<c128 *>(smem_raw);
    const int tid = threadIdx.x;
    const int S = kp.nsticks, band = blockIdx.y;
    const int t1 = tid / C::TT, u1 = tid % C::TT;      // pass 2 (gather side): u fastest
    const int t2 = tid % QM_ZT, u2 = tid / QM_ZT;      // pass 1 (stick-plane side): stick fastest
    TwRow<C::R2> twb;
    load_twrow(twb, tw, u2, C::R1);
    const c128 *Wb = W + (size_t)band * C::N * S;
    const size_t boff = (size_t)band * kp.ng;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int s0 = tile * QM_ZT;
        const int ns = min(QM_ZT, S - s0);
        if (t2 < ns) zfwd_step1_load<C>(Wb + s0 + t2, S, lines + t2 * LP, u2, twb);
        __syncthreads();
        if (t1 < ns) {
            const int4 q = kp.stick_info[s0 + t1];
            const Pruned pr = make_pruned<C>((int)(short)(q.x & 0xffff), q.x >> 16, (int)(short)(q.y & 0xffff), q.y >> 16, u1, 1);
            zfwd_step2_gather<C>(lines + t1 * LP, out + boff + q.z, kinetic ? psi_in + boff + q.z : nullptr, kp.g2 + q.z, pr, u1,
                                 kinetic != 0);
        }
        __syncthreads();
    }
}

// MODE 0 apply, 1 g2r (write natural-order box), 2 r2g (read natural-order box)
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
#ifdef QM_ABLATE_GBAR     /* timing experiment only: results are wrong */
    return;
#endif
    if constexpr (G == 32) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "r"(G) : "memory");
}

// Persistent: a CTA walks the (band, z-plane) pairs pl = blockIdx.x, blockIdx.x + gridDim.x, ...  Between two x phases
// the y-forward pass of the plane just finished and the y-backward pass of the next plane run as ONE loop over
// row chunks (a row of the plane array is consumed and refilled by the same team), so there are two CTA-wide
// barriers per plane.  The next plane's stick values of a row are fetched into registers (quarter rule,
// prefetch_quarter) before the y-forward work of that row starts, which hides their latency.
template <class C, int MODE>
__global__ void __launch_bounds__(QM_PLANE_MAX_THREADS)
k_plane(QmKPlanDev kp, QmGridDev gd, c128 *__restrict__ W, c128 *__restrict__ box, int ngroups, double scale,
        int stagger_ns, int nplanes, int quarter)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int G = QM_GROUP;
    constexpr int SL = qm_scratch_pitch(C::L, C::TT);    // scratch line pitch
    constexpr int TPG = G / C::TT;                       // teams (lines) per group
    constexpr int RP = C::L | 1;                         // plane row pitch (== kp.rowpitch, host checks)
    constexpr int NPRE = 2 * Quarter<C>::Q;
    constexpr bool HAS_BACK = MODE != 2, HAS_FWD = MODE != 1;
    const int X = kp.nx, S = kp.nsticks;
    c128 *A = reinterpret_cast<c128 *>(smem_raw);
    c128 *scr = A + (((size_t)X * RP + 7) & ~(size_t)7);
    int4 *rowinfo_s = reinterpret_cast<int4 *>(scr + (size_t)ngroups * TPG * SL);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int grp = tid / G, gl = tid % G;
    const int team = gl / C::TT, u = gl % C::TT;
    const bool team_ok = team < TPG;
    const int slot = qm_team_slot<C::TT, TPG>(team);     // line of the group's chunk this team works on
    const int n3 = gd.ax[2].n;

    // per-thread twiddle rows (u is fixed for the whole kernel)
    TwRow<C::R1> twa;
    load_twrow(twa, gd.tw[0], u, C::R2);
    TwRow<C::R2> twb_store;
    if constexpr (C::R1 != C::R2) load_twrow(twb_store, gd.tw[0], u, C::R1);
    const auto &twb = [&]() -> const TwRow<C::R2> & {
        if constexpr (C::R1 == C::R2) return twa; else return twb_store;
    }();

    for (int i = tid; i < X; i += nthr) rowinfo_s[i] = kp.row_info[i];
    __syncthreads();
    auto row_pruned = [&](int r, int &sbase) {
        const int4 q = rowinfo_s[r];
        sbase = q.z;
        return make_pruned<C>((int)(short)(q.x & 0xffff), q.x >> 16, (int)(short)(q.y & 0xffff), q.y >> 16, u, 1);
    };
#ifdef QM_PLANE_TIMING
    long long tacc[3] = {0, 0, 0}, t0 = clock64(), t1;
#define QM_TICK(i) do { t1 = clock64(); tacc[i] += t1 - t0; t0 = t1; } while (0)
#else
#define QM_TICK(i) do {} while (0)
#endif
    const int row0 = grp * TPG + slot, rstride = ngroups * TPG;
    for (int pl = blockIdx.x, prev = -1;; prev = pl, pl += gridDim.x) {
        const bool have_cur = pl < nplanes;
        const bool do_back = HAS_BACK && have_cur, do_fwd = HAS_FWD && prev >= 0;
        // ---- merged y phase: y-forward of plane `prev`, y-backward of plane `pl`, row chunk by row chunk ----
        if (do_back || do_fwd) {
            const c128 *Wcur = W + (size_t)(have_cur ? pl : 0) * S;
            c128 *Wprev = W + (size_t)(prev >= 0 ? prev : 0) * S;
            for (int r = row0; r - slot < X; r += rstride) {
                const bool ok = team_ok && r < X;
                int sbase = 0;
                Pruned pr{0u, 0u, 0, 0};
                if (ok) pr = row_pruned(r, sbase);
                c128 pre[NPRE];
                if (do_back && quarter && ok) prefetch_quarter<C>(SpaceGlobal{}, Wcur + sbase, C::R2, pr, pre);
                if (do_fwd) {
                    if (ok) lineB_step1<C>(A + r * RP, u, twb);
                    group_barrier<G>(grp);
                    if (ok) prunedB_step2<C>(SpaceGlobal{}, A + r * RP, Wprev + sbase, C::R2, pr, u);
                }
                if (do_back) {
                    // the team that read row r in the step above is the one that refills it: no barrier needed
                    if (ok) {
                        if (quarter) prunedA_step1_pre<C>(pre, A + r * RP, u, twa);
                        else prunedA_step1<C>(SpaceGlobal{}, Wcur + sbase, C::R2, pr, A + r * RP, u, twa);
                    }
                    group_barrier<G>(grp);
                    if (ok) lineA_step2<C>(A + r * RP, u);
                }
            }
        }
        if (!have_cur) break;
        __syncthreads();
        QM_TICK(0);
        // ---- x phase of plane `pl` ----
        {
            // (re)derived per plane on purpose: keeping it live through the y phase costs registers there
            const Pruned px = make_pruned<C>(kp.x_iv.x, kp.x_iv.y, kp.x_iv.z, kp.x_iv.w, u, RP);
            const int band = pl / n3, p = pl - band * n3;
            const int z = (p / gd.ax[2].r2) + gd.ax[2].r1 * (p % gd.ax[2].r2);
            c128 *myscr = scr + (size_t)(grp * TPG + team) * SL;
            const double *vplane = gd.vt + (size_t)p * C::N * VLayout<C>::COL;
            VRow<C::R2> vr;
            // De-phase the groups: they all do identical load -> FP64 -> store bursts, and when they run in
            // lock step the shared-memory pipe and the FP64 pipe are used alternately instead of together.
            if (stagger_ns > 0) __nanosleep((unsigned)(grp * stagger_ns));
            const int col0 = grp * TPG + slot;
            if constexpr (MODE == 0) {       // V of the first column: in flight while step 1 runs
                if (team_ok && col0 < C::N) load_vrow<C>(vr, vplane + (size_t)col0 * VLayout<C>::COL, u);
            }
            for (int col = col0; col - slot < C::N; col += ngroups * TPG) {
                const bool ok = team_ok && col < C::N;
                c128 *Acol = A + C::pos(col);
                if constexpr (MODE != 2) {
                    if (ok) prunedA_step1<C>(SpaceShared{}, Acol, C::R2 * RP, px, myscr, u, twa);
                    group_barrier<G>(grp);
                }
                if (ok) {
                    const int y = (col / C::R2) + C::R1 * (col % C::R2);
                    c128 *bx = nullptr;
                    if constexpr (MODE != 0) bx = box + (size_t)band * C::N * C::N * n3 + (size_t)y * n3 + z;
                    xcol_step2<C, MODE>(myscr, u, twb, vr, bx, (long)C::N * n3, scale);
                }
                if constexpr (MODE == 0) {   // prefetch V of this team's next column behind steps 3 and 1
                    const int ncol = col + ngroups * TPG;
                    if (team_ok && ncol < C::N) load_vrow<C>(vr, vplane + (size_t)ncol * VLayout<C>::COL, u);
                }
                group_barrier<G>(grp);
                if constexpr (MODE != 1) {
                    // no barrier after step 3: the scratch column a thread reads here is exactly the one it
                    // overwrites in the next iteration's step 1 (MODE 2 has no step 1 and writes rows: barrier).
                    if (ok) prunedB_step2<C>(SpaceShared{}, myscr, Acol, C::R2 * RP, px, u);
                    if constexpr (MODE == 2) group_barrier<G>(grp);
                }
            }
        }
        __syncthreads();
        QM_TICK(1);
    }
#ifdef QM_PLANE_TIMING
    QM_TICK(2);
    if (tid == 0 && (blockIdx.x == 0 || blockIdx.x == 77 || blockIdx.x == 147))
        printf("cta %d clk: y %lld x %lld tail %lld\n", blockIdx.x, tacc[0], tacc[1], tacc[2]);
#endif
}
