// CUDA kernels of the pruned 3-D FFT path (sm_100a).  DESIGN.md section 6.
//   k_zinv  : a1+a2(z)  scatter sphere -> z-sticks, backward z-FFT, write stick planes  W[band][p][S]
//   k_plane : a2(y,x)+a3+a4(x,y)  per (band, z-plane): y-FFT on X rows, x-FFT 'X->N1', V multiply,
//             x-FFT 'N1->X', y-FFT, all in shared memory; reads/writes only the S stick values
//   k_zfwd  : a4(z)+a5  forward z-FFT, gather to the sphere, + 1/2|k+G|^2 psi_in
#pragma once
#include <cuda_runtime.h>
#include "fft_phases.cuh"
#include "async_copy.cuh"
#include "tmem_rows.cuh"
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
    pdl_launch_dependents();
    pdl_wait();                 // psi may come from the previous kernel; W is still read by it
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
    pdl_launch_dependents();
    if (tid == 0) {
        mbar_init(wbar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        pdl_wait();             // W comes from the previous kernel
        mbar_expect_tx(wbar, TILE_BYTES);
        bulk_g2s(stage, Wb + (size_t)blockIdx.x * C::N * QM_ZT, TILE_BYTES, wbar);
    }
    TwRow<C::R2> twb;
    load_twrow(twb, tw, u2, C::R1);
    pdl_wait();
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
#ifndef QM_PLANE_TW_TMEM
#define QM_PLANE_TW_TMEM 1      /* per-thread twiddle rows live in tensor memory (tmem_rows.cuh) instead of registers */
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
    const int4 *rowtab_s;       // [X][TT] hoisted addressing of every (row, u): Pruned with the row's first stick folded in, or nullptr
    int X, ngroups, n3, quarter;
    size_t wband;
    uint32_t tw_a, tw_b;        // TMEM addresses of this thread's twiddle rows (QM_PLANE_TW_TMEM)
};
// Branch-free lines.  The plane kernel never branches on "does this thread have a line": a thread without one (a team
// beyond the last row / column, a lane beyond the last team, a lane u >= R of a pass with fewer than TT butterflies) is
// pointed at a line nobody reads -- its team's scratch line while that is idle, else the group's sink line -- and its
// global accesses are masked off.  Idle lanes cost the same issue slots either way, and the warp stays convergent, which
// tcgen05.ld (below) needs; ptxas also spills the transform's registers around a tcgen05.ld that sits between two
// divergent regions (measured: 600-800 B of spills per thread), and not around one in straight-line code.
//
// The tail of a first pass (twiddle multiply + store).  With the rows in tensor memory the factors are brought in
// QM_TW_CHUNK at a time.  DIRB: false = backward first pass (stepA1_tail), true = forward (stepB1_tail).
#ifndef QM_TW_CHUNK
#define QM_TW_CHUNK 4
#endif
#ifndef QM_TW_PIPELINE
#define QM_TW_PIPELINE 1        /* read chunk c + 1 from tensor memory while chunk c is multiplied */
#endif
// Which line factorisations park their rows in tensor memory: those whose rows would take 44 registers or more (12 x 12: 44,
// 12 x 8: 72).  Measured per size, tensor memory against registers: 96 = 12 x 8 -20 %, 144 = 12 x 12 -5 %, 48 = 6 x 8 (48
// registers) equal, 32 = 4 x 8 (40 registers) +12 %: short rows are cheaper to keep than to fetch.
#ifndef QM_TW_TMEM_MIN_REGS
#define QM_TW_TMEM_MIN_REGS 44
#endif
template <class C> constexpr bool plane_tw_tmem =
    (QM_PLANE_TW_TMEM != 0) && (4 * (C::R1 - 1) + (C::R1 != C::R2 ? 4 * (C::R2 - 1) : 0) >= QM_TW_TMEM_MIN_REGS);

template <class C, bool DIRB, int NR, int R, class L>
__device__ __forceinline__ void plane_tail(const c128 (&t)[NR][R], const L (&dst)[NR], int u, const TwRow<R> &in_regs, uint32_t taddr)
{
  if constexpr (plane_tw_tmem<C> && QM_TW_PIPELINE) {
    // chunk c + 1 is read while chunk c is multiplied: two raw register sets, used alternately
    constexpr int NCH = (R + QM_TW_CHUNK - 1) / QM_TW_CHUNK;
    int raw[2][4][4];
    auto lo = [](int c) constexpr { return c == 0 ? 1 : c * QM_TW_CHUNK; };
    auto hi = [](int c) constexpr { return (c + 1) * QM_TW_CHUNK < R ? (c + 1) * QM_TW_CHUNK : R; };
    if constexpr (lo(0) < hi(0)) tmem_issue<hi(0) - lo(0)>(raw[0], taddr + 4 * lo(0));
    static_for<NCH>([&](auto I) {
        constexpr int c = decltype(I)::value;
        constexpr int j0 = c * QM_TW_CHUNK, j1 = hi(c), l0 = lo(c);
        TwChunk<l0, (l0 < j1 ? j1 : l0 + 1)> ch;
        if constexpr (l0 < j1) tmem_land(ch, raw[c & 1]);
        if constexpr (c + 1 < NCH) tmem_issue<hi(c + 1) - lo(c + 1)>(raw[(c + 1) & 1], taddr + 4 * lo(c + 1));
        static_for<NR>([&](auto II) {
            constexpr int i = decltype(II)::value;
            if constexpr (DIRB) stepB1_tail_range<C, j0, j1, false>(t[i], dst[i], u, ch);
            else stepA1_tail_range<C, j0, j1, false>(t[i], dst[i], u, ch);
        });
    });
  } else if constexpr (plane_tw_tmem<C>) {
    static_for<(R + QM_TW_CHUNK - 1) / QM_TW_CHUNK>([&](auto I) {
        constexpr int j0 = decltype(I)::value * QM_TW_CHUNK, j1 = j0 + QM_TW_CHUNK < R ? j0 + QM_TW_CHUNK : R;
        constexpr int l0 = j0 == 0 ? 1 : j0;            // factor 0 is 1 and is not stored
        TwChunk<l0, (l0 < j1 ? j1 : l0 + 1)> ch;
        if constexpr (l0 < j1) tmem_load_chunk(ch, taddr);        static_for<NR>([&](auto II) {
            constexpr int i = decltype(II)::value;
            if constexpr (DIRB) stepB1_tail_range<C, j0, j1, false>(t[i], dst[i], u, ch);
            else stepA1_tail_range<C, j0, j1, false>(t[i], dst[i], u, ch);
        });
    });
  } else {
    static_for<NR>([&](auto II) {
        constexpr int i = decltype(II)::value;
        if constexpr (DIRB) stepB1_tail_range<C, 0, R, false>(t[i], dst[i], u, in_regs);
        else stepA1_tail_range<C, 0, R, false>(t[i], dst[i], u, in_regs);
    });
  }
}
// Scratch lines: one per team, plus one sink line per group (behind the group's team lines) when some lane of a group
// can be without work in a pass (R1 != R2, or G not a multiple of TT).
template <class C> struct PlaneGeom {
    static constexpr int G = QM_GROUP, TPG = G / C::TT;
    static constexpr bool SINK = (C::R1 != C::R2) || (G % C::TT != 0);
    static constexpr int LPG = TPG + (SINK ? 1 : 0);     // scratch lines per group
};
template <class C> struct PlaneIds {
    static constexpr int G = QM_GROUP, TPG = G / C::TT;
    int grp, team, u, slot; bool team_ok;
    int u1, u2;           // u clamped for passes with R1 / R2 butterflies per line
    bool a1, a2;          // this lane has a butterfly in such a pass
    int scr_line, sink_line;
    __device__ PlaneIds() {
        const int tid = threadIdx.x, gl = tid % G;
        grp = tid / G; team = gl / C::TT; u = gl % C::TT;
        team_ok = team < TPG;
        slot = qm_team_slot<C::TT, TPG>(team);
        a1 = team_ok && u < C::R1; a2 = team_ok && u < C::R2;
        u1 = u < C::R1 ? u : 0; u2 = u < C::R2 ? u : 0;
        sink_line = grp * PlaneGeom<C>::LPG + (PlaneGeom<C>::SINK ? TPG : 0);
        scr_line = grp * PlaneGeom<C>::LPG + (team_ok ? team : TPG);
    }
};

template <class C, int MODE>
__device__ __forceinline__ void plane_y_phase(const PlaneCtx cx, c128 *__restrict__ W, int pl, int prev, bool have_cur,
                                              const TwRow<C::R1> &twa, const TwRow<C::R2> &twb)
{
    constexpr int G = QM_GROUP, TPG = G / C::TT, RP = C::L | 1, NPRE = 2 * Quarter<C>::Q;
    constexpr int SL = qm_scratch_pitch(C::L, C::TT);
    constexpr bool HAS_BACK = MODE != 2, HAS_FWD = MODE != 1 && MODE != 3;
    const PlaneIds<C> id;
    const int grp = id.grp, slot = id.slot, X = cx.X, n3 = cx.n3, quarter = cx.quarter & 1;
    const bool do_back = HAS_BACK && have_cur, do_fwd = HAS_FWD && prev >= 0;
    if (!(do_back || do_fwd)) return;
    const SLine As = qm_sline(cx.A);
    // where a lane without work reads and writes: the scratch lines are idle during the y phase
    const SLine junk = qm_sline(cx.scr + (size_t)id.scr_line * SL);
    const int pc = have_cur ? pl : 0, pp = prev >= 0 ? prev : 0;
    const WView Wcur = qm_wview(W + (size_t)(pc / n3) * cx.wband, pc % n3, n3);
    const WView Wprev = qm_wview(W + (size_t)(pp / n3) * cx.wband, pp % n3, n3);
    // A team works on NR rows per round (rows r, r + rstride, ...).  NR = 1: two rows per round spill at the register
    // budget of this kernel and were measured slower; the helpers below take row arrays.
    constexpr int NR = 1;
    const int rstride = cx.ngroups * TPG;
    for (int r0 = grp * TPG + slot; r0 - slot < X; r0 += NR * rstride) {      // same trip count for a whole group
        int sbase[NR];
        Pruned pr[NR];
        c128 pre[NR][NPRE];
        SLine row1[NR], row2[NR];          // the row as seen by passes with R1 / R2 butterflies
#pragma unroll
        for (int i = 0; i < NR; ++i) {
            const int r = r0 + i * rstride;
            const bool ok = id.team_ok && r < X;
            if (cx.rowtab_s) {
                const int4 e = cx.rowtab_s[(ok ? r : 0) * C::TT + id.u];
                sbase[i] = 0;
                pr[i] = Pruned{(unsigned)e.x, (unsigned)e.y, e.z, e.w};
                if (!ok) pr[i].m1 = pr[i].m2 = 0u;
            } else {
                const int4 q = cx.rowinfo_s[ok ? r : 0];
                sbase[i] = q.z;
                pr[i] = make_pruned_packed<C>(q.x, q.y, id.u2, 1);
                if (!(ok && id.a2)) pr[i].m1 = pr[i].m2 = 0u;          // no global access at all
            }
            row1[i] = (ok && id.a1) ? As + r * RP : junk;
            row2[i] = (ok && id.a2) ? As + r * RP : junk;
            if (do_back && quarter) prefetch_quarter<C>(Wcur + sbase[i], C::R2, pr[i], pre[i]);
        }
        if (do_fwd) {
            c128 t[NR][C::R2];
#pragma unroll
            for (int i = 0; i < NR; ++i) lineB_step1_head<C, false>(row1[i], id.u1, t[i]);
            plane_tail<C, true>(t, row1, id.u1, twb, cx.tw_b);
            group_barrier<G>(grp);
#pragma unroll
            for (int i = 0; i < NR; ++i) {
                if (quarter) prunedB_step2_quarter<C, false>(row2[i], Wprev + sbase[i], C::R2, pr[i], id.u2);
                else prunedB_step2<C, false>(row2[i], Wprev + sbase[i], C::R2, pr[i], id.u2);
            }
        }
        // the team that read the row in the step above is the one that refills it: no barrier needed
        if (do_back) {
            c128 t[NR][C::R1];
#pragma unroll
            for (int i = 0; i < NR; ++i) {
                if (quarter) prunedA_step1_pre_head<C, false>(pre[i], t[i], id.u2);
                else prunedA_step1_head<C, false>(Wcur + sbase[i], C::R2, pr[i], t[i], id.u2);
            }
            plane_tail<C, false>(t, row2, id.u2, twa, cx.tw_a);
            group_barrier<G>(grp);
#pragma unroll
            for (int i = 0; i < NR; ++i) lineA_step2<C, false>(row1[i], id.u1);
        }
    }
}

template <class C, int MODE>
__device__ __forceinline__ void plane_x_phase(const PlaneCtx cx, const short4 x_iv, const double *__restrict__ vt,
                                           c128 *__restrict__ box, const c128 *__restrict__ box2, int npair2, int pl,
                                           double scale,
                                           double *__restrict__ rhot, const TwRow<C::R1> &twa, const TwRow<C::R2> &twb)
{
    constexpr int G = QM_GROUP, TPG = G / C::TT, RP = C::L | 1;
    constexpr int SL = qm_scratch_pitch(C::L, C::TT);    // scratch line pitch
    const PlaneIds<C> id;
    const int grp = id.grp, slot = id.slot, n3 = cx.n3, nteams = cx.ngroups * TPG;
    const bool xq = (cx.quarter & 2) != 0;               // quarter rule holds for the x rows: 2Q loads / stores per column
    const SLine As = qm_sline(cx.A);
    const Pruned px = make_pruned<C>(x_iv.x, x_iv.y, x_iv.z, x_iv.w, id.u2, RP);
    const Pruned pnone = Pruned{0u, 0u, 0, 0};
    const int band = pl / n3, p = pl - band * n3;
    // a team's scratch line; lanes beyond the last team and lanes without a butterfly in a pass use the group's sink line
    const SLine sink = qm_sline(cx.scr + (size_t)id.sink_line * SL);
    const SLine teamscr = qm_sline(cx.scr + (size_t)id.scr_line * SL);
    const SLine scrA[1] = {id.a2 ? teamscr : sink}, scrB[1] = {id.a1 ? teamscr : sink};
    const double *vplane = vt + (size_t)p * C::N * VLayout<C>::COL;
    VRow<C::R2> vr;
    const int col0 = grp * TPG + slot;
    auto vcol = [&](int c) { return vplane + (size_t)(c < C::N ? c : C::N - 1) * VLayout<C>::COL; };
    if constexpr (MODE == 0) load_vrow<C>(vr, vcol(col0), id.u1);       // V of the first column: in flight while step 1 runs
    for (int col = col0; col - slot < C::N; col += nteams) {      // same trip count for a whole group
        const bool ok = id.team_ok && col < C::N;
        const int colc = col < C::N ? col : C::N - 1;    // a column that exists, for the addresses of lanes without one
        const SLine Acol = As + C::pos(col);
        const Pruned pxc = (ok && id.a2) ? px : pnone;   // plane-array accesses of a lane without work are masked off
        if constexpr (MODE != 2) {
            c128 t[1][C::R1];
            if (xq) {
                c128 pre[2 * Quarter<C>::Q];
                prefetch_quarter<C>(Acol, C::R2 * RP, pxc, pre);
                prunedA_step1_pre_head<C, false>(pre, t[0], id.u2);
            } else prunedA_step1_head<C, false>(Acol, C::R2 * RP, pxc, t[0], id.u2);
            plane_tail<C, false>(t, scrA, id.u2, twa, cx.tw_a);
            group_barrier<G>(grp);
        }
        if constexpr (MODE == 3) {
            // scale = weight * occupation of this band; rhot = running density of this plane in the V layout
            if (ok) xcol_density<C>(teamscr, id.u, rhot + ((size_t)p * C::N + col) * VLayout<C>::COL, scale);
        } else {
            // transposed boxes (fft_phases.cuh BoxT): column (p, col) of state `band`; with a second operand the plane
            // index counts pairs: band = a * npair2 + b, first operand state a, second operand state b (MODE 2)
            c128 *bx = nullptr;
            const c128 *bx2 = nullptr;
            const size_t coloff = ((size_t)p * C::N + colc) * C::N, boxsz = (size_t)C::N * C::N * n3;
            if constexpr (MODE == 1) bx = box + (size_t)band * boxsz + coloff;
            if constexpr (MODE == 2) {
                bx = box + (size_t)(npair2 > 0 ? band / npair2 : band) * boxsz + coloff;
                if (npair2 > 0) bx2 = box2 + (size_t)(band % npair2) * boxsz + coloff;
            }
            if constexpr (MODE == 4) bx2 = box2 + coloff;
            c128 t[1][C::R2];
            xcol_step2_head<C, MODE, false>(scrB[0], id.u1, vr, bx, bx2, scale, t[0], ok && id.a1);
            if constexpr (MODE != 1) plane_tail<C, true>(t, scrB, id.u1, twb, cx.tw_b);
        }
        if constexpr (MODE == 0)     // prefetch V of this team's next column behind steps 3 and 1
            load_vrow<C>(vr, vcol(col + nteams), id.u1);
        group_barrier<G>(grp);
        if constexpr (MODE != 1 && MODE != 3) {
            // no barrier after step 3: the scratch column a thread reads here is exactly the one it
            // overwrites in the next iteration's step 1 (MODE 2 has no step 1 and writes rows: barrier).
            if (xq) prunedB_step2_quarter<C, false>(scrA[0], Acol, C::R2 * RP, pxc, id.u2);
            else prunedB_step2<C, false>(scrA[0], Acol, C::R2 * RP, pxc, id.u2);
            if constexpr (MODE == 2) group_barrier<G>(grp);
        }
    }
}

template <class C, int MODE>
__global__ void __launch_bounds__(QM_PLANE_MAX_THREADS)
k_plane(QmKPlanDev kp, QmGridDev gd, c128 *__restrict__ W, c128 *__restrict__ box, const c128 *__restrict__ box2,
        int npair2, int ngroups, double scale, int nplanes, int quarter, const double *__restrict__ occ,
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
    int4 *rowinfo_s = reinterpret_cast<int4 *>(cx.scr + (size_t)ngroups * PlaneGeom<C>::LPG * SL);
    cx.rowinfo_s = rowinfo_s;
    for (int i = threadIdx.x; i < cx.X; i += blockDim.x) rowinfo_s[i] = kp.row_info[i];
    // (quarter & 4): room for the hoisted y addressing of every (row, u), worked out once per kernel
    int4 *rowtab_s = rowinfo_s + cx.X + 1;                 // one int4 in between holds the tensor-memory base address
    cx.rowtab_s = (quarter & 4) ? rowtab_s : nullptr;
    if (quarter & 4) {
        for (int i = threadIdx.x; i < cx.X * C::TT; i += blockDim.x) {
            const int r = i / C::TT, uu = i % C::TT;
            const int4 q = kp.row_info[r];
            Pruned pr = make_pruned_packed<C>(q.x, q.y, uu < C::R2 ? uu : 0, 1);
            if (uu >= C::R2) pr.m1 = pr.m2 = 0u;
            rowtab_s[i] = int4{(int)pr.m1, (int)pr.m2, pr.c1 + q.z, pr.c2 + q.z};
        }
    }
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
    cx.tw_a = cx.tw_b = 0;
    uint32_t tmem_base = 0, tmem_cols = 0;
    if constexpr (plane_tw_tmem<C>) {
        // ... and parked in tensor memory: 4 columns per factor in the warp's lane window, one column range per warp of an
        // SM sub-partition (warps w, w+4, w+8, ... share a lane window)
        constexpr int ROWCOLS = 4 * C::R1 + (C::R1 != C::R2 ? 4 * C::R2 : 0);
        uint32_t &tmem_base_s = *reinterpret_cast<uint32_t *>(rowinfo_s + cx.X);      // the 16 bytes behind the row table
        tmem_cols = (uint32_t)qm_tmem_cols_pow2(ROWCOLS * (int)((blockDim.x / 32 + 3) / 4));
        if (threadIdx.x < 32) tmem_alloc(&tmem_base_s, tmem_cols);
        tmem_fence_before_sync();
        __syncthreads();
        tmem_fence_after_sync();
        tmem_base = tmem_base_s;
        cx.tw_a = tmem_warp_addr(tmem_base, 0, ROWCOLS);
        cx.tw_b = C::R1 != C::R2 ? cx.tw_a + 4 * C::R1 : cx.tw_a;
        tmem_store_row(cx.tw_a, twa);
        if constexpr (C::R1 != C::R2) tmem_store_row(cx.tw_b, twb_store);
        tmem_wait_st();
    }
    pdl_launch_dependents();
    pdl_wait();                 // the stick planes (and boxes) come from the previous kernel
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
        plane_x_phase<C, MODE>(cx, kp.x_iv, gd.vt, box, box2, npair2, pl, sc, rhot, twa, twb);
        __syncthreads();
        prev = pl;
    }
    if constexpr (plane_tw_tmem<C>) {
        tmem_fence_before_sync();
        __syncthreads();
        if (threadIdx.x < 32) tmem_dealloc(tmem_base, tmem_cols);
    }
}
