// CUDA kernels of the pruned 3-D FFT path (sm_100a).  DESIGN.md section 6.
//   k_zinv  : a1+a2(z)  scatter sphere -> z-sticks, backward z-FFT, write stick planes  W[band][p][S]
//   k_plane : a2(y,x)+a3+a4(x,y)  per (band, z-plane): y-FFT on X rows, x-FFT 'X->N1', V multiply,
//             x-FFT 'N1->X', y-FFT, all in shared memory; reads/writes only the S stick values
//   k_zfwd  : a4(z)+a5  forward z-FFT, gather to the sphere, + 1/2|k+G|^2 psi_in
#pragma once
#include <cuda_runtime.h>
#include "fft_phases.cuh"
#include "qm_plan.h"

template <class C>
__global__ void __launch_bounds__(256)
k_zinv(QmKPlanDev kp, const c128 *__restrict__ tw, const c128 *__restrict__ psi,
       c128 *__restrict__ W, int TS)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int LP = C::L | 1;
    c128 *lines = reinterpret_cast<c128 *>(smem_raw);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int s0 = blockIdx.x * TS;
    const int ns = min(TS, kp.nsticks - s0);
    const int band = blockIdx.y;
    const int S = kp.nsticks;
    const int t = tid / C::TT, u = tid % C::TT;
    c128 *tw_s = lines + TS * LP;
    const TwTable twa{tw_s, u};

    for (int i = tid; i < C::N; i += nthr) tw_s[i] = tw[i];
    for (int i = tid; i < TS * LP; i += nthr) lines[i] = c128{0.0, 0.0};
    __syncthreads();
    const int g0 = kp.stick_off[s0], g1 = kp.stick_off[s0 + ns];
    const c128 *psib = psi + (size_t)band * kp.ng;
    for (int g = g0 + tid; g < g1; g += nthr)
        lines[(kp.g_stick[g] - s0) * LP + kp.g_zpos[g]] = psib[g];
    __syncthreads();
    if (t < ns) lineA_step1<C>(lines + t * LP, u, twa);
    __syncthreads();
    if (t < ns) lineA_step2<C>(lines + t * LP, u);
    __syncthreads();
    c128 *Wb = W + (size_t)band * C::N * S;
    for (int i = tid; i < C::N * TS; i += nthr) {
        const int p = i / TS, tt = i % TS;
        if (tt < ns) Wb[(size_t)p * S + s0 + tt] = lines[tt * LP + C::pos(p)];
    }
}

template <class C>
__global__ void __launch_bounds__(256)
k_zfwd(QmKPlanDev kp, const c128 *__restrict__ tw, const c128 *__restrict__ W,
       const c128 *__restrict__ psi_in, c128 *__restrict__ out, int TS, int kinetic)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int LP = C::L | 1;
    constexpr int GPT = 4;            // gather elements per thread kept in registers across the FFT
    c128 *lines = reinterpret_cast<c128 *>(smem_raw);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int s0 = blockIdx.x * TS;
    const int ns = min(TS, kp.nsticks - s0);
    const int band = blockIdx.y;
    const int S = kp.nsticks;
    const int t = tid / C::TT, u = tid % C::TT;
    c128 *tw_s = lines + TS * LP;
    const TwTable twb{tw_s, u};
    for (int i = tid; i < C::N; i += nthr) tw_s[i] = tw[i];

    const c128 *Wb = W + (size_t)band * C::N * S;
    for (int i = tid; i < C::N * TS; i += nthr) {
        const int p = i / TS, tt = i % TS;
        if (tt < ns) lines[tt * LP + C::pos(p)] = Wb[(size_t)p * S + s0 + tt];
    }
    // the gather's own inputs (positions, 1/2|k+G|^2 psi_in) are fetched now, behind the transform
    const int g0 = kp.stick_off[s0], g1 = kp.stick_off[s0 + ns];
    const size_t boff = (size_t)band * kp.ng;
    int gpos[GPT];
    c128 kin[GPT];
#pragma unroll
    for (int j = 0; j < GPT; ++j) {
        const int g = g0 + tid + j * nthr;
        gpos[j] = -1; kin[j] = c128{0.0, 0.0};
        if (g < g1) {
            gpos[j] = (kp.g_stick[g] - s0) * LP + kp.g_zpos[g];
            if (kinetic) {
                const c128 x = psi_in[boff + g];
                const double h = 0.5 * kp.g2[g];
                kin[j] = c128{h * x.x, h * x.y};
            }
        }
    }
    __syncthreads();
    if (t < ns) lineB_step1<C>(lines + t * LP, u, twb);
    __syncthreads();
    if (t < ns) lineB_step2<C>(lines + t * LP, u);
    __syncthreads();
#pragma unroll
    for (int j = 0; j < GPT; ++j) {
        const int g = g0 + tid + j * nthr;
        if (g < g1) out[boff + g] = lines[gpos[j]] + kin[j];
    }
    for (int g = g0 + tid + GPT * nthr; g < g1; g += nthr) {     // sticks longer than the register budget
        c128 v = lines[(kp.g_stick[g] - s0) * LP + kp.g_zpos[g]];
        if (kinetic) {
            const c128 x = psi_in[boff + g];
            const double h = 0.5 * kp.g2[g];
            v.x += h * x.x; v.y += h * x.y;
        }
        out[boff + g] = v;
    }
}

// MODE 0 apply, 1 g2r (write natural-order box), 2 r2g (read natural-order box)
//
// One CTA per (band, z-plane).  The CTA is split into independent groups of 64 threads (two warps =
// 64/TT teams of TT threads, one team per line); a group walks its own rows / columns and only
// synchronises with itself (named barrier), so the groups hide each other's latencies.  CTA-wide
// barriers remain only between the four phases (load | y backward | x round trip | y forward | store).
constexpr int QM_GROUP = 64;
#ifndef QM_PLANE_MAX_THREADS
#define QM_PLANE_MAX_THREADS 384
#endif
// Scratch lines of neighbouring teams: with 12-thread teams a quarter-warp straddles two teams as 4+4
// threads, and their unit-stride 16-byte accesses are conflict free iff the pitch is 4 (mod 8); else odd.
__host__ __device__ constexpr int qm_scratch_pitch(int len, int tt) { return tt == 12 ? len + ((12 - len % 8) % 8) : (len | 1); }
__device__ __forceinline__ void group_barrier(int grp) {
    asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "r"(QM_GROUP) : "memory");
}

template <class C, int MODE>
__global__ void __launch_bounds__(QM_PLANE_MAX_THREADS)
k_plane(QmKPlanDev kp, QmGridDev gd, c128 *__restrict__ W, c128 *__restrict__ box, int ngroups, double scale,
        int stagger_ns)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int SL = qm_scratch_pitch(C::L, C::TT);    // scratch line pitch
    constexpr int TPG = QM_GROUP / C::TT;                // teams (lines) per group
    const int X = kp.nx, rowpitch = kp.rowpitch, S = kp.nsticks;
    c128 *A = reinterpret_cast<c128 *>(smem_raw);
    c128 *scr = A + (size_t)X * rowpitch;
    int4 *rowinfo_s = reinterpret_cast<int4 *>(scr + (size_t)ngroups * TPG * SL);
    const XRows xr{kp.x_iv.x, kp.x_iv.y, kp.x_iv.z, kp.x_iv.w};
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int grp = tid / QM_GROUP, gl = tid % QM_GROUP;
    const int team = gl / C::TT, u = gl % C::TT;
    const bool team_ok = team < TPG;
    const int p = blockIdx.x, band = blockIdx.y;
    const int n3 = gd.ax[2].n;
    c128 *Wp = W + ((size_t)band * n3 + p) * S;

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
    auto row_info = [&](int r) {
        const int4 q = rowinfo_s[r];
        return RowInfo{(int)(short)(q.x & 0xffff), q.x >> 16, (int)(short)(q.y & 0xffff), q.y >> 16, q.z};
    };
    if constexpr (MODE != 2) {
        for (int rc = grp; rc * TPG < X; rc += ngroups) {
            const int r = rc * TPG + team;
            const bool ok = team_ok && r < X;
            if (ok) lineA_step1_gin<C>(A + r * rowpitch, Wp, row_info(r), u, twa);
            group_barrier(grp);
            if (ok) lineA_step2<C>(A + r * rowpitch, u);
        }
    }
    __syncthreads();
    {
        const int z = (p / gd.ax[2].r2) + gd.ax[2].r1 * (p % gd.ax[2].r2);
        c128 *myscr = scr + (size_t)(grp * TPG + team) * SL;
        const double *vplane = gd.vt + (size_t)p * C::N * C::N;
        VRow<C::R2> vr;
        // De-phase the groups: they all do identical load -> FP64 -> store bursts, and when they run in
        // lock step the shared-memory pipe and the FP64 pipe are used alternately instead of together.
        if (stagger_ns > 0) __nanosleep((unsigned)(grp * stagger_ns));
        if constexpr (MODE == 0) {       // V of the first column: in flight while step 1 runs
            const int col0 = grp * TPG + team;
            if (team_ok && col0 < C::N) load_vrow<C>(vr, vplane + (size_t)col0 * C::N, u);
        }
        for (int cc = grp; cc * TPG < C::N; cc += ngroups) {
            const int col = cc * TPG + team;
            const bool ok = team_ok && col < C::N;
            const int colpos = C::pos(col);
            if constexpr (MODE != 2) {
                if (ok) xcol_step1<C>(A, rowpitch, colpos, xr, myscr, u, twa);
                group_barrier(grp);
            }
            if (ok) {
                const int y = (col / C::R2) + C::R1 * (col % C::R2);
                c128 *bx = nullptr;
                if constexpr (MODE != 0) bx = box + (size_t)band * C::N * C::N * n3 + (size_t)y * n3 + z;
                xcol_step2<C, MODE>(myscr, u, twb, vr, bx, (long)C::N * n3, scale);
            }
            if constexpr (MODE == 0) {   // prefetch V of this team's next column behind steps 3 and 1
                const int ncol = col + ngroups * TPG;
                if (team_ok && ncol < C::N) load_vrow<C>(vr, vplane + (size_t)ncol * C::N, u);
            }
            group_barrier(grp);
            if constexpr (MODE != 1) {
                // no barrier after step 3: the scratch column a thread reads here is exactly the one it
                // overwrites in the next iteration's step 1 (MODE 2 has no step 1 and writes rows: barrier).
                if (ok) xcol_step3<C>(A, rowpitch, colpos, xr, myscr, u);
                if constexpr (MODE == 2) group_barrier(grp);
            }
        }
    }
    __syncthreads();
    if constexpr (MODE != 1) {
        for (int rc = grp; rc * TPG < X; rc += ngroups) {
            const int r = rc * TPG + team;
            const bool ok = team_ok && r < X;
            if (ok) lineB_step1<C>(A + r * rowpitch, u, twb);
            group_barrier(grp);
            if (ok) lineB_step2_gout<C>(A + r * rowpitch, Wp, row_info(r), u);
        }
    }
}
