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
    c128 *tw_s = reinterpret_cast<c128 *>(smem_raw);
    c128 *lines = tw_s + C::N;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int s0 = blockIdx.x * TS;
    const int ns = min(TS, kp.nsticks - s0);
    const int band = blockIdx.y;
    const int S = kp.nsticks;

    for (int i = tid; i < C::N; i += nthr) tw_s[i] = tw[i];
    for (int i = tid; i < TS * LP; i += nthr) lines[i] = c128{0.0, 0.0};
    __syncthreads();
    const int g0 = kp.stick_off[s0], g1 = kp.stick_off[s0 + ns];
    const c128 *psib = psi + (size_t)band * kp.ng;
    for (int g = g0 + tid; g < g1; g += nthr)
        lines[(kp.g_stick[g] - s0) * LP + kp.g_zpos[g]] = psib[g];
    __syncthreads();
    const int t = tid / C::TT, u = tid % C::TT;
    if (t < ns) lineA_step1<C>(lines + t * LP, u, tw_s);
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
    c128 *tw_s = reinterpret_cast<c128 *>(smem_raw);
    c128 *lines = tw_s + C::N;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int s0 = blockIdx.x * TS;
    const int ns = min(TS, kp.nsticks - s0);
    const int band = blockIdx.y;
    const int S = kp.nsticks;

    for (int i = tid; i < C::N; i += nthr) tw_s[i] = tw[i];
    const c128 *Wb = W + (size_t)band * C::N * S;
    for (int i = tid; i < C::N * TS; i += nthr) {
        const int p = i / TS, tt = i % TS;
        if (tt < ns) lines[tt * LP + C::pos(p)] = Wb[(size_t)p * S + s0 + tt];
    }
    __syncthreads();
    const int t = tid / C::TT, u = tid % C::TT;
    if (t < ns) lineB_step1<C>(lines + t * LP, u, tw_s);
    __syncthreads();
    if (t < ns) lineB_step2<C>(lines + t * LP, u);
    __syncthreads();
    const int g0 = kp.stick_off[s0], g1 = kp.stick_off[s0 + ns];
    const size_t boff = (size_t)band * kp.ng;
    for (int g = g0 + tid; g < g1; g += nthr) {
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
template <class C, int MODE>
__global__ void __launch_bounds__(512)
k_plane(QmKPlanDev kp, QmGridDev gd, c128 *__restrict__ W, c128 *__restrict__ box, int ncol, double scale)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int SL = C::L | 1;                         // scratch line pitch
    const int X = kp.nx, rowpitch = kp.rowpitch, S = kp.nsticks;
    c128 *tw_s = reinterpret_cast<c128 *>(smem_raw);
    c128 *A = tw_s + C::N;
    c128 *scr = A + (size_t)X * rowpitch;
    short *xrow_s = reinterpret_cast<short *>(scr + (size_t)ncol * SL);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int p = blockIdx.x, band = blockIdx.y;
    const int n3 = gd.ax[2].n;
    c128 *Wp = W + ((size_t)band * n3 + p) * S;

    for (int i = tid; i < C::N; i += nthr) { tw_s[i] = gd.tw[0][i]; xrow_s[i] = kp.xrow[i]; }
    if constexpr (MODE != 2) {
        for (int i = tid; i < X * rowpitch; i += nthr) A[i] = c128{0.0, 0.0};
        __syncthreads();
        for (int s = tid; s < S; s += nthr) A[kp.stick_apos[s]] = Wp[s];
        __syncthreads();
        for (int base = 0; base < X * C::TT; base += nthr) {
            const int task = base + tid;
            if (task < X * C::TT) lineA_step1<C>(A + (task / C::TT) * rowpitch, task % C::TT, tw_s);
        }
        __syncthreads();
        for (int base = 0; base < X * C::TT; base += nthr) {
            const int task = base + tid;
            if (task < X * C::TT) lineA_step2<C>(A + (task / C::TT) * rowpitch, task % C::TT);
        }
    }
    __syncthreads();
    {
        const int c = tid / C::TT, u = tid % C::TT;
        const int z = (p / gd.ax[2].r2) + gd.ax[2].r1 * (p % gd.ax[2].r2);
        c128 *myscr = scr + (size_t)c * SL;
        for (int cbase = 0; cbase < C::N; cbase += ncol) {
            const int col = cbase + c;
            const bool active = (c < ncol) && (col < C::N);
            const int colpos = C::pos(col);
            if constexpr (MODE != 2) {
                if (active) xcol_step1<C>(A, rowpitch, colpos, xrow_s, myscr, u, tw_s);
                __syncthreads();
            }
            if (active) {
                const int y = (col / C::R2) + C::R1 * (col % C::R2);
                const double *v = nullptr;
                c128 *bx = nullptr;
                if constexpr (MODE == 0) v = gd.vt + ((size_t)p * C::N + col) * C::N;
                else bx = box + (size_t)band * C::N * C::N * n3 + (size_t)y * n3 + z;
                xcol_step2<C, MODE>(myscr, u, tw_s, v, bx, (long)C::N * n3, scale);
            }
            __syncthreads();
            if constexpr (MODE != 1) {
                if (active) xcol_step3<C>(A, rowpitch, colpos, xrow_s, myscr, u);
                __syncthreads();
            }
        }
    }
    if constexpr (MODE != 1) {
        for (int base = 0; base < X * C::TT; base += nthr) {
            const int task = base + tid;
            if (task < X * C::TT) lineB_step1<C>(A + (task / C::TT) * rowpitch, task % C::TT, tw_s);
        }
        __syncthreads();
        for (int base = 0; base < X * C::TT; base += nthr) {
            const int task = base + tid;
            if (task < X * C::TT) lineB_step2<C>(A + (task / C::TT) * rowpitch, task % C::TT);
        }
        __syncthreads();
        for (int s = tid; s < S; s += nthr) Wp[s] = A[kp.stick_apos[s]];
    }
}
