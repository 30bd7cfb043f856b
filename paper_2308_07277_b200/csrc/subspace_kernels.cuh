// Subspace products on the FP64 tensor cores (DMMA m8n8k4), sm_100a.
//   S[i][j] = <a_i|b_j> = sum_G conj(a_i(G)) b_j(G)        PAPER.md:767 (WavefunG.vdot as ZGEMM), 1034 (Davidson)
// a: [na][ng], b: [nb][ng] row-major complex128 (the caller's wavefunction blocks, untouched), S: [na][nb].
// A CTA owns a 64 x 64 tile of S and a contiguous range of K (split-K over the sphere so that every SM has
// work whatever na, nb are); one producer warp streams 32-wide K slices of the 64 + 64 rows into a 3-stage
// shared-memory ring with bulk asynchronous row copies (mbarrier complete_tx), 8 consumer warps issue DMMA.
// Complex products by the 3M scheme as in the projector GEMMs.  Split partials are summed in a fixed order
// by k_sub_reduce (deterministic, no atomics).
#pragma once
#include <cuda_runtime.h>
#include "fft_reg.cuh"
#include "async_copy.cuh"
#include "proj_kernels.cuh"     // dmma884

#ifndef QM_SG_KS
#define QM_SG_KS 32      /* K slice per stage: 512-byte row copies; 256-byte ones are bulk-copy issue bound (2x slower) */
#endif
#ifndef QM_SG_ST
#define QM_SG_ST 3
#endif
constexpr int SG_T = 64, SG_KS = QM_SG_KS, SG_PITCH = SG_KS + 4, SG_ST = QM_SG_ST, SG_CW = 8;
constexpr int SG_ROW_BYTES = SG_PITCH * 16;                          // rows 4 (mod 8) sixteen-byte words apart
constexpr int SG_STAGE_BYTES = 2 * SG_T * SG_ROW_BYTES;
constexpr int SG_SMEM = SG_ST * SG_STAGE_BYTES + 2 * SG_ST * 8 + 16;

__global__ void __launch_bounds__((SG_CW + 1) * 32, 1)
k_sub_gemm(const c128 *__restrict__ a, int na, const c128 *__restrict__ b, int nb, int ng, int ntn, int nsplit,
           c128 *__restrict__ part, int ldp)      // part[split][na_pad][ldp], ldp = nb_pad
{
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + SG_ST * SG_STAGE_BYTES);
    uint64_t *empty = full + SG_ST;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tm = blockIdx.x / ntn, tn = blockIdx.x % ntn, split = blockIdx.y;
    const int nkc = (ng + SG_KS - 1) / SG_KS;
    const int kc0 = (int)((long long)split * nkc / nsplit), kc1 = (int)((long long)(split + 1) * nkc / nsplit);
    const int nit = kc1 - kc0;
    const int va = min(SG_T, na - tm * SG_T), vb = min(SG_T, nb - tn * SG_T);     // valid rows of the two operands

    if (threadIdx.x == 0) {
        for (int s = 0; s < SG_ST; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], SG_CW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    {   // rows that do not exist (ragged na / nb) stay zero for the whole kernel
        double2 *z = reinterpret_cast<double2 *>(smem);
        for (int i = threadIdx.x; i < SG_ST * SG_STAGE_BYTES / 16; i += blockDim.x) z[i] = make_double2(0.0, 0.0);
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();

    if (warp == SG_CW) {
        // ---- producer warp: one row copy per operand row and stage (4 rows per lane) ----
        for (int it = 0; it < nit; ++it) {
            const int s = it % SG_ST;
            if (it >= SG_ST) mbar_wait(&empty[s], ((it / SG_ST) - 1) & 1);
            unsigned char *stage = smem + s * SG_STAGE_BYTES;
            const int kc = kc0 + it;
            const int nk = min(SG_KS, ng - kc * SG_KS);
            if (nk < SG_KS) {                   // ragged K tail: clear what the short copies will not write
                for (int r = lane; r < 2 * SG_T; r += 32) {
                    double2 *row = reinterpret_cast<double2 *>(stage + r * SG_ROW_BYTES);
                    for (int k = nk; k < SG_KS; ++k) row[k] = make_double2(0.0, 0.0);
                }
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            }
            __syncwarp();
            if (lane == 0) mbar_expect_tx(&full[s], (uint32_t)((va + vb) * nk * 16));
            __syncwarp();
            for (int r = lane; r < SG_T; r += 32) {
                if (r < va)
                    bulk_g2s(stage + r * SG_ROW_BYTES, a + (size_t)(tm * SG_T + r) * ng + (size_t)kc * SG_KS,
                             (uint32_t)(nk * 16), &full[s]);
                if (r < vb)
                    bulk_g2s(stage + (SG_T + r) * SG_ROW_BYTES, b + (size_t)(tn * SG_T + r) * ng + (size_t)kc * SG_KS,
                             (uint32_t)(nk * 16), &full[s]);
            }
        }
    } else {
        // ---- consumer warps: 16 rows of a (wm) x 32 rows of b (wn) ----
        const int r8 = lane >> 2, c = lane & 3;
        const int wm = warp & 3, wn = warp >> 2;
        double t1[2][4][2], t2[2][4][2], t3[2][4][2];
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) { t1[i][j][e] = 0.0; t2[i][j][e] = 0.0; t3[i][j][e] = 0.0; }
        int aoff[2], boff[4];
#pragma unroll
        for (int i = 0; i < 2; ++i) aoff[i] = (wm * 16 + i * 8 + r8) * SG_ROW_BYTES + c * 16;
#pragma unroll
        for (int j = 0; j < 4; ++j) boff[j] = (SG_T + wn * 32 + j * 8 + r8) * SG_ROW_BYTES + c * 16;
        for (int it = 0; it < nit; ++it) {
            const int s = it % SG_ST;
            mbar_wait(&full[s], (it / SG_ST) & 1);
            const unsigned char *stage = smem + s * SG_STAGE_BYTES;
#pragma unroll
            for (int kk = 0; kk < SG_KS / 4; ++kk) {
                double2 av[2], bv[4];
#pragma unroll
                for (int i = 0; i < 2; ++i) av[i] = lds_c128(stage, aoff[i] + 4 * kk * 16);
#pragma unroll
                for (int j = 0; j < 4; ++j) bv[j] = lds_c128(stage, boff[j] + 4 * kk * 16);
                double bs[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) bs[j] = bv[j].x + bv[j].y;
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    const double as = av[i].x - av[i].y;
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        dmma884(t1[i][j][0], t1[i][j][1], av[i].x, bv[j].x);
                        dmma884(t2[i][j][0], t2[i][j][1], av[i].y, bv[j].y);
                        dmma884(t3[i][j][0], t3[i][j][1], as, bs[j]);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[s]);
        }
        // conj(a) b:  re = T1 + T2,  im = T3 - T1 + T2
        const size_t plane = (size_t)((na + SG_T - 1) / SG_T) * SG_T * ldp;
        c128 *P = part + (size_t)split * plane;
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int row = tm * SG_T + wm * 16 + i * 8 + r8, col = tn * SG_T + wn * 32 + j * 8 + 2 * c;
#pragma unroll
                for (int e = 0; e < 2; ++e)
                    P[(size_t)row * ldp + col + e] =
                        c128{t1[i][j][e] + t2[i][j][e], t3[i][j][e] - t1[i][j][e] + t2[i][j][e]};
            }
    }
}

// S[i][j] = sum over splits of part[split][i][j], fixed order
__global__ void k_sub_reduce(const c128 *__restrict__ part, int nsplit, size_t plane, int ldp, int na, int nb,
                             c128 *__restrict__ s_out)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= na * nb) return;
    const int i = idx / nb, j = idx % nb;
    const c128 *src = part + (size_t)i * ldp + j;
    double sr[4] = {0.0, 0.0, 0.0, 0.0}, si[4] = {0.0, 0.0, 0.0, 0.0};
    int s = 0;
    for (; s + 4 <= nsplit; s += 4) {
#pragma unroll
        for (int q = 0; q < 4; ++q) { const double2 v = ldg_c128(src + (size_t)(s + q) * plane); sr[q] += v.x; si[q] += v.y; }
    }
    for (; s < nsplit; ++s) { const double2 v = ldg_c128(src + (size_t)s * plane); sr[0] += v.x; si[0] += v.y; }
    s_out[idx] = c128{(sr[0] + sr[1]) + (sr[2] + sr[3]), (si[0] + si[1]) + (si[2] + si[3])};
}
