// Non-local projector kernels on the FP64 tensor cores (DMMA m8n8k4), sm_100a.
//   a6  P = beta^H psi          PAPER.md:153-161 (eq. 14), 767 ("vdot" as ZGEMM)
//   a7  Q = D P                 block-diagonal real-symmetric D (ONCV multi-projector)
//   a8  out += beta Q
// Complex products are four real DMMA chains (re/im split in registers; beta stays interleaved in HBM).
#pragma once
#include <cuda_runtime.h>
#include "fft_reg.cuh"

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__device__ __forceinline__ double2 ldg_c128(const c128 *p) {
    return __ldg(reinterpret_cast<const double2 *>(p));
}

// ---------------------------------------------------------------------------------------------
// v1 kernels: fragments loaded straight from global memory (L1/L2 give the reuse).
// beta: [nproj_pad][ldb] zero padded (library copy).  psi: caller's [nb][ng].
// Ppart: [nsplit][nproj_pad][nbp].
template <int MT, int NT, int WARPS>
__global__ void __launch_bounds__(WARPS * 32)
k_proj1_direct(const c128 *__restrict__ beta, int ldb, const c128 *__restrict__ psi, int ng,
               int nb, int band0, int nbp, int nproj_pad, c128 *__restrict__ Ppart, int kchunk)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int r = lane >> 2, c = lane & 3;
    const int j0 = (blockIdx.x * WARPS + warp) * 8 * MT;
    if (j0 >= nproj_pad) return;
    const int kbeg = blockIdx.y * kchunk;
    const int kend = min(ng, kbeg + kchunk);
    double cre[MT][NT][2], cim[MT][NT][2];
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j) { cre[i][j][0] = cre[i][j][1] = cim[i][j][0] = cim[i][j][1] = 0.0; }
    const c128 *bp[MT];
#pragma unroll
    for (int i = 0; i < MT; ++i) bp[i] = beta + (size_t)(j0 + i * 8 + r) * ldb + c;
    const c128 *pp[NT];
#pragma unroll
    for (int j = 0; j < NT; ++j) pp[j] = psi + (size_t)min(band0 + j * 8 + r, nb - 1) * ng + c;
#pragma unroll 2
    for (int k = kbeg; k < kend; k += 4) {
        double2 a[MT], b[NT];
        const bool ok = (k + c) < kend;
#pragma unroll
        for (int i = 0; i < MT; ++i) a[i] = ldg_c128(bp[i] + k);      // beta is zero padded past ng
#pragma unroll
        for (int j = 0; j < NT; ++j) b[j] = ok ? ldg_c128(pp[j] + k) : make_double2(0.0, 0.0);
#pragma unroll
        for (int i = 0; i < MT; ++i)
#pragma unroll
            for (int j = 0; j < NT; ++j) {
                // conj(a) * b = (ar br + ai bi) + i (ar bi - ai br)
                dmma884(cre[i][j][0], cre[i][j][1], a[i].x, b[j].x);
                dmma884(cre[i][j][0], cre[i][j][1], a[i].y, b[j].y);
                dmma884(cim[i][j][0], cim[i][j][1], a[i].x, b[j].y);
                dmma884(cim[i][j][0], cim[i][j][1], a[i].y, -b[j].x);
            }
    }
    c128 *P = Ppart + (size_t)blockIdx.y * nproj_pad * nbp;
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j) {
            const int row = j0 + i * 8 + r, col = j * 8 + 2 * c;
            P[(size_t)row * nbp + col] = c128{cre[i][j][0], cim[i][j][0]};
            P[(size_t)row * nbp + col + 1] = c128{cre[i][j][1], cim[i][j][1]};
        }
}

// P[j][n] = sum_s Ppart[s][j][n]  (fixed order => deterministic)
__global__ void k_reduce_p(const c128 *__restrict__ Ppart, int nsplit, int count, c128 *__restrict__ P)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    double sr = 0.0, si = 0.0;
    for (int s = 0; s < nsplit; ++s) {
        const double2 v = ldg_c128(Ppart + (size_t)s * count + i);
        sr += v.x; si += v.y;
    }
    P[i] = c128{sr, si};
}

// Q[i][n] = sum_{j in block(i)} D[blk][i%db][j%db] P[j][n];  rows >= nproj are written as zero.
__global__ void k_dmul(const double *__restrict__ D, int db, int nproj, int nproj_pad, int nbp,
                       const c128 *__restrict__ P, c128 *__restrict__ Q)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= nproj_pad * nbp) return;
    const int i = idx / nbp, n = idx % nbp;
    double sr = 0.0, si = 0.0;
    if (i < nproj) {
        const int blk = i / db, ii = i % db;
        const double *d = D + ((size_t)blk * db + ii) * db;
        for (int j = 0; j < db; ++j) {
            const double2 v = ldg_c128(P + (size_t)(blk * db + j) * nbp + n);
            sr += d[j] * v.x; si += d[j] * v.y;
        }
    }
    Q[idx] = c128{sr, si};
}

// out[n][g] += sum_i beta[i][g] Q[i][n]
template <int MT, int NT, int WARPS>
__global__ void __launch_bounds__(WARPS * 32)
k_proj2_direct(const c128 *__restrict__ beta, int ldb, const c128 *__restrict__ Q, int nbp, int nproj_pad,
               int ng, int nb, int band0, c128 *__restrict__ out)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int r = lane >> 2, c = lane & 3;
    const int g0 = (blockIdx.x * WARPS + warp) * 8 * MT;
    if (g0 >= ng) return;
    double cre[MT][NT][2], cim[MT][NT][2];
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j) { cre[i][j][0] = cre[i][j][1] = cim[i][j][0] = cim[i][j][1] = 0.0; }
    const c128 *bp = beta + (size_t)c * ldb + g0 + r;          // ldb >= roundup(ng, 8*MT*WARPS): in bounds
    const c128 *qp = Q + (size_t)c * nbp + r;
#pragma unroll 2
    for (int k = 0; k < nproj_pad; k += 4) {
        double2 a[MT], b[NT];
#pragma unroll
        for (int i = 0; i < MT; ++i) a[i] = ldg_c128(bp + (size_t)k * ldb + i * 8);
#pragma unroll
        for (int j = 0; j < NT; ++j) b[j] = ldg_c128(qp + (size_t)k * nbp + j * 8);
#pragma unroll
        for (int i = 0; i < MT; ++i)
#pragma unroll
            for (int j = 0; j < NT; ++j) {
                // a * b = (ar br - ai bi) + i (ar bi + ai br)
                dmma884(cre[i][j][0], cre[i][j][1], a[i].x, b[j].x);
                dmma884(cre[i][j][0], cre[i][j][1], a[i].y, -b[j].y);
                dmma884(cim[i][j][0], cim[i][j][1], a[i].x, b[j].y);
                dmma884(cim[i][j][0], cim[i][j][1], a[i].y, b[j].x);
            }
    }
#pragma unroll
    for (int i = 0; i < MT; ++i) {
        const int g = g0 + i * 8 + r;
        if (g >= ng) continue;
#pragma unroll
        for (int j = 0; j < NT; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int n = band0 + j * 8 + 2 * c + e;
                if (n < nb) {
                    c128 *o = out + (size_t)n * ng + g;
                    c128 v = *o;
                    v.x += cre[i][j][e]; v.y += cim[i][j][e];
                    *o = v;
                }
            }
    }
}

// ---------------------------------------------------------------------------------------------
// Peak probes: register-resident DMMA / DFMA loops (roofline denominators for the projector GEMMs).
__global__ void k_probe_dmma(double *sink, int iters)
{
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; ++i) { c[i][0] = threadIdx.x * 1e-9; c[i][1] = i * 1e-9; }
    const double a = 1.0 + 1e-12 * threadIdx.x, b = 1.0 - 1e-12 * threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) dmma884(c[i][0], c[i][1], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
    if (s == 123.456) sink[0] = s;
}
__global__ void k_probe_dfma(double *sink, int iters)
{
    double c[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = threadIdx.x * 1e-9 + i;
    const double a = 1.0 + 1e-12 * threadIdx.x, b = 1e-13 * threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) c[i] = fma(c[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += c[i];
    if (s == 123.456) sink[0] = s;
}
