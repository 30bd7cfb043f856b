// Exchange probes: what it costs to hand one complex128 per thread to another thread of the warp, per mechanism.
// They back the choice of shared memory for the transposes between radix passes (north_star (2) names
// warp-shuffle butterflies) and of tensor memory for the twiddle rows, with numbers instead of an argument.
//   mode 0  shared memory: STS.128 to the partner's slot, __syncwarp, LDS.128 of the own slot (what k_plane does per element)
//   mode 1  warp shuffle: 4 x SHFL.32 (a 16-byte element is four 32-bit shuffles) from a lane-dependent source
//   mode 2  tensor memory read: tcgen05.ld 32x32b.x4 of a thread-private element (no exchange: the twiddle-row fetch)
// Every mode runs `iters` dependent rounds on every warp of a full grid; the caller converts to ns per warp-element.
#pragma once
#include "tmem_rows.cuh"

template <int MODE>
__global__ void __launch_bounds__(384) k_probe_exchange(double *sink, int iters)
{
    __shared__ __align__(16) c128 buf[384];
    __shared__ uint32_t tmem_base_s;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int partner = (lane * 5 + 3) & 31;                 // a fixed permutation of the lanes
    c128 v{1.0 + threadIdx.x * 1e-9, 2.0 - threadIdx.x * 1e-9};
    uint32_t taddr = 0, tcols = 0;
    if constexpr (MODE == 2) {
        tcols = (uint32_t)qm_tmem_cols_pow2(4 * ((blockDim.x / 32 + 3) / 4));
        if (threadIdx.x < 32) tmem_alloc(&tmem_base_s, tcols);
        tmem_fence_before_sync(); __syncthreads(); tmem_fence_after_sync();
        taddr = tmem_warp_addr(tmem_base_s, 0, 4);
        tmem_st_c128(taddr, v);
        tmem_wait_st();
    }
    for (int it = 0; it < iters; ++it) {
        if constexpr (MODE == 0) {
            buf[warp * 32 + partner] = v;
            __syncwarp();
            v = buf[warp * 32 + lane];
            __syncwarp();
        } else if constexpr (MODE == 1) {
            int a = __double2loint(v.x), b = __double2hiint(v.x), c = __double2loint(v.y), d = __double2hiint(v.y);
            a = __shfl_sync(0xffffffffu, a, partner); b = __shfl_sync(0xffffffffu, b, partner);
            c = __shfl_sync(0xffffffffu, c, partner); d = __shfl_sync(0xffffffffu, d, partner);
            v = c128{__hiloint2double(b, a), __hiloint2double(d, c)};
        } else {
            TwChunk<0, 1> ch;
            tmem_load_chunk(ch, taddr);
            v = c128{v.x + ch.w[0].x * 1e-30, v.y + ch.w[0].y * 1e-30};
        }
    }
    if (v.x + v.y == 123.456) sink[0] = v.x;
    if constexpr (MODE == 2) {
        tmem_fence_before_sync(); __syncthreads();
        if (threadIdx.x < 32) tmem_dealloc(tmem_base_s, tcols);
    }
}
