// Tensor memory (TMEM, 256 KB per SM on sm_100a) as a per-thread store for rows of constants.
//
// The plane kernel keeps one or two rows of twiddle factors per thread (exp(-2 pi i u j / N), j < R, for the thread's
// fixed u).  In registers they cost 4 (R - 1) registers per row for the whole kernel, which is what caps the kernel at
// 12 warps per SM; in shared memory every use would cost a 16-byte access on the pipe the kernel is bound by.  TMEM has
// its own datapath: with the 32x32b shape of tcgen05.st / tcgen05.ld lane i of a warp owns TMEM lane 32 (warp % 4) + i,
// so a column range private to the warp is thread-private storage.  A row is written once at kernel start and read back
// (tcgen05.ld, SASS LDTM) right before it is used, when the transform's temporaries are dead.
//
// tcgen05.ld / .st / .wait are .sync.aligned: every lane of the warp must execute them convergently; the callers fetch
// rows outside the `if (line exists)` branches.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "fft_phases.cuh"

__host__ __device__ constexpr int qm_tmem_cols_pow2(int c) { return c <= 32 ? 32 : c <= 64 ? 64 : c <= 128 ? 128 : c <= 256 ? 256 : 512; }

// One warp allocates `ncols` columns (a power of two >= 32) and publishes the base address through shared memory.
__device__ __forceinline__ void tmem_alloc(uint32_t *slot_smem, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(slot_smem)), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t base, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// Address of column `col0 + colstride * (warp / 4)` in this warp's lane window.  The warp index goes through a
// broadcast shuffle so that the compiler knows the address is warp-uniform (tcgen05.ld / .st take it from a uniform register).
__device__ __forceinline__ uint32_t tmem_warp_addr(uint32_t base, int col0, int colstride) {
    const uint32_t warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    return base + (((warp & 3u) * 32u) << 16) + (uint32_t)(col0 + colstride * (int)(warp >> 2));
}

__device__ __forceinline__ void tmem_st_c128(uint32_t taddr, c128 v) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};"
                 ::"r"(taddr), "r"(__double2loint(v.x)), "r"(__double2hiint(v.x)), "r"(__double2loint(v.y)), "r"(__double2hiint(v.y)) : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// row[j] (j = 1 .. R-1) at columns taddr + 4 j; row[0] is 1 and is not stored
template <int R> __device__ __forceinline__ void tmem_store_row(uint32_t taddr, const TwRow<R> &t) {
    static_for<R>([&](auto I) {
        constexpr int j = decltype(I)::value;
        if constexpr (j > 0) tmem_st_c128(taddr + 4 * j, t.w[j]);
    });
}
// Reads factors [J0, J1) of a row back (at most four): load(s) and wait are one asm statement, so no use of the loaded
// registers can be scheduled ahead of the wait.
template <int J0, int J1> __device__ __forceinline__ void tmem_load_chunk(TwChunk<J0, J1> &t, uint32_t taddr) {
    constexpr int K = J1 - J0;
    static_assert(K >= 1 && K <= 4, "chunk of 1..4 factors");
    int r[4][4];
    const uint32_t a = taddr + 4 * J0;
    if constexpr (K == 4)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];\n"
                     "tcgen05.wait::ld.sync.aligned;"
                     : "=r"(r[0][0]), "=r"(r[0][1]), "=r"(r[0][2]), "=r"(r[0][3]), "=r"(r[1][0]), "=r"(r[1][1]), "=r"(r[1][2]), "=r"(r[1][3]),
                       "=r"(r[2][0]), "=r"(r[2][1]), "=r"(r[2][2]), "=r"(r[2][3]), "=r"(r[3][0]), "=r"(r[3][1]), "=r"(r[3][2]), "=r"(r[3][3])
                     : "r"(a) : "memory");
    else if constexpr (K == 3)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%12];\n"
                     "tcgen05.ld.sync.aligned.32x32b.x4.b32 {%8, %9, %10, %11}, [%13];\n"
                     "tcgen05.wait::ld.sync.aligned;"
                     : "=r"(r[0][0]), "=r"(r[0][1]), "=r"(r[0][2]), "=r"(r[0][3]), "=r"(r[1][0]), "=r"(r[1][1]), "=r"(r[1][2]), "=r"(r[1][3]),
                       "=r"(r[2][0]), "=r"(r[2][1]), "=r"(r[2][2]), "=r"(r[2][3])
                     : "r"(a), "r"(a + 8) : "memory");
    else if constexpr (K == 2)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];\n"
                     "tcgen05.wait::ld.sync.aligned;"
                     : "=r"(r[0][0]), "=r"(r[0][1]), "=r"(r[0][2]), "=r"(r[0][3]), "=r"(r[1][0]), "=r"(r[1][1]), "=r"(r[1][2]), "=r"(r[1][3])
                     : "r"(a) : "memory");
    else
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];\n"
                     "tcgen05.wait::ld.sync.aligned;"
                     : "=r"(r[0][0]), "=r"(r[0][1]), "=r"(r[0][2]), "=r"(r[0][3]) : "r"(a) : "memory");
    static_for<K>([&](auto I) {
        constexpr int i = decltype(I)::value;
        t.w[i] = c128{__hiloint2double(r[i][1], r[i][0]), __hiloint2double(r[i][3], r[i][2])};
    });
}

// The same in two halves, so that the next chunk's read is in flight while the current chunk is used: issue (tcgen05.ld
// only) and land (tcgen05.wait::ld, then the raw registers pass through an empty asm statement so that no use can be
// scheduled ahead of the wait).  tcgen05.wait::ld covers every read issued before it.
template <int K> __device__ __forceinline__ void tmem_issue(int (&r)[4][4], uint32_t a) {
    static_assert(K >= 1 && K <= 4, "chunk of 1..4 factors");
    if constexpr (K == 4)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                     : "=r"(r[0][0]), "=r"(r[0][1]), "=r"(r[0][2]), "=r"(r[0][3]), "=r"(r[1][0]), "=r"(r[1][1]), "=r"(r[1][2]), "=r"(r[1][3]),
                       "=r"(r[2][0]), "=r"(r[2][1]), "=r"(r[2][2]), "=r"(r[2][3]), "=r"(r[3][0]), "=r"(r[3][1]), "=r"(r[3][2]), "=r"(r[3][3])
                     : "r"(a) : "memory");
    else if constexpr (K == 3)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%12];\n"
                     "tcgen05.ld.sync.aligned.32x32b.x4.b32 {%8, %9, %10, %11}, [%13];"
                     : "=r"(r[0][0]), "=r"(r[0][1]), "=r"(r[0][2]), "=r"(r[0][3]), "=r"(r[1][0]), "=r"(r[1][1]), "=r"(r[1][2]), "=r"(r[1][3]),
                       "=r"(r[2][0]), "=r"(r[2][1]), "=r"(r[2][2]), "=r"(r[2][3])
                     : "r"(a), "r"(a + 8) : "memory");
    else if constexpr (K == 2)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                     : "=r"(r[0][0]), "=r"(r[0][1]), "=r"(r[0][2]), "=r"(r[0][3]), "=r"(r[1][0]), "=r"(r[1][1]), "=r"(r[1][2]), "=r"(r[1][3])
                     : "r"(a) : "memory");
    else
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                     : "=r"(r[0][0]), "=r"(r[0][1]), "=r"(r[0][2]), "=r"(r[0][3]) : "r"(a) : "memory");
}
template <int J0, int J1> __device__ __forceinline__ void tmem_land(TwChunk<J0, J1> &t, int (&r)[4][4]) {
    constexpr int K = J1 - J0;
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    static_for<K>([&](auto I) {
        constexpr int i = decltype(I)::value;
        asm volatile("" : "+r"(r[i][0]), "+r"(r[i][1]), "+r"(r[i][2]), "+r"(r[i][3]));
        t.w[i] = c128{__hiloint2double(r[i][1], r[i][0]), __hiloint2double(r[i][3], r[i][2])};
    });
}
