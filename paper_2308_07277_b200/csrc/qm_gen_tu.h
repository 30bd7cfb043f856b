// One translation unit of the unfused passes (gen_kernels.cuh): QM_GEN_TU = 0..4 -> the x pass of that MODE for every
// supported FFT length; QM_GEN_TU = 5 -> the two y passes.  Included by qm_genx0.cu ... qm_genx4.cu and qm_geny.cu, so
// that they compile in parallel with the fused-kernel units.
#include "qm_internal.h"
#include "gen_kernels.cuh"

#define QM_CAT2(a, b) a##b
#define QM_CAT(a, b) QM_CAT2(a, b)

namespace {
#if QM_GEN_TU == 5
template <class C, bool BACK> int launch_gen_y(qm_gspace *g, KPoint *kp, c128 *W, c128 *slab, int bp0, int nbp, cudaStream_t st) {
    using GG = GenGeom<C>;
    const long long items = (long long)nbp * kp->nx;
    if (items * GG::TPG >= (1LL << 31)) return fail(QM_EINVAL, "unfused y pass: too many rows in one launch");
    // persistent: a CTA walks row chunks gridDim.x apart (twiddle rows loaded once); several CTAs per SM hide latency
    const long long nchunks = (items + GG::TPG - 1) / GG::TPG;
    int &per_sm = kp->gen_y_per_sm[BACK ? 1 : 0];
    if (per_sm == 0) {
        CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_gen_y<C, BACK>, GEN_GROUP, GG::y_smem()));
        per_sm = std::max(1, per_sm);
    }
    const unsigned grid = (unsigned)std::min<long long>(nchunks, (long long)g->sm_count * std::max(1, per_sm));
    const size_t wband = (size_t)((kp->nsticks + QM_ZT - 1) / QM_ZT) * QM_ZT * g->grid[2];
    g->prof.begin(QM_K_GENY, st);
    CU_TRY(qm_launch_pdl(k_gen_y<C, BACK>, dim3(grid), dim3(GEN_GROUP), GG::y_smem(), st, g->pdl, kp->plan(), (const c128 *)g->d_tw[1].p,
                         W, slab, g->grid[2], bp0, nbp, kp->y_quarter ? 1 : 0, wband));
    g->prof.end(st);
    g->launches++;
    CU_TRY(cudaGetLastError());
    return QM_OK;
}
#else
template <class C, int MODE> int launch_gen_x(qm_gspace *g, KPoint *kp, c128 *slab, int bp0, int nbp, const PlaneArgs &a,
                                              cudaStream_t st) {
    using GG = GenGeom<C>;
    const size_t smem = GG::x_smem(kp->nx);
    if (smem > (size_t)g->max_smem) return fail(QM_EGRID, "x tile of the unfused path does not fit shared memory");
    const int n2 = g->grid[1], n3 = g->grid[2];
    const int nchunk = (n2 + GG::TC - 1) / GG::TC;
    const long long tiles = (long long)(MODE == 3 ? n3 : nbp) * nchunk;
    // persistent: a CTA walks tiles gridDim.x apart; as many CTAs as are resident
    int &per_sm = kp->gen_x_per_sm[MODE];
    if (per_sm == 0) {
        CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_gen_x<C, MODE>, GG::XG * GEN_GROUP, smem));
        per_sm = std::max(1, per_sm);
    }
    const unsigned grid = (unsigned)std::min<long long>(tiles, (long long)g->sm_count * std::max(1, per_sm));
    g->prof.begin(QM_K_GENX, st);
    CU_TRY(qm_launch_pdl(k_gen_x<C, MODE>, dim3(grid), dim3(GG::XG * GEN_GROUP), smem, st, g->pdl, kp->plan(), (const c128 *)g->d_tw[0].p,
                         (const double *)g->d_vt.p, slab, a.box, a.box2, a.npair2, a.scale, n2, n3, bp0, nbp,
                         (kp->y_quarter ? 1 : 0) | (kp->x_quarter ? 2 : 0), a.occ, a.rhot));
    g->prof.end(st);
    g->launches++;
    CU_TRY(cudaGetLastError());
    return QM_OK;
}
#endif
}  // namespace

#if QM_GEN_TU == 5
int qm_launch_gen_y(qm_gspace *g, KPoint *kp, bool back, c128 *W, c128 *slab, int bp0, int nbp, cudaStream_t st) {
    switch (g->grid[1]) {
#define X(N, A, B)                                                                              \
    case N: return back ? launch_gen_y<LineCfg<A, B>, true>(g, kp, W, slab, bp0, nbp, st)        \
                        : launch_gen_y<LineCfg<A, B>, false>(g, kp, W, slab, bp0, nbp, st);
        QM_FOR_SIZES_ALL(X)
#undef X
    }
    return fail(QM_EGRID, "unsupported FFT length (axis 2)");
}
int qm_prepare_gen_y(qm_gspace *g) {
    switch (g->grid[1]) {
#define X(N, A, B)                                                                                                    \
    case N:                                                                                                           \
        CU_TRY(cudaFuncSetAttribute(k_gen_y<LineCfg<A, B>, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,         \
                                    (int)GenGeom<LineCfg<A, B>>::y_smem()));                                           \
        CU_TRY(cudaFuncSetAttribute(k_gen_y<LineCfg<A, B>, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,        \
                                    (int)GenGeom<LineCfg<A, B>>::y_smem()));                                           \
        for (KPoint *kp : g->kpts) {                                                                                  \
            CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&kp->gen_y_per_sm[0], k_gen_y<LineCfg<A, B>, false>, \
                                                                 GEN_GROUP, GenGeom<LineCfg<A, B>>::y_smem()));        \
            CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&kp->gen_y_per_sm[1], k_gen_y<LineCfg<A, B>, true>,  \
                                                                 GEN_GROUP, GenGeom<LineCfg<A, B>>::y_smem()));        \
            kp->gen_y_per_sm[0] = std::max(1, kp->gen_y_per_sm[0]);                                                   \
            kp->gen_y_per_sm[1] = std::max(1, kp->gen_y_per_sm[1]);                                                   \
        }                                                                                                             \
        return QM_OK;
        QM_FOR_SIZES_ALL(X)
#undef X
    }
    return fail(QM_EGRID, "unsupported FFT length (axis 2)");
}
#else
int QM_CAT(qm_launch_gen_x_m, QM_GEN_TU)(qm_gspace *g, KPoint *kp, c128 *slab, int bp0, int nbp, const PlaneArgs &a, cudaStream_t st) {
    switch (g->grid[0]) {
#define X(N, A, B) case N: return launch_gen_x<LineCfg<A, B>, QM_GEN_TU>(g, kp, slab, bp0, nbp, a, st);
        QM_FOR_SIZES_ALL(X)
#undef X
    }
    return fail(QM_EGRID, "unsupported FFT length (axis 1)");
}
int QM_CAT(qm_prepare_gen_x_m, QM_GEN_TU)(qm_gspace *g) {
    switch (g->grid[0]) {
#define X(N, A, B)                                                                                                              \
    case N: CU_TRY(cudaFuncSetAttribute(k_gen_x<LineCfg<A, B>, QM_GEN_TU>, cudaFuncAttributeMaxDynamicSharedMemorySize,          \
                                        g->max_smem));                                                                           \
        for (KPoint *kp : g->kpts) {    /* the x tile must fit, and its occupancy is asked once, here */                         \
            const size_t smem = GenGeom<LineCfg<A, B>>::x_smem(kp->nx);                                                          \
            if (smem > (size_t)g->max_smem) return fail(QM_EGRID, "x tile of the unfused path does not fit shared memory");      \
            int &per_sm = kp->gen_x_per_sm[QM_GEN_TU];                                                                           \
            CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_gen_x<LineCfg<A, B>, QM_GEN_TU>,                     \
                                                                 GenGeom<LineCfg<A, B>>::XG * GEN_GROUP, smem));                 \
            per_sm = std::max(1, per_sm);                                                                                        \
        }                                                                                                                        \
        return QM_OK;
        QM_FOR_SIZES_ALL(X)
#undef X
    }
    return fail(QM_EGRID, "unsupported FFT length (axis 1)");
}
#endif
