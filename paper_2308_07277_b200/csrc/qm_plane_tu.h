// One translation unit of the fused xy-plane kernel: every supported FFT length for ONE mode (QM_TU_MODE), so that the
// five modes compile in parallel.  Included by qm_plane0.cu ... qm_plane4.cu.
#include "qm_internal.h"

#define QM_CAT2(a, b) a##b
#define QM_CAT(a, b) QM_CAT2(a, b)

namespace {

template <class C, int MODE> int launch_plane(qm_gspace *g, KPoint *kp, c128 *W, int nb, const PlaneArgs &a, cudaStream_t st) {
    // two resident CTAs per SM (half the groups each) when two plane arrays fit: each walks its own planes, so the
    // CTA-wide barriers and the load / compute / store phases of one CTA overlap the other's work (measured with the
    // twiddle rows in tensor memory: cfg4 -5 %, cfg3 -15 %, cfg2 -11 % plane-kernel time; cfg5's plane array allows one)
    int cps = MODE == 3 ? 1 : (g->plane_ctas_per_sm > 0 ? g->plane_ctas_per_sm : 2);
    int ngroups = plane_groups(g, kp, cps);
    // every resident CTA allocates its own tensor-memory columns (512 per SM): one CTA per SM if two do not fit
    // (one CTA always fits: a build whose thread limit needs more than an SM's 512 columns does not compile)
    static_assert(!plane_tw_tmem<C> ||
                      (4 * C::R1 + (C::R1 != C::R2 ? 4 * C::R2 : 0)) * ((QM_PLANE_MAX_THREADS / 32 + 3) / 4) <= 512,
                  "QM_PLANE_MAX_THREADS: the twiddle rows of this line factorisation do not fit 512 tensor-memory columns");
    if (plane_tw_tmem<C> && cps > 1 && ngroups > 0) {
        const int rowcols = 4 * C::R1 + (C::R1 != C::R2 ? 4 * C::R2 : 0);
        if (cps * qm_tmem_cols_pow2(rowcols * ((ngroups * PLANE_GROUP / 32 + 3) / 4)) > 512) ngroups = 0;
    }
    if (ngroups == 0) { cps = 1; ngroups = plane_groups(g, kp, 1); }
    size_t smem = plane_smem(g, kp, ngroups);
    if (ngroups == 0 || smem > (size_t)g->max_smem)
        return fail(QM_EGRID, "plane kernel does not fit shared memory for this grid / sphere");
    // the per-(row, u) addressing table of the y phase, when there is room for it beside the plane array
    const size_t budget = cps == 1 ? (size_t)g->max_smem : ((size_t)g->max_smem + 1024) / cps - 1024;
    const bool rowtab = smem + plane_rowtab_bytes(g, kp) <= budget;
    if (rowtab) smem += plane_rowtab_bytes(g, kp);
    QmGridDev gd;
    for (int i = 0; i < 3; ++i) { gd.ax[i] = g->ax[i]; gd.tw[i] = g->d_tw[i].p; }
    gd.vt = g->d_vt.p;
    const int nplanes = g->grid[2] * nb;
    // persistent: one CTA per SM walks the (band, z-plane) list; density mode: one CTA per z-plane, all bands
    const int grid = MODE == 3 ? std::min(g->grid[2], g->sm_count) : std::min(nplanes, g->sm_count * cps);
    g->prof.begin(QM_K_PLANE, st);
    CU_TRY(qm_launch_pdl(k_plane<C, MODE>, dim3(grid), dim3(ngroups * PLANE_GROUP), smem, st, g->pdl, kp->plan(), gd, W, a.box, a.box2,
                         a.npair2, ngroups, a.scale, nplanes,
                         (kp->y_quarter ? 1 : 0) | (kp->x_quarter ? 2 : 0) | (rowtab ? 4 : 0), a.occ, a.rhot));
    g->prof.end(st);
    g->launches++;
    CU_TRY(cudaGetLastError());
    return QM_OK;
}

}  // namespace

int QM_CAT(qm_launch_plane_m, QM_TU_MODE)(qm_gspace *g, KPoint *kp, c128 *W, int nb, const PlaneArgs &a, cudaStream_t st) {
    switch (g->grid[0]) {
#define X(N, A, B) case N: return launch_plane<LineCfg<A, B>, QM_TU_MODE>(g, kp, W, nb, a, st);
        QM_FOR_SIZES(X)
#undef X
    }
    return fail(QM_EGRID, "unsupported FFT length (axes 1,2)");
}

int QM_CAT(qm_prepare_plane_m, QM_TU_MODE)(qm_gspace *g) {
    switch (g->grid[0]) {
#define X(N, A, B)                                                                                                       \
    case N: CU_TRY(cudaFuncSetAttribute(k_plane<LineCfg<A, B>, QM_TU_MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                        g->max_smem));                                                                    \
        return QM_OK;
        QM_FOR_SIZES(X)
#undef X
    }
    return fail(QM_EGRID, "unsupported FFT length (axes 1,2)");
}
