// Launches of the z-stick kernels (k_zinv: scatter + backward z transform; k_zfwd: forward z transform + gather) for
// every supported FFT length.  Own translation unit: compiled in parallel with the plane kernels.
#include "qm_internal.h"

namespace {

template <class C, bool PH> int launch_zinv(qm_gspace *g, KPoint *kp, const c128 *psi, const c128 *phase, c128 *W, int nb,
                                            cudaStream_t st) {
    const int ntiles = (kp->nsticks + QM_ZT - 1) / QM_ZT;
    dim3 grid(z_grid_x(g, ntiles, nb, g->z_cta_per_sm), nb);
    g->prof.begin(QM_K_ZINV, st);
    CU_TRY(qm_launch_pdl(k_zinv<C, PH>, grid, dim3(QM_ZT * C::TT), qm_z_smem<C>(), st, g->pdl, kp->plan(), g->d_tw[2].p, psi, phase, W,
                         ntiles, kp->z_quarter ? 1 : 0));
    g->prof.end(st);
    g->launches++;
    CU_TRY(cudaGetLastError());
    return QM_OK;
}
template <class C, int GM> int launch_zfwd(qm_gspace *g, KPoint *kp, const c128 *W, const c128 *aux, c128 *out, int nb,
                                           double scale, cudaStream_t st) {
    const int ntiles = (kp->nsticks + QM_ZT - 1) / QM_ZT;
    dim3 grid(z_grid_x(g, ntiles, nb, g->z_cta_per_sm), nb);
    g->prof.begin(QM_K_ZFWD, st);
    CU_TRY(qm_launch_pdl(k_zfwd<C, GM>, grid, dim3(QM_ZT * C::TT), qm_z_smem<C>(), st, g->pdl, kp->plan(), g->d_tw[2].p, W, aux, out,
                         ntiles, scale, kp->z_quarter ? 1 : 0));
    g->prof.end(st);
    g->launches++;
    CU_TRY(cudaGetLastError());
    return QM_OK;
}
template <class C> int prep_z_kernels() {
    const int smem = (int)qm_z_smem<C>();
    CU_TRY(cudaFuncSetAttribute(k_zinv<C, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    CU_TRY(cudaFuncSetAttribute(k_zinv<C, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    CU_TRY(cudaFuncSetAttribute(k_zfwd<C, GM_PLAIN>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    CU_TRY(cudaFuncSetAttribute(k_zfwd<C, GM_KINETIC>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    CU_TRY(cudaFuncSetAttribute(k_zfwd<C, GM_PHASE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    CU_TRY(cudaFuncSetAttribute(k_zfwd<C, GM_CONJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    return QM_OK;
}
}  // namespace

int qm_launch_zinv(qm_gspace *g, KPoint *kp, const c128 *psi, const c128 *phase, c128 *W, int nb, cudaStream_t st) {
    switch (g->grid[2]) {
#define X(N, A, B)                                                                               \
    case N: return phase ? launch_zinv<LineCfg<A, B>, true>(g, kp, psi, phase, W, nb, st)         \
                         : launch_zinv<LineCfg<A, B>, false>(g, kp, psi, nullptr, W, nb, st);
        QM_FOR_SIZES_ALL(X)
#undef X
    }
    return fail(QM_EGRID, "unsupported FFT length (axis 3)");
}

template <class C> static int zfwd_by_mode(qm_gspace *g, KPoint *kp, int gm, const c128 *W, const c128 *aux, c128 *out, int nb,
                                           double scale, cudaStream_t st) {
    switch (gm) {
        case GM_PLAIN: return launch_zfwd<C, GM_PLAIN>(g, kp, W, aux, out, nb, scale, st);
        case GM_KINETIC: return launch_zfwd<C, GM_KINETIC>(g, kp, W, aux, out, nb, scale, st);
        case GM_PHASE: return launch_zfwd<C, GM_PHASE>(g, kp, W, aux, out, nb, scale, st);
        case GM_CONJ: return launch_zfwd<C, GM_CONJ>(g, kp, W, aux, out, nb, scale, st);
    }
    return fail(QM_EINVAL, "bad gather mode");
}
int qm_launch_zfwd(qm_gspace *g, KPoint *kp, int gm, const c128 *W, const c128 *aux, c128 *out, int nb, double scale,
                   cudaStream_t st) {
    switch (g->grid[2]) {
#define X(N, A, B) case N: return zfwd_by_mode<LineCfg<A, B>>(g, kp, gm, W, aux, out, nb, scale, st);
        QM_FOR_SIZES_ALL(X)
#undef X
    }
    return fail(QM_EGRID, "unsupported FFT length (axis 3)");
}

int qm_prepare_z(qm_gspace *g) {
    switch (g->grid[2]) {
#define X(N, A, B) case N: return prep_z_kernels<LineCfg<A, B>>();
        QM_FOR_SIZES_ALL(X)
#undef X
    }
    return fail(QM_EGRID, "unsupported FFT length (axis 3)");
}
