// C ABI of libqm_hpsi (see include/qm_hpsi.h).  Host-side set-up (G-sphere, stick tables) and
// kernel launches.  No CPU fallback: compute entry points fail with QM_ECUDA without a device.
#include "qm_internal.h"
#include "proj_kernels.cuh"
#include "subspace_kernels.cuh"
#include <cstdint>
#include <mutex>

thread_local std::string qm_g_err;

namespace {

int build_kpoint(qm_gspace *g, KPoint *kp, bool strict = false) {
    std::string msg;
    const int rc = qm_build_tables(g->lattice, g->recip, strict ? kp->ecut_override : g->ecut, g->grid, g->ax, kp, &msg, strict);
    if (rc == -1) return fail(QM_EGRID, msg);
    if (rc != 0) return fail(QM_EINVAL, msg);
    CU_TRY(kp->d_rowinfo.upload(kp->rowinfo));
    CU_TRY(kp->d_stickinfo.upload(kp->stickinfo));
    CU_TRY(kp->d_g2.upload(kp->g2));
    return QM_OK;
}

// every entry point that touches the device: the handle belongs to one device, which must be current
int check_device(const qm_gspace *g) {
    int dev = -1;
    CU_TRY(cudaGetDevice(&dev));
    if (dev != g->device)
        return fail(QM_EINVAL, "handle was created on CUDA device " + std::to_string(g->device) + ", current device is " +
                                   std::to_string(dev));
    return QM_OK;
}

template <bool PH> int dispatch_zinv(qm_gspace *g, KPoint *kp, const c128 *psi, const c128 *phase, c128 *W, int nb,
                                     cudaStream_t st) {
    return qm_launch_zinv(g, kp, psi, PH ? phase : nullptr, W, nb, st);
}
template <int GM> int dispatch_zfwd(qm_gspace *g, KPoint *kp, const c128 *W, const c128 *aux, c128 *out, int nb, double scale,
                                    cudaStream_t st) {
    return qm_launch_zfwd(g, kp, GM, W, aux, out, nb, scale, st);
}
// Unfused path: bands per slab pass (the slab of half-transformed planes is bounded, not proportional to the call)
size_t gen_slab_per_band(const qm_gspace *g, const KPoint *kp) { return (size_t)g->grid[2] * kp->nx * g->grid[1]; }
int gen_sub_bands(const qm_gspace *g, const KPoint *kp, int nb) {
    const size_t budget = (size_t)1 << 25;          // c128 elements: 512 MB
    return (int)std::max<size_t>(1, std::min<size_t>((size_t)nb, budget / std::max<size_t>(1, gen_slab_per_band(g, kp))));
}
template <int MODE> int launch_gen_x(qm_gspace *g, KPoint *kp, c128 *slab, int bp0, int nbp, const PlaneArgs &a, cudaStream_t st) {
    if constexpr (MODE == 0) return qm_launch_gen_x_m0(g, kp, slab, bp0, nbp, a, st);
    else if constexpr (MODE == 1) return qm_launch_gen_x_m1(g, kp, slab, bp0, nbp, a, st);
    else if constexpr (MODE == 2) return qm_launch_gen_x_m2(g, kp, slab, bp0, nbp, a, st);
    else if constexpr (MODE == 3) return qm_launch_gen_x_m3(g, kp, slab, bp0, nbp, a, st);
    else return qm_launch_gen_x_m4(g, kp, slab, bp0, nbp, a, st);
}
// y backward | x round trip of MODE | y forward, a bounded number of bands at a time (gen_kernels.cuh)
template <int MODE> int run_general(qm_gspace *g, KPoint *kp, c128 *W, int nb, const PlaneArgs &a, cudaStream_t st) {
    const int n3 = g->grid[2], sub = gen_sub_bands(g, kp, nb);
    CU_TRY(kp->d_slab.resize((size_t)sub * gen_slab_per_band(g, kp)));
    for (int b0 = 0; b0 < nb; b0 += sub) {
        const int n = std::min(sub, nb - b0), bp0 = b0 * n3, nbp = n * n3;
        int rc;
        if constexpr (MODE != 2) { rc = qm_launch_gen_y(g, kp, true, W, kp->d_slab.p, bp0, nbp, st); if (rc) return rc; }
        rc = launch_gen_x<MODE>(g, kp, kp->d_slab.p, bp0, nbp, a, st); if (rc) return rc;
        if constexpr (MODE == 0 || MODE == 2 || MODE == 4) {
            rc = qm_launch_gen_y(g, kp, false, W, kp->d_slab.p, bp0, nbp, st); if (rc) return rc;
        }
    }
    return QM_OK;
}
template <int MODE> int dispatch_plane(qm_gspace *g, KPoint *kp, c128 *W, int nb, const PlaneArgs &a, cudaStream_t st) {
    if (!g->fused) return run_general<MODE>(g, kp, W, nb, a, st);
    if constexpr (MODE == 0) return qm_launch_plane_m0(g, kp, W, nb, a, st);
    else if constexpr (MODE == 1) return qm_launch_plane_m1(g, kp, W, nb, a, st);
    else if constexpr (MODE == 2) return qm_launch_plane_m2(g, kp, W, nb, a, st);
    else if constexpr (MODE == 3) return qm_launch_plane_m3(g, kp, W, nb, a, st);
    else return qm_launch_plane_m4(g, kp, W, nb, a, st);
}

// Opt every kernel this handle can launch into its dynamic shared memory ONCE, at handle creation, on the handle's
// device (function attributes are per device; nothing of this kind is left on the hot path).
int prepare_kernels(qm_gspace *g) {
    int rc = qm_prepare_z(g); if (rc) return rc;
    if (g->fused) {
        rc = qm_prepare_plane_m0(g); if (rc) return rc;
        rc = qm_prepare_plane_m1(g); if (rc) return rc;
        rc = qm_prepare_plane_m2(g); if (rc) return rc;
        rc = qm_prepare_plane_m3(g); if (rc) return rc;
        rc = qm_prepare_plane_m4(g); if (rc) return rc;
    } else {
        rc = qm_prepare_gen_y(g); if (rc) return rc;
        rc = qm_prepare_gen_x_m0(g); if (rc) return rc;
        rc = qm_prepare_gen_x_m1(g); if (rc) return rc;
        rc = qm_prepare_gen_x_m2(g); if (rc) return rc;
        rc = qm_prepare_gen_x_m3(g); if (rc) return rc;
        rc = qm_prepare_gen_x_m4(g); if (rc) return rc;
    }
    CU_TRY(cudaFuncSetAttribute(k_proj1_pipe<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, P1Cfg<16>::SMEM));
    CU_TRY(cudaFuncSetAttribute(k_proj2_sk<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, P2Cfg<16>::SMEM));
    CU_TRY(cudaFuncSetAttribute(k_proj1_pipe<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, P1Cfg<32>::SMEM));
    CU_TRY(cudaFuncSetAttribute(k_proj2_sk<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, P2Cfg<32>::SMEM));
    CU_TRY(cudaFuncSetAttribute(k_sub_gemm, cudaFuncAttributeMaxDynamicSharedMemorySize, SG_SMEM));
    return QM_OK;
}

// rho[x][y][z] = scale * rhot[p][col][j][u][e]   (inverse of k_relayout_v's index map; fft_phases.cuh VLayout)
__global__ void k_density_out(const double *__restrict__ rhot, double *__restrict__ rho, QmAxis a1, QmAxis a2, QmAxis a3,
                              double scale)
{
    const int r2e = a1.r2 + (a1.r2 & 1), colsz = a1.r1 * r2e;
    const size_t total = (size_t)a3.n * a2.n * colsz;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int e = (int)(i % colsz);
        const int u = (e >> 1) % a1.r1, k2 = 2 * ((e >> 1) / a1.r1) + (e & 1);
        if (k2 >= a1.r2) continue;
        const int col = (int)((i / colsz) % a2.n);
        const int p = (int)(i / ((size_t)colsz * a2.n));
        const int x = u + a1.r1 * k2;
        const int y = (col / a2.r2) + a2.r1 * (col % a2.r2);
        const int z = (p / a3.r2) + a3.r1 * (p % a3.r2);
        rho[((size_t)x * a2.n + y) * a3.n + z] = scale * rhot[i];
    }
}

__global__ void k_relayout_v(const double *__restrict__ v, double *__restrict__ vt, QmAxis a1, QmAxis a2, QmAxis a3,
                             double scale)
{
    // vt[p][col][j][u][e] = scale * v[x = u + r1*(2j+e)][y(col)][z(p)]   (pairs; fft_phases.cuh VLayout)
    const int r2e = a1.r2 + (a1.r2 & 1), colsz = a1.r1 * r2e;
    const size_t total = (size_t)a3.n * a2.n * colsz;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int e = (int)(i % colsz);
        const int u = (e >> 1) % a1.r1, k2 = 2 * ((e >> 1) / a1.r1) + (e & 1);
        const int col = (int)((i / colsz) % a2.n);
        const int p = (int)(i / ((size_t)colsz * a2.n));
        const int x = u + a1.r1 * k2;
        const int y = (col / a2.r2) + a2.r1 * (col % a2.r2);
        const int z = (p / a3.r2) + a3.r1 * (p % a3.r2);
        vt[i] = (k2 < a1.r2) ? scale * v[((size_t)x * a2.n + y) * a3.n + z] : 0.0;
    }
}

// Transposed box <-> natural C-order box (fft_phases.cuh BoxT): boxt[b][(p * n2 + col) * n1 + x] <-> box[b][(x * n2 + y) * n3 + z],
// p / col the transposed labels of z / y.  TO_T: natural -> transposed, else transposed -> natural.  nb boxes.
template <bool TO_T>
__global__ void k_box_relayout(const c128 *__restrict__ src, c128 *__restrict__ dst, QmAxis a1, QmAxis a2, QmAxis a3, int nb)
{
    const size_t boxsz = (size_t)a1.n * a2.n * a3.n, total = boxsz * nb;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const size_t b = i / boxsz, e = i % boxsz;                 // e indexes the transposed box
        const int x = (int)(e % a1.n), col = (int)((e / a1.n) % a2.n), p = (int)(e / ((size_t)a1.n * a2.n));
        const int y = (col / a2.r2) + a2.r1 * (col % a2.r2);
        const int z = (p / a3.r2) + a3.r1 * (p % a3.r2);
        const size_t nat = b * boxsz + ((size_t)x * a2.n + y) * a3.n + z;
        if (TO_T) dst[i] = src[nat]; else dst[nat] = src[i];
    }
}

// split-operator tables (eq. 53; reading A22)
//   field[(p * n2 + col) * n1 + x] = exp(-i dt V(x, y, z)) / N      (transposed-box layout; 1/N of the FFT pair folded in)
//   phase[g] = exp(-i dt |k+G|^2 / 4)                               (exp(-i (dt/2) T), T = 1/2 |k+G|^2)
__global__ void k_so_field(const double *__restrict__ v, c128 *__restrict__ field, QmAxis a1, QmAxis a2, QmAxis a3, double dt)
{
    const size_t boxsz = (size_t)a1.n * a2.n * a3.n;
    const double inv = 1.0 / (double)boxsz;
    for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < boxsz; e += (size_t)gridDim.x * blockDim.x) {
        const int x = (int)(e % a1.n), col = (int)((e / a1.n) % a2.n), p = (int)(e / ((size_t)a1.n * a2.n));
        const int y = (col / a2.r2) + a2.r1 * (col % a2.r2);
        const int z = (p / a3.r2) + a3.r1 * (p % a3.r2);
        double sn, cs;
        sincos(-dt * v[((size_t)x * a2.n + y) * a3.n + z], &sn, &cs);
        field[e] = c128{cs * inv, sn * inv};
    }
}
__global__ void k_so_phase(const double *__restrict__ g2, c128 *__restrict__ phase, int ng, double dt)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ng) return;
    double sn, cs;
    sincos(-dt * (0.5 * g2[i]) / 2.0, &sn, &cs);
    phase[i] = c128{cs, sn};
}

int check_handle(const qm_gspace *g, int k) {
    if (!g) return fail(QM_EINVAL, "null handle");
    if (k < 0 || k >= (int)g->kpts.size()) return fail(QM_EINVAL, "k-point index out of range");
    return check_device(g);
}

size_t w_elems_per_band(const qm_gspace *g, const KPoint *kp) {        // W is blocked by stick tile (WView)
    return ((size_t)kp->nsticks + QM_ZT - 1) / QM_ZT * QM_ZT * g->grid[2];
}
// bands per internal pass of the FFT path: the stick planes of one pass stay inside the L2 cache, so that what
// k_zinv writes is still there when the plane kernel and k_zfwd read it
int fft_chunk_bands(const qm_gspace *g, const KPoint *kp) {
    if (g->fft_chunk > 0) return g->fft_chunk;
    const size_t per_band = w_elems_per_band(g, kp) * sizeof(c128);
    const size_t budget = g->l2_bytes ? g->l2_bytes / 4 * 3 : (size_t)64 << 20;
    return (int)std::min<size_t>(64, std::max<size_t>(16, budget / std::max<size_t>(per_band, 1)));
}
int ensure_workspace(qm_gspace *g, KPoint *kp, int nb) {
    CU_TRY(kp->d_W.resize((size_t)std::min(nb, fft_chunk_bands(g, kp)) * w_elems_per_band(g, kp)));
    if (!g->fused) {
        const int n = std::min(nb, fft_chunk_bands(g, kp));
        CU_TRY(kp->d_slab.resize((size_t)gen_sub_bands(g, kp, n) * gen_slab_per_band(g, kp)));
    }
    return QM_OK;
}
struct NlPlan { int nsplit, nrows_pad, ncta2; size_t pcount; };
NlPlan nl_plan(const qm_gspace *g, const KPoint *kp) {
    NlPlan p;
    // split-K: one CTA per SM, but at least 8 K slices per split -- the reduction kernel sums the splits of an entry one
    // after the other, and on small spheres 148 two-slice splits cost more there than they save in GEMM 1
    p.nsplit = std::max(1, std::min({kp->nkc, g->sm_count * P1_OCC / std::max(1, kp->nmblk), std::max(1, kp->nkc / 8)}));
    p.nrows_pad = kp->nmblk * P1_ROWS;
    p.pcount = (size_t)p.nrows_pad * P_NB_MAX;       // sized for the widest band tile
    p.ncta2 = (int)std::min<long long>((long long)kp->ngt * kp->nic, 2LL * g->sm_count);
    return p;
}
int ensure_nonlocal_workspace(qm_gspace *g, KPoint *kp) {
    if (kp->nproj == 0) return QM_OK;
    const NlPlan p = nl_plan(g, kp);
    CU_TRY(kp->d_Ppart.resize(p.pcount * p.nsplit));
    CU_TRY(kp->d_P.resize(p.pcount));
    CU_TRY(kp->d_qt.resize((size_t)kp->nic * P2Cfg<P_NB_MAX>::Q_DOUBLES));
    CU_TRY(kp->d_part.resize((size_t)2 * p.ncta2 * P2Cfg<P_NB_MAX>::PART));
    CU_TRY(kp->d_pdesc.resize((size_t)2 * p.ncta2));
    return QM_OK;
}

// One pass of the projector pair over NB bands starting at band0, in two halves: project (P = beta^H psi, split-K
// reduction, Q = D P; needs psi_in only) and expand (out += beta Q; needs the local part of out to be there).
template <int NB>
void nonlocal_project(qm_gspace *g, KPoint *kp, const NlPlan &p, const c128 *psi_in, int nb, int band0, cudaStream_t st) {
    const int nsplit = p.nsplit, nrows_pad = p.nrows_pad;
    const size_t pcount = (size_t)nrows_pad * NB;
    g->prof.begin(QM_K_PROJ1, st);
    qm_launch_pdl(k_proj1_pipe<NB>, dim3(kp->nmblk, nsplit), dim3((P1_CW + 1) * 32), P1Cfg<NB>::SMEM, st, g->pdl,
                  (const c128 *)kp->d_beta1.p, kp->nkc, psi_in, kp->ng, nb, band0, kp->d_Ppart.p, nrows_pad, nsplit);
    g->prof.end(st);
    const int qcount = kp->nic * P2_KS * NB;
    if (16 % kp->dblock == 0 && kp->nic * P2_KS <= nrows_pad) {
        g->prof.begin(QM_K_PREDUCE, st);      // fused split-K reduction + D multiply
        qm_launch_pdl(k_reduce_dmul<NB>, dim3((kp->nic * P2_KS) / 16), dim3(16 * NB), 0, st, g->pdl, (const c128 *)kp->d_Ppart.p, nsplit,
                      nrows_pad, (const double *)kp->d_D.p, kp->dblock, kp->nproj, kp->d_qt.p);
        g->prof.end(st);
        g->launches += 2;
    } else {
        g->prof.begin(QM_K_PREDUCE, st);
        k_reduce_p2<<<(unsigned)((pcount + 255) / 256), 256, 0, st>>>(kp->d_Ppart.p, nsplit, (int)pcount, kp->d_P.p);
        g->prof.end(st);
        g->prof.begin(QM_K_DMUL, st);
        k_dmul_tiles<NB><<<(qcount + 255) / 256, 256, 0, st>>>(kp->d_D.p, kp->dblock, kp->nproj, kp->nic, kp->d_P.p,
                                                               kp->d_qt.p);
        g->prof.end(st);
        g->launches += 3;
    }
}
template <int NB>
void nonlocal_expand(qm_gspace *g, KPoint *kp, const NlPlan &p, c128 *out, int nb, int band0, cudaStream_t st) {
    const int ncta2 = p.ncta2;
    g->prof.begin(QM_K_PROJ2, st);
    qm_launch_pdl(k_proj2_sk<NB>, dim3(ncta2), dim3((P2_CW + 1) * 32), P2Cfg<NB>::SMEM, st, g->pdl, (const c128 *)kp->d_beta2.p, kp->nic,
                  kp->ngt, (const double *)kp->d_qt.p, kp->ng, nb, band0, out, kp->d_part.p, kp->d_pdesc.p);
    qm_launch_pdl(k_proj2_fixup<NB>, dim3(2 * ncta2), dim3(256), 0, st, g->pdl, (const c128 *)kp->d_part.p, (const int *)kp->d_pdesc.p,
                  2 * ncta2, kp->ng, nb, band0, out);
    g->prof.end(st);
    g->launches += 2;
}
// 32-band passes while more than 16 bands remain (beta is streamed once per pass), then one 16-band pass
inline bool pass_is_32(int nb, int band0) { return nb - band0 > P_NB; }
void nl_project(qm_gspace *g, KPoint *kp, const NlPlan &p, const c128 *psi_in, int nb, int band0, cudaStream_t st) {
    if (pass_is_32(nb, band0)) nonlocal_project<32>(g, kp, p, psi_in, nb, band0, st);
    else nonlocal_project<16>(g, kp, p, psi_in, nb, band0, st);
}
void nl_expand(qm_gspace *g, KPoint *kp, const NlPlan &p, c128 *out, int nb, int band0, cudaStream_t st) {
    if (pass_is_32(nb, band0)) nonlocal_expand<32>(g, kp, p, out, nb, band0, st);
    else nonlocal_expand<16>(g, kp, p, out, nb, band0, st);
}

// The whole apply: local part (FFT path) and projectors.  The first pass's projection needs psi_in only, so it runs on
// the k-point's side stream beside the FFT path (fork / join by events: the tails of the FFT kernels and of GEMM 1 fill each
// other's idle SMs; also valid under stream capture); everything else is ordered on `st`.
int run_local(qm_gspace *g, KPoint *kp, const c128 *in, c128 *out, int nb, int kind, cudaStream_t st);
int run_apply(qm_gspace *g, KPoint *kp, const c128 *psi_in, c128 *out, int nb, cudaStream_t st) {
    if (kp->nproj == 0) return run_local(g, kp, psi_in, out, nb, 0, st);
    const NlPlan p = nl_plan(g, kp);
    // Not while the per-kernel profiler is on: its event pairs would time kernels that share the device.  Measured at cfg5
    // (beta 1.1 GB, streamed beside the stick planes the FFT kernels hand each other through L2): 20.3-20.8 k band-applies/s
    // with the overlap, 20.1-20.4 k without; +4 % end to end; cfg1 27 -> 21 us per apply, cfg3 +10 %, cfg4 +2.5 %.
    const bool overlap = g->nl_overlap && kp->side_stream != nullptr && !g->prof.on;
    if (overlap) {
        CU_TRY(cudaEventRecord(kp->ev_fork, st));
        CU_TRY(cudaStreamWaitEvent(kp->side_stream, kp->ev_fork, 0));
        nl_project(g, kp, p, psi_in, nb, 0, kp->side_stream);
        CU_TRY(cudaEventRecord(kp->ev_join, kp->side_stream));
    }
    const int rc = run_local(g, kp, psi_in, out, nb, 0, st);
    if (overlap) CU_TRY(cudaStreamWaitEvent(st, kp->ev_join, 0));       // join even if the local part failed (stream capture)
    if (rc) return rc;
    if (!overlap) nl_project(g, kp, p, psi_in, nb, 0, st);
    nl_expand(g, kp, p, out, nb, 0, st);
    for (int band0 = pass_is_32(nb, 0) ? 32 : 16; band0 < nb; band0 += pass_is_32(nb, band0) ? 32 : 16) {
        nl_project(g, kp, p, psi_in, nb, band0, st);
        nl_expand(g, kp, p, out, nb, band0, st);
    }
    CU_TRY(cudaGetLastError());
    return QM_OK;
}

// the local part of the path for nb bands, in passes of fft_chunk_bands (stick planes stay L2 resident)
//   kind 0: H apply (V real, kinetic gather)   kind 1: split-operator step (phases + complex field)
int run_local(qm_gspace *g, KPoint *kp, const c128 *in, c128 *out, int nb, int kind, cudaStream_t st) {
    const int chunk = fft_chunk_bands(g, kp);
    for (int b0 = 0; b0 < nb; b0 += chunk) {
        const int n = std::min(chunk, nb - b0);
        const c128 *pin = in + (size_t)b0 * kp->ng;
        c128 *pout = out + (size_t)b0 * kp->ng;
        int rc;
        PlaneArgs a;
        if (kind == 0) {
            rc = dispatch_zinv<false>(g, kp, pin, nullptr, kp->d_W.p, n, st); if (rc) return rc;
            rc = dispatch_plane<0>(g, kp, kp->d_W.p, n, a, st); if (rc) return rc;
            rc = dispatch_zfwd<GM_KINETIC>(g, kp, kp->d_W.p, pin, pout, n, 1.0, st); if (rc) return rc;
        } else {
            a.box2 = g->d_sofield.p;
            rc = dispatch_zinv<true>(g, kp, pin, kp->d_sophase.p, kp->d_W.p, n, st); if (rc) return rc;
            rc = dispatch_plane<4>(g, kp, kp->d_W.p, n, a, st); if (rc) return rc;
            rc = dispatch_zfwd<GM_PHASE>(g, kp, kp->d_W.p, kp->d_sophase.p, pout, n, 1.0, st); if (rc) return rc;
        }
    }
    return QM_OK;
}

}  // namespace

extern "C" {

QM_API const char *qm_last_error(void) { return qm_g_err.c_str(); }
QM_API const char *qm_version(void) { return "qm_hpsi 0.2 (sm_100a)"; }

QM_API int qm_fft_size_supported(int n) { return qm_find_size(n) ? 1 : 0; }

QM_API int qm_gspace_create(const double *lattice_bohr, double ecutwfc_ry, const int *fft_grid,
                     const double *kpts_cryst, int nk, qm_gspace **out)
{
    if (!lattice_bohr || !fft_grid || !out || nk < 1 || !(ecutwfc_ry > 0.0))
        return fail(QM_EINVAL, "qm_gspace_create: bad argument");
    if (!kpts_cryst && nk != 1) return fail(QM_EINVAL, "qm_gspace_create: kpts_cryst is NULL with nk > 1");
    *out = nullptr;
    for (int i = 0; i < 3; ++i)
        if (!qm_find_size(fft_grid[i])) return fail(QM_EGRID, "unsupported FFT length " + std::to_string(fft_grid[i]));
    int dev = 0, count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || count == 0)
        return fail(QM_ECUDA, "no CUDA device (there is no CPU fallback)");
    qm_gspace *g = new (std::nothrow) qm_gspace();
    if (!g) return fail(QM_ENOMEM, "host allocation failed");
    std::memcpy(g->lattice, lattice_bohr, sizeof(g->lattice));
    qm_reciprocal(g->lattice, g->recip);
    g->ecut = ecutwfc_ry;
    for (int i = 0; i < 3; ++i) { g->grid[i] = fft_grid[i]; g->ax[i] = qm_make_axis(*qm_find_size(fft_grid[i])); }
    int rc = QM_OK;
    auto bail = [&](int code) { delete g; return code; };
    {
        int l2 = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&g->sm_count, cudaDevAttrMultiProcessorCount, dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&g->max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev);
        if (e != cudaSuccess) { fail(QM_ECUDA, cudaGetErrorString(e)); return bail(QM_ECUDA); }
        g->device = dev;
        g->l2_bytes = (size_t)std::max(l2, 0);
    }
    for (int a = 0; a < 3; ++a) {
        const int n = g->grid[a];
        std::vector<c128> tw(n);
        for (int j = 0; j < n; ++j) {
            // exact octant symmetries first, long double elsewhere
            const long double ang = -2.0L * 3.14159265358979323846264338327950288L * (long double)j / (long double)n;
            double c = (double)cosl(ang), s = (double)sinl(ang);
            if ((4 * j) % n == 0) {
                const int q = (4 * j) / n;
                const double cc[4] = {1, 0, -1, 0}, ss[4] = {0, -1, 0, 1};
                c = cc[q]; s = ss[q];
            }
            tw[j] = c128{c, s};
        }
        cudaError_t e = g->d_tw[a].upload(tw);
        if (e != cudaSuccess) { fail(QM_ECUDA, cudaGetErrorString(e)); return bail(QM_ECUDA); }
    }
    for (int ik = 0; ik < nk; ++ik) {
        KPoint *kp = new (std::nothrow) KPoint();
        if (!kp) { fail(QM_ENOMEM, "host allocation failed"); return bail(QM_ENOMEM); }
        g->kpts.push_back(kp);
        for (int i = 0; i < 3; ++i) kp->k[i] = kpts_cryst ? kpts_cryst[3 * ik + i] : 0.0;
        rc = build_kpoint(g, kp);
        if (rc != QM_OK) return bail(rc);
    }
    // The fused plane kernel takes the box when x and y share one line factorisation (n1 == n2 <= 144) and the plane
    // array of every k-point fits one SM's shared memory; every other legal box goes through the unfused passes.
    g->fused = g->grid[0] == g->grid[1] && g->grid[0] <= kQmFusedMax;
    if (g->fused)
        for (const KPoint *kp : g->kpts)
            if (plane_smem(g, kp, 1) > (size_t)g->max_smem) g->fused = false;
    if (const char *e = getenv("QM_FORCE_UNFUSED")) if (atoi(e) > 0) g->fused = false;
    if (const char *e = getenv("QM_NL_OVERLAP")) g->nl_overlap = atoi(e) != 0;
    if (const char *e = getenv("QM_PDL")) g->pdl = atoi(e) != 0;
    rc = prepare_kernels(g);
    if (rc != QM_OK) return bail(rc);
    if (const char *e = getenv("QM_Z_CTA_PER_SM")) g->z_cta_per_sm = std::max(1, atoi(e));
    if (const char *e = getenv("QM_PLANE_CTAS")) g->plane_ctas_per_sm = std::max(0, atoi(e));
    if (const char *e = getenv("QM_FFT_CHUNK")) g->fft_chunk = std::max(0, atoi(e));
    *out = g;
    return QM_OK;
}

QM_API int qm_gspace_destroy(qm_gspace *g) { delete g; return QM_OK; }

QM_API int qm_gspace_num_k(const qm_gspace *g, int *nk) {
    if (!g || !nk) return fail(QM_EINVAL, "null argument");
    *nk = (int)g->kpts.size(); return QM_OK;
}
static int check_k(const qm_gspace *g, int k) {
    if (!g) return fail(QM_EINVAL, "null handle");
    if (k < 0 || k >= (int)g->kpts.size()) return fail(QM_EINVAL, "k-point index out of range");
    return QM_OK;
}
QM_API int qm_gspace_num_g(const qm_gspace *g, int k, int *ng) {
    int rc = check_k(g, k); if (rc) return rc;
    if (!ng) return fail(QM_EINVAL, "null argument");
    *ng = g->kpts[k]->ng; return QM_OK;
}
QM_API int qm_gspace_num_sticks(const qm_gspace *g, int k, int *nsticks, int *nxcols) {
    int rc = check_k(g, k); if (rc) return rc;
    if (nsticks) *nsticks = g->kpts[k]->nsticks;
    if (nxcols) *nxcols = g->kpts[k]->nx;
    return QM_OK;
}
QM_API int qm_gspace_get_index_map(const qm_gspace *g, int k, int32_t *idx_host) {
    int rc = check_k(g, k); if (rc) return rc;
    if (!idx_host) return fail(QM_EINVAL, "null argument");
    std::memcpy(idx_host, g->kpts[k]->idx.data(), g->kpts[k]->idx.size() * sizeof(int32_t)); return QM_OK;
}
QM_API int qm_gspace_get_miller(const qm_gspace *g, int k, int32_t *m_host) {
    int rc = check_k(g, k); if (rc) return rc;
    if (!m_host) return fail(QM_EINVAL, "null argument");
    std::memcpy(m_host, g->kpts[k]->miller.data(), g->kpts[k]->miller.size() * sizeof(int32_t)); return QM_OK;
}
QM_API int qm_gspace_get_g2(const qm_gspace *g, int k, double *g2_host) {
    int rc = check_k(g, k); if (rc) return rc;
    if (!g2_host) return fail(QM_EINVAL, "null argument");
    std::memcpy(g2_host, g->kpts[k]->g2.data(), g->kpts[k]->g2.size() * sizeof(double)); return QM_OK;
}
QM_API int qm_gspace_alias_free(const qm_gspace *g, int k, int *flag) {
    int rc = check_k(g, k); if (rc) return rc;
    if (!flag) return fail(QM_EINVAL, "null argument");
    *flag = 1;
    for (int i = 0; i < 3; ++i) if (4 * g->kpts[k]->mmax[i] + 1 > g->grid[i]) *flag = 0;
    return QM_OK;
}

QM_API int qm_set_vloc(qm_gspace *g, const double *V_r_dev, void *stream) {
    if (!g || !V_r_dev) return fail(QM_EINVAL, "qm_set_vloc: null argument");
    int rc = check_device(g); if (rc) return rc;
    const size_t n = (size_t)g->grid[0] * g->grid[1] * g->grid[2];
    const size_t r2e = (size_t)g->ax[0].r2 + (g->ax[0].r2 & 1);
    CU_TRY(g->d_vt.resize((size_t)g->grid[2] * g->grid[1] * g->ax[0].r1 * r2e));
    k_relayout_v<<<g->sm_count * 4, 256, 0, (cudaStream_t)stream>>>(V_r_dev, g->d_vt.p, g->ax[0], g->ax[1], g->ax[2],
                                                                   1.0 / (double)n);
    g->launches++;
    CU_TRY(cudaGetLastError());
    g->v_set = true;
    return QM_OK;
}

QM_API int qm_set_nonlocal(qm_gspace *g, int k, const qm_c128 *beta_kG_dev, int nproj, const double *D_dev, int d_block,
                    void *stream) {
    int rc = check_handle(g, k); if (rc) return rc;
    KPoint *kp = g->kpts[k];
    if (nproj < 0) return fail(QM_EINVAL, "qm_set_nonlocal: nproj < 0");
    if (kp->nl_set && (nproj != kp->nproj || (nproj > 0 && d_block != kp->dblock))) kp->ws_gen++;   // batch plans of this k go stale
    if (nproj == 0) { kp->nproj = 0; kp->nl_set = true; return QM_OK; }
    if (!beta_kG_dev || !D_dev || d_block <= 0 || nproj % d_block != 0)
        return fail(QM_EINVAL, "qm_set_nonlocal: bad beta / D / d_block");
    cudaStream_t st = (cudaStream_t)stream;
    const int nmblk = (nproj + P1_ROWS - 1) / P1_ROWS, nkc = (kp->ng + P1_KS - 1) / P1_KS;
    const int ngt = (kp->ng + P2_G - 1) / P2_G, nic = (nproj + P2_KS - 1) / P2_KS;
    CU_TRY(kp->d_beta1.resize((size_t)nmblk * nkc * P1_ROWS * P1_KS));
    CU_TRY(kp->d_beta2.resize((size_t)ngt * nic * P2_KS * P2_G));
    const size_t dcount = (size_t)nproj * d_block;
    CU_TRY(kp->d_D.resize(dcount));
    const c128 *src = reinterpret_cast<const c128 *>(beta_kG_dev);
    k_tile_beta1<<<g->sm_count * 8, 256, 0, st>>>(src, kp->ng, nproj, kp->d_beta1.p, nmblk, nkc);
    k_tile_beta2<<<g->sm_count * 8, 256, 0, st>>>(src, kp->ng, nproj, kp->d_beta2.p, ngt, nic);
    g->launches += 2;
    CU_TRY(cudaGetLastError());
    CU_TRY(cudaMemcpyAsync(kp->d_D.p, D_dev, dcount * sizeof(double), cudaMemcpyDeviceToDevice, st));
    if (!kp->side_stream) {
        int prio_lo = 0, prio_hi = 0;                      // lowest priority: kernels of the caller's stream get free SMs first
        CU_TRY(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
        CU_TRY(cudaStreamCreateWithPriority(&kp->side_stream, cudaStreamNonBlocking, prio_lo));
        CU_TRY(cudaEventCreateWithFlags(&kp->ev_fork, cudaEventDisableTiming));
        CU_TRY(cudaEventCreateWithFlags(&kp->ev_join, cudaEventDisableTiming));
    }
    kp->nproj = nproj; kp->dblock = d_block; kp->nl_set = true;
    kp->nmblk = nmblk; kp->nkc = nkc; kp->ngt = ngt; kp->nic = nic;
    return ensure_nonlocal_workspace(g, kp);        // projector workspaces do not depend on nbands: sized here, once
}

QM_API int qm_reserve(qm_gspace *g, int k, int nbands) {
    int rc = check_handle(g, k); if (rc) return rc;
    if (nbands <= 0) return fail(QM_EINVAL, "qm_reserve: nbands <= 0");
    KPoint *kp = g->kpts[k];
    rc = ensure_workspace(g, kp, nbands); if (rc) return rc;
    return ensure_nonlocal_workspace(g, kp);
}

QM_API int qm_apply_h(qm_gspace *g, const qm_c128 *psi_in_dev, qm_c128 *psi_out_dev, int nbands, int k, void *stream) {
    int rc = check_handle(g, k); if (rc) return rc;
    if (!psi_in_dev || !psi_out_dev || nbands <= 0) return fail(QM_EINVAL, "qm_apply_h: bad argument");
    KPoint *kp = g->kpts[k];
    if (!g->v_set) return fail(QM_ENOTSET, "qm_apply_h before qm_set_vloc");
    if (!kp->nl_set) return fail(QM_ENOTSET, "qm_apply_h before qm_set_nonlocal for this k");
    const c128 *in = reinterpret_cast<const c128 *>(psi_in_dev);
    c128 *out = reinterpret_cast<c128 *>(psi_out_dev);
    const size_t bytes = (size_t)nbands * kp->ng * sizeof(c128);
    const char *a = (const char *)in, *b = (const char *)out;
    if (a < b + bytes && b < a + bytes) return fail(QM_EINVAL, "qm_apply_h: psi_in and psi_out overlap");
    cudaStream_t st = (cudaStream_t)stream;
    rc = ensure_workspace(g, kp, nbands); if (rc) return rc;
    return run_apply(g, kp, in, out, nbands, st);
}

QM_API int qm_split_operator_set(qm_gspace *g, const double *V_r_dev, double dt, void *stream) {
    if (!g || !V_r_dev) return fail(QM_EINVAL, "qm_split_operator_set: null argument");
    int rc = check_device(g); if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)g->grid[0] * g->grid[1] * g->grid[2];
    CU_TRY(g->d_sofield.resize(n));
    k_so_field<<<g->sm_count * 4, 256, 0, st>>>(V_r_dev, g->d_sofield.p, g->ax[0], g->ax[1], g->ax[2], dt);
    g->launches++;
    for (KPoint *kp : g->kpts) {
        CU_TRY(kp->d_sophase.resize((size_t)kp->ng));
        k_so_phase<<<(kp->ng + 255) / 256, 256, 0, st>>>(kp->d_g2.p, kp->d_sophase.p, kp->ng, dt);
        g->launches++;
    }
    CU_TRY(cudaGetLastError());
    g->so_set = true; g->so_dt = dt;
    return QM_OK;
}

QM_API int qm_split_operator_propagate(qm_gspace *g, int k, const qm_c128 *psi_in_dev, qm_c128 *psi_out_dev, int nbands,
                                       void *stream) {
    int rc = check_handle(g, k); if (rc) return rc;
    if (!psi_in_dev || !psi_out_dev || nbands <= 0) return fail(QM_EINVAL, "qm_split_operator_propagate: bad argument");
    if (!g->so_set) return fail(QM_ENOTSET, "qm_split_operator_propagate before qm_split_operator_set");
    KPoint *kp = g->kpts[k];
    const c128 *in = reinterpret_cast<const c128 *>(psi_in_dev);
    c128 *out = reinterpret_cast<c128 *>(psi_out_dev);
    const size_t bytes = (size_t)nbands * kp->ng * sizeof(c128);
    const char *a = (const char *)in, *b = (const char *)out;
    if (a < b + bytes && b < a + bytes) return fail(QM_EINVAL, "qm_split_operator_propagate: psi_in and psi_out overlap");
    rc = ensure_workspace(g, kp, nbands); if (rc) return rc;
    return run_local(g, kp, in, out, nbands, 1, (cudaStream_t)stream);
}

QM_API int qm_mtxel_create(qm_gspace *g, int k_bra, int k_ket, double ecut_eps_ry, qm_mtxel **out) {
    int rc = check_handle(g, k_bra); if (rc) return rc;
    rc = check_handle(g, k_ket); if (rc) return rc;
    if (!out || !(ecut_eps_ry > 0.0)) return fail(QM_EINVAL, "qm_mtxel_create: bad argument");
    *out = nullptr;
    qm_mtxel *m = new (std::nothrow) qm_mtxel();
    if (!m) return fail(QM_ENOMEM, "host allocation failed");
    m->g = g; m->k_bra = k_bra; m->k_ket = k_ket;
    for (int i = 0; i < 3; ++i) m->sph.k[i] = g->kpts[k_bra]->k[i] - g->kpts[k_ket]->k[i];      // q = (k+q) - k
    m->sph.ecut_override = ecut_eps_ry;
    rc = build_kpoint(g, &m->sph, true);
    if (rc == QM_OK && g->fused && plane_smem(g, &m->sph, 1) > (size_t)g->max_smem)
        rc = fail(QM_EGRID, "plane working set of the epsilon sphere exceeds shared memory");
    if (rc != QM_OK) { delete m; return rc; }
    *out = m;
    return QM_OK;
}
QM_API int qm_mtxel_destroy(qm_mtxel *m) { delete m; return QM_OK; }
QM_API int qm_mtxel_num_g(const qm_mtxel *m, int *ng) {
    if (!m || !ng) return fail(QM_EINVAL, "null argument");
    *ng = m->sph.ng; return QM_OK;
}
QM_API int qm_mtxel_get_miller(const qm_mtxel *m, int32_t *miller_host) {
    if (!m || !miller_host) return fail(QM_EINVAL, "null argument");
    std::memcpy(miller_host, m->sph.miller.data(), m->sph.miller.size() * sizeof(int32_t)); return QM_OK;
}
QM_API int qm_mtxel_get_index_map(const qm_mtxel *m, int32_t *idx_host) {
    if (!m || !idx_host) return fail(QM_EINVAL, "null argument");
    std::memcpy(idx_host, m->sph.idx.data(), m->sph.idx.size() * sizeof(int32_t)); return QM_OK;
}

// scatter + backward FFT of `n` states of k-point kp into transposed boxes (unnormalised synthesis, reading A5/A20)
static int synth_boxes(qm_gspace *g, KPoint *kp, const c128 *psi, int n, c128 *boxes, cudaStream_t st) {
    const size_t boxsz = (size_t)g->grid[0] * g->grid[1] * g->grid[2];
    int rc = ensure_workspace(g, kp, n); if (rc) return rc;
    const int chunk = fft_chunk_bands(g, kp);
    for (int b0 = 0; b0 < n; b0 += chunk) {
        const int c = std::min(chunk, n - b0);
        rc = dispatch_zinv<false>(g, kp, psi + (size_t)b0 * kp->ng, nullptr, kp->d_W.p, c, st); if (rc) return rc;
        PlaneArgs a; a.box = boxes + (size_t)b0 * boxsz; a.scale = 1.0;
        rc = dispatch_plane<1>(g, kp, kp->d_W.p, c, a, st); if (rc) return rc;
    }
    return QM_OK;
}

QM_API int qm_matrix_elements(qm_mtxel *m, const qm_c128 *bra_dev, int nbra, const qm_c128 *ket_dev, int nket,
                              qm_c128 *out_dev, void *stream) {
    if (!m || !bra_dev || !ket_dev || !out_dev || nbra <= 0 || nket <= 0) return fail(QM_EINVAL, "qm_matrix_elements: bad argument");
    qm_gspace *g = m->g;
    int rc = check_device(g); if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    KPoint *kb = g->kpts[m->k_bra], *kk = g->kpts[m->k_ket];
    const size_t boxsz = (size_t)g->grid[0] * g->grid[1] * g->grid[2];
    const size_t wpair = w_elems_per_band(g, &m->sph);
    // bras per pass: the stick planes of (bras x nket) pairs within ~512 MB
    const size_t cap = ((size_t)512 << 20) / sizeof(c128);
    const int bpass = (int)std::max<size_t>(1, std::min<size_t>((size_t)nbra, cap / std::max<size_t>(1, wpair * nket)));
    CU_TRY(m->d_ketbox.resize(boxsz * nket));
    CU_TRY(m->d_brabox.resize(boxsz * bpass));
    CU_TRY(m->d_Wp.resize(wpair * bpass * nket));
    rc = synth_boxes(g, kk, reinterpret_cast<const c128 *>(ket_dev), nket, m->d_ketbox.p, st); if (rc) return rc;
    c128 *out = reinterpret_cast<c128 *>(out_dev);
    for (int a0 = 0; a0 < nbra; a0 += bpass) {
        const int na = std::min(bpass, nbra - a0);
        rc = synth_boxes(g, kb, reinterpret_cast<const c128 *>(bra_dev) + (size_t)a0 * kb->ng, na, m->d_brabox.p, st);
        if (rc) return rc;
        // pair (a, b): forward transform of phi_a(r) conj(phi_b(r)) pruned to the epsilon sphere, then
        // M_ab(G) = conj(F(G)) / N  = (1/N) sum_r conj(phi_a) phi_b exp(+i G.r)          (eq. 56, reading A21)
        PlaneArgs pa; pa.box = m->d_brabox.p; pa.box2 = m->d_ketbox.p; pa.npair2 = nket;
        rc = dispatch_plane<2>(g, &m->sph, m->d_Wp.p, na * nket, pa, st); if (rc) return rc;
        rc = dispatch_zfwd<GM_CONJ>(g, &m->sph, m->d_Wp.p, nullptr, out + (size_t)a0 * nket * m->sph.ng, na * nket,
                                    1.0 / (double)boxsz, st);
        if (rc) return rc;
    }
    return QM_OK;
}

QM_API int qm_batch_plan_create(qm_gspace *g, int nitems, const int *k, const qm_c128 *const *psi_in_dev,
                                qm_c128 *const *psi_out_dev, const int *nbands, qm_batch_plan **out) {
    if (!g || !k || !psi_in_dev || !psi_out_dev || !nbands || !out || nitems <= 0)
        return fail(QM_EINVAL, "qm_batch_plan_create: bad argument");
    *out = nullptr;
    int rc = check_device(g); if (rc) return rc;
    if (g->prof.on) return fail(QM_EINVAL, "qm_batch_plan_create: switch the per-kernel profiler off first");
    for (int i = 0; i < nitems; ++i) {              // nothing may allocate while the graph is being captured
        rc = check_handle(g, k[i]); if (rc) return rc;
        if (nbands[i] <= 0 || !psi_in_dev[i] || !psi_out_dev[i]) return fail(QM_EINVAL, "qm_batch_plan_create: bad item");
        rc = qm_reserve(g, k[i], nbands[i]); if (rc) return rc;
    }
    constexpr int MAXB = 16;
    const int nbranch = std::min<int>(MAXB, (int)g->kpts.size());
    cudaStream_t s0 = nullptr, sb[MAXB] = {nullptr};
    cudaEvent_t fork = nullptr, join[MAXB] = {nullptr};
    bool used[MAXB] = {false};
    qm_batch_plan *p = new (std::nothrow) qm_batch_plan();
    if (!p) return fail(QM_ENOMEM, "host allocation failed");
    p->g = g;
    auto cleanup = [&]() {
        if (fork) cudaEventDestroy(fork);
        for (int b = 0; b < nbranch; ++b) { if (join[b]) cudaEventDestroy(join[b]); if (sb[b]) cudaStreamDestroy(sb[b]); }
        if (s0) cudaStreamDestroy(s0);
    };
    cudaError_t e = cudaStreamCreateWithFlags(&s0, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&fork, cudaEventDisableTiming);
    for (int b = 0; b < nbranch && e == cudaSuccess; ++b) {
        e = cudaStreamCreateWithFlags(&sb[b], cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&join[b], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) { cleanup(); delete p; return fail(QM_ECUDA, cudaGetErrorString(e)); }
    const unsigned long long l0 = g->launches;
    e = cudaStreamBeginCapture(s0, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) { cleanup(); delete p; return fail(QM_ECUDA, cudaGetErrorString(e)); }
    // k-points have their own work spaces: one branch per k-point (modulo MAXB), items of a branch in list order
    rc = QM_OK;
    e = cudaEventRecord(fork, s0);
    for (int i = 0; i < nitems && rc == QM_OK && e == cudaSuccess; ++i) {
        const int b = k[i] % nbranch;
        if (!used[b]) { e = cudaStreamWaitEvent(sb[b], fork, 0); used[b] = true; if (e != cudaSuccess) break; }
        rc = qm_apply_h(g, psi_in_dev[i], psi_out_dev[i], nbands[i], k[i], sb[b]);
    }
    for (int b = 0; b < nbranch && e == cudaSuccess; ++b)
        if (used[b]) { e = cudaEventRecord(join[b], sb[b]); if (e == cudaSuccess) e = cudaStreamWaitEvent(s0, join[b], 0); }
    cudaGraph_t graph = nullptr;
    const cudaError_t e2 = cudaStreamEndCapture(s0, &graph);
    p->launches = g->launches - l0;
    g->launches = l0;                               // capturing launched nothing
    for (int i = 0; i < nitems; ++i) {
        bool seen = false;
        for (const auto &kg : p->gens) seen = seen || kg.first == k[i];
        if (!seen) p->gens.emplace_back(k[i], g->kpts[k[i]]->ws_gen);
    }
    if (rc == QM_OK && (e != cudaSuccess || e2 != cudaSuccess)) rc = fail(QM_ECUDA, cudaGetErrorString(e != cudaSuccess ? e : e2));
    if (rc == QM_OK) {
        p->graph = graph;
        const cudaError_t e3 = cudaGraphInstantiate(&p->exec, graph, 0);
        if (e3 != cudaSuccess) rc = fail(QM_ECUDA, cudaGetErrorString(e3));
    } else if (graph) cudaGraphDestroy(graph);
    cleanup();
    if (rc != QM_OK) { delete p; return rc; }
    *out = p;
    return QM_OK;
}
QM_API int qm_batch_plan_launch(qm_batch_plan *p, void *stream) {
    if (!p || !p->exec) return fail(QM_EINVAL, "qm_batch_plan_launch: null plan");
    int rc = check_device(p->g); if (rc) return rc;
    for (const auto &kg : p->gens)
        if (p->g->kpts[kg.first]->ws_gen != kg.second)
            return fail(QM_EINVAL, "qm_batch_plan_launch: stale plan -- a work space of k-point " + std::to_string(kg.first) +
                                   " was re-allocated by a larger call, or its projector shape changed, after the plan "
                                   "was created; destroy the plan and create it again");
    CU_TRY(cudaGraphLaunch(p->exec, (cudaStream_t)stream));
    p->g->launches += p->launches;
    return QM_OK;
}
QM_API int qm_batch_plan_destroy(qm_batch_plan *p) { delete p; return QM_OK; }

QM_API int qm_host_synchronize(qm_gspace *g) {
    if (!g) return fail(QM_EINVAL, "null handle");
    if (!g->pipe.init) return QM_OK;
    int rc = check_device(g); if (rc) return rc;
    CU_TRY(cudaStreamSynchronize(g->pipe.s_in));
    CU_TRY(cudaStreamSynchronize(g->pipe.s_out));
    return QM_OK;
}

QM_API int qm_apply_h_host_async(qm_gspace *g, const qm_c128 *psi_in_host, qm_c128 *psi_out_host, int nbands, int k,
                                 void *stream) {
    int rc = check_handle(g, k); if (rc) return rc;
    if (!psi_in_host || !psi_out_host || nbands <= 0) return fail(QM_EINVAL, "qm_apply_h_host: bad argument");
    KPoint *kp = g->kpts[k];
    HostPipe &hp = g->pipe;
    if (!hp.init) {
        CU_TRY(cudaStreamCreateWithFlags(&hp.s_in, cudaStreamNonBlocking));
        CU_TRY(cudaStreamCreateWithFlags(&hp.s_out, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CU_TRY(cudaEventCreateWithFlags(&hp.in_ready[i], cudaEventDisableTiming));
            CU_TRY(cudaEventCreateWithFlags(&hp.compute_done[i], cudaEventDisableTiming));
            CU_TRY(cudaEventCreateWithFlags(&hp.out_done[i], cudaEventDisableTiming));
        }
        hp.init = true;
    }
    const int sl = hp.slot;
    hp.slot ^= 1;
    const size_t count = (size_t)nbands * kp->ng;
    if (hp.in[sl].n < count || hp.out[sl].n < count) {      // growing a slot: nothing may still be using it
        rc = qm_host_synchronize(g); if (rc) return rc;
        CU_TRY(cudaStreamSynchronize((cudaStream_t)stream));
        CU_TRY(hp.in[sl].resize(count));
        CU_TRY(hp.out[sl].resize(count));
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (hp.used[sl]) CU_TRY(cudaStreamWaitEvent(hp.s_in, hp.compute_done[sl], 0));    // slot's last apply has read it
    CU_TRY(cudaMemcpyAsync(hp.in[sl].p, psi_in_host, count * sizeof(c128), cudaMemcpyHostToDevice, hp.s_in));
    CU_TRY(cudaEventRecord(hp.in_ready[sl], hp.s_in));
    CU_TRY(cudaStreamWaitEvent(st, hp.in_ready[sl], 0));
    if (hp.used[sl]) CU_TRY(cudaStreamWaitEvent(st, hp.out_done[sl], 0));             // slot's last result has left
    rc = qm_apply_h(g, reinterpret_cast<const qm_c128 *>(hp.in[sl].p), reinterpret_cast<qm_c128 *>(hp.out[sl].p),
                    nbands, k, stream);
    if (rc) return rc;
    CU_TRY(cudaEventRecord(hp.compute_done[sl], st));
    CU_TRY(cudaStreamWaitEvent(hp.s_out, hp.compute_done[sl], 0));
    CU_TRY(cudaMemcpyAsync(psi_out_host, hp.out[sl].p, count * sizeof(c128), cudaMemcpyDeviceToHost, hp.s_out));
    CU_TRY(cudaEventRecord(hp.out_done[sl], hp.s_out));
    hp.used[sl] = true;
    return QM_OK;
}

QM_API int qm_subspace(qm_gspace *g, int k, const qm_c128 *a_dev, int na, const qm_c128 *b_dev, int nb,
                qm_c128 *s_dev, void *stream)
{
    int rc = check_handle(g, k); if (rc) return rc;
    if (!a_dev || !b_dev || !s_dev || na <= 0 || nb <= 0) return fail(QM_EINVAL, "qm_subspace: bad argument");
    KPoint *kp = g->kpts[k];
    cudaStream_t st = (cudaStream_t)stream;
    const int ntm = (na + SG_T - 1) / SG_T, ntn = (nb + SG_T - 1) / SG_T;
    const int nkc = (kp->ng + SG_KS - 1) / SG_KS;
    const int nsplit = std::max(1, std::min(nkc, g->sm_count / (ntm * ntn)));
    const int ldp = ntn * SG_T;
    const size_t plane = (size_t)ntm * SG_T * ldp;
    CU_TRY(g->d_subpart.resize(plane * nsplit));
    g->prof.begin(QM_K_SUBGEMM, st);
    k_sub_gemm<<<dim3(ntm * ntn, nsplit), (SG_CW + 1) * 32, SG_SMEM, st>>>(
        reinterpret_cast<const c128 *>(a_dev), na, reinterpret_cast<const c128 *>(b_dev), nb, kp->ng, ntn, nsplit,
        g->d_subpart.p, ldp);
    g->prof.end(st);
    g->prof.begin(QM_K_SUBREDUCE, st);
    k_sub_reduce<<<(na * nb + 255) / 256, 256, 0, st>>>(g->d_subpart.p, nsplit, plane, ldp, na, nb,
                                                       reinterpret_cast<c128 *>(s_dev));
    g->prof.end(st);
    g->launches += 2;
    CU_TRY(cudaGetLastError());
    return QM_OK;
}

// ---- qm_subspace_static: the subspace product without any device allocation (include/qm_hpsi.h) -----------------------
// For callers that cannot cudaMalloc (their own pool owns the device, a cudaMalloc would stall their other streams, or
// their memory budget is fixed when the library is loaded), the split-K partial sums of S = A^H B live in the array
// below, which is part of the library image: 2^20 complex128 = 16 MiB on every GPU that loads the library, until exit.
//
// `qm_substat_part` means two different things.  In DEVICE code (k_sub_reduce_static) it is the array.  In HOST code it
// is only a handle that stands for the array: it is NOT a device address, and a kernel that is handed
// `qm_substat_part` as a pointer argument from the host would write to a host address (a fault, or on machines where
// the GPU can reach host memory, silent corruption).  The host gets the real address with cudaGetSymbolAddress, once
// per device and with that device current (substat_setup), and passes THAT to k_sub_gemm.
static __device__ __align__(256) c128 qm_substat_part[QM_SUBSPACE_STATIC_MAX_ELEMS];

// k_sub_reduce with the partial sums read from the static array (named directly: this is device code).  Same
// summation order as k_sub_reduce, so both entry points return the same bits.
__global__ void k_sub_reduce_static(int nsplit, size_t plane, int ldp, int na, int nb, c128 *__restrict__ s_out)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= na * nb) return;
    const int i = idx / nb, j = idx % nb;
    const c128 *src = qm_substat_part + (size_t)i * ldp + j;
    double sr[4] = {0.0, 0.0, 0.0, 0.0}, si[4] = {0.0, 0.0, 0.0, 0.0};
    int s = 0;
    for (; s + 4 <= nsplit; s += 4) {
#pragma unroll
        for (int q = 0; q < 4; ++q) { const double2 v = ldg_c128(src + (size_t)(s + q) * plane); sr[q] += v.x; si[q] += v.y; }
    }
    for (; s < nsplit; ++s) { const double2 v = ldg_c128(src + (size_t)s * plane); sr[0] += v.x; si[0] += v.y; }
    s_out[idx] = c128{(sr[0] + sr[1]) + (sr[2] + sr[3]), (si[0] + si[1]) + (si[2] + si[3])};
}

namespace {
constexpr int SUBSTAT_MAX_DEVICES = 64;
struct SubStatDev { bool ready = false; c128 *part = nullptr; int sm_count = 0; };
SubStatDev substat_dev[SUBSTAT_MAX_DEVICES];
std::mutex substat_mu;

// First call on a device: the array's address ON THAT DEVICE, its SM count, and the shared-memory opt-in of the GEMM
// (function attributes are per device; no handle was necessarily created here).  None of these allocates.
int substat_setup(const SubStatDev **out) {
    int dev = -1;
    CU_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= SUBSTAT_MAX_DEVICES) return fail(QM_EINVAL, "qm_subspace_static: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(substat_mu);
    SubStatDev &d = substat_dev[dev];
    if (!d.ready) {
        c128 *ptr = nullptr;
        CU_TRY(cudaGetSymbolAddress((void **)&ptr, qm_substat_part));
        if (!ptr) return fail(QM_ECUDA, "qm_subspace_static: cudaGetSymbolAddress returned a null address");
        CU_TRY(cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, dev));
        CU_TRY(cudaFuncSetAttribute(k_sub_gemm, cudaFuncAttributeMaxDynamicSharedMemorySize, SG_SMEM));
        d.part = ptr;
        d.ready = true;
    }
    *out = &d;
    return QM_OK;
}
}  // namespace

QM_API int qm_subspace_static(const qm_c128 *a_dev, int na, const qm_c128 *b_dev, int nb, int ng, qm_c128 *s_dev,
                              void *stream)
{
    if (!a_dev || !b_dev || !s_dev || na <= 0 || nb <= 0 || ng <= 0)
        return fail(QM_EINVAL, "qm_subspace_static: bad argument");
    if (((uintptr_t)a_dev | (uintptr_t)b_dev | (uintptr_t)s_dev) & 15)
        return fail(QM_EINVAL, "qm_subspace_static: a, b and s must be 16-byte aligned");
    const long long ntm = ((long long)na + SG_T - 1) / SG_T, ntn = ((long long)nb + SG_T - 1) / SG_T;
    const long long plane_ll = ntm * SG_T * ntn * SG_T;
    if (plane_ll > (long long)QM_SUBSPACE_STATIC_MAX_ELEMS)
        return fail(QM_EINVAL, "qm_subspace_static: a block of " + std::to_string(na) + " x " + std::to_string(nb) +
                                   " states needs " + std::to_string(plane_ll) + " partial sums per K split, the static "
                                   "work space holds " + std::to_string(QM_SUBSPACE_STATIC_MAX_ELEMS) +
                                   " (e.g. 1024 x 1024); use qm_subspace for larger blocks");
    const SubStatDev *d = nullptr;
    int rc = substat_setup(&d); if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const int tiles = (int)(ntm * ntn), ldp = (int)ntn * SG_T;
    const size_t plane = (size_t)plane_ll;
    const int nkc = (ng + SG_KS - 1) / SG_KS;
    int nsplit = std::max(1, std::min(nkc, d->sm_count / tiles));                  // qm_subspace's choice ...
    nsplit = (int)std::min<size_t>((size_t)nsplit, QM_SUBSPACE_STATIC_MAX_ELEMS / plane);   // ... as far as the array holds it
    // k_sub_gemm writes every element of every [split] plane that k_sub_reduce_static reads: nothing to clear
    k_sub_gemm<<<dim3(tiles, nsplit), (SG_CW + 1) * 32, SG_SMEM, st>>>(
        reinterpret_cast<const c128 *>(a_dev), na, reinterpret_cast<const c128 *>(b_dev), nb, ng, (int)ntn, nsplit,
        d->part, ldp);
    k_sub_reduce_static<<<(na * nb + 255) / 256, 256, 0, st>>>(nsplit, plane, ldp, na, nb, reinterpret_cast<c128 *>(s_dev));
    CU_TRY(cudaGetLastError());
    return QM_OK;
}

// one term of the Taylor series: t = c * h (the next power's input), out += t
__global__ void k_taylor_axpy(const c128 *__restrict__ h, double cr, double ci, c128 *__restrict__ t, c128 *__restrict__ out,
                              size_t n, int keep_t)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const c128 x = h[i];
        const c128 v = c128{cr * x.x - ci * x.y, cr * x.y + ci * x.x};
        if (keep_t) t[i] = v;
        c128 o = out[i];
        o.x += v.x; o.y += v.y;
        out[i] = o;
    }
}

QM_API int qm_taylor_propagate(qm_gspace *g, int k, const qm_c128 *psi_in_dev, qm_c128 *psi_out_dev, int nbands, double dt,
                        int order, void *stream) {
    int rc = check_handle(g, k); if (rc) return rc;
    if (!psi_in_dev || !psi_out_dev || nbands <= 0 || order < 0) return fail(QM_EINVAL, "qm_taylor_propagate: bad argument");
    KPoint *kp = g->kpts[k];
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)nbands * kp->ng;
    CU_TRY(g->d_tay_h.resize(n));
    CU_TRY(g->d_tay_t.resize(n));
    CU_TRY(cudaMemcpyAsync(psi_out_dev, psi_in_dev, n * sizeof(c128), cudaMemcpyDeviceToDevice, st));     // r = 0 term
    const qm_c128 *src = psi_in_dev;
    for (int r = 1; r <= order; ++r) {
        rc = qm_apply_h(g, src, reinterpret_cast<qm_c128 *>(g->d_tay_h.p), nbands, k, stream); if (rc) return rc;
        // t_r = (-i dt / r) H t_{r-1}  =>  t_r = (-i dt)^r / r!  H^r psi     (eq. 52)
        k_taylor_axpy<<<g->sm_count * 8, 256, 0, st>>>(g->d_tay_h.p, 0.0, -dt / r, g->d_tay_t.p,
                                                       reinterpret_cast<c128 *>(psi_out_dev), n, r < order ? 1 : 0);
        g->launches++;
        src = reinterpret_cast<const qm_c128 *>(g->d_tay_t.p);
    }
    CU_TRY(cudaGetLastError());
    return QM_OK;
}

static size_t qm_rhot_elems(const qm_gspace *g) {
    const size_t r2e = (size_t)g->ax[0].r2 + (g->ax[0].r2 & 1);
    return (size_t)g->grid[2] * g->grid[1] * g->ax[0].r1 * r2e;
}
QM_API int qm_density_reset(qm_gspace *g, void *stream) {
    if (!g) return fail(QM_EINVAL, "null handle");
    int rc = check_device(g); if (rc) return rc;
    const size_t n = qm_rhot_elems(g);
    CU_TRY(g->d_rhot.resize(n));
    CU_TRY(cudaMemsetAsync(g->d_rhot.p, 0, n * sizeof(double), (cudaStream_t)stream));
    g->rho_open = true;
    return QM_OK;
}
QM_API int qm_density_accumulate(qm_gspace *g, int k, const qm_c128 *psi_dev, int nbands, const double *occ_dev,
                          double weight, void *stream) {
    int rc = check_handle(g, k); if (rc) return rc;
    if (!psi_dev || !occ_dev || nbands <= 0) return fail(QM_EINVAL, "qm_density_accumulate: bad argument");
    if (!g->rho_open) return fail(QM_ENOTSET, "qm_density_accumulate before qm_density_reset");
    KPoint *kp = g->kpts[k];
    cudaStream_t st = (cudaStream_t)stream;
    rc = ensure_workspace(g, kp, nbands); if (rc) return rc;
    const int chunk = fft_chunk_bands(g, kp);
    for (int b0 = 0; b0 < nbands; b0 += chunk) {        // band order is kept: the running sum stays deterministic
        const int n = std::min(chunk, nbands - b0);
        rc = dispatch_zinv<false>(g, kp, reinterpret_cast<const c128 *>(psi_dev) + (size_t)b0 * kp->ng, nullptr, kp->d_W.p, n, st);
        if (rc) return rc;
        PlaneArgs a; a.scale = weight; a.occ = occ_dev + b0; a.rhot = g->d_rhot.p;
        rc = dispatch_plane<3>(g, kp, kp->d_W.p, n, a, st); if (rc) return rc;
    }
    return QM_OK;
}
QM_API int qm_density_get(qm_gspace *g, double *rho_dev, double scale, void *stream) {
    if (!g || !rho_dev) return fail(QM_EINVAL, "qm_density_get: null argument");
    if (!g->rho_open) return fail(QM_ENOTSET, "qm_density_get before qm_density_reset");
    int rc = check_device(g); if (rc) return rc;
    k_density_out<<<g->sm_count * 4, 256, 0, (cudaStream_t)stream>>>(g->d_rhot.p, rho_dev, g->ax[0], g->ax[1], g->ax[2], scale);
    g->launches++;
    CU_TRY(cudaGetLastError());
    return QM_OK;
}

QM_API int qm_apply_h_host(qm_gspace *g, const qm_c128 *psi_in_host, qm_c128 *psi_out_host, int nbands, int k,
                           void *stream) {
    int rc = qm_apply_h_host_async(g, psi_in_host, psi_out_host, nbands, k, stream);
    if (rc) return rc;
    return qm_host_synchronize(g);
}

QM_API int qm_debug_g2r(qm_gspace *g, const qm_c128 *psi_g_dev, qm_c128 *box_r_dev, int nbands, int k, void *stream) {
    int rc = check_handle(g, k); if (rc) return rc;
    if (!psi_g_dev || !box_r_dev || nbands <= 0) return fail(QM_EINVAL, "qm_debug_g2r: bad argument");
    KPoint *kp = g->kpts[k];
    cudaStream_t st = (cudaStream_t)stream;
    const size_t boxsz = (size_t)g->grid[0] * g->grid[1] * g->grid[2];
    rc = ensure_workspace(g, kp, nbands); if (rc) return rc;
    const int chunk = fft_chunk_bands(g, kp);
    CU_TRY(g->d_boxt.resize(boxsz * std::min(chunk, nbands)));
    for (int b0 = 0; b0 < nbands; b0 += chunk) {
        const int n = std::min(chunk, nbands - b0);
        rc = dispatch_zinv<false>(g, kp, reinterpret_cast<const c128 *>(psi_g_dev) + (size_t)b0 * kp->ng, nullptr, kp->d_W.p, n, st);
        if (rc) return rc;
        PlaneArgs a; a.box = g->d_boxt.p; a.scale = 1.0 / (double)boxsz;
        rc = dispatch_plane<1>(g, kp, kp->d_W.p, n, a, st); if (rc) return rc;
        k_box_relayout<false><<<g->sm_count * 8, 256, 0, st>>>(g->d_boxt.p, reinterpret_cast<c128 *>(box_r_dev) + (size_t)b0 * boxsz,
                                                              g->ax[0], g->ax[1], g->ax[2], n);
        g->launches++;
    }
    CU_TRY(cudaGetLastError());
    return QM_OK;
}

QM_API int qm_debug_r2g(qm_gspace *g, const qm_c128 *box_r_dev, qm_c128 *psi_g_dev, int nbands, int k, void *stream) {
    int rc = check_handle(g, k); if (rc) return rc;
    if (!psi_g_dev || !box_r_dev || nbands <= 0) return fail(QM_EINVAL, "qm_debug_r2g: bad argument");
    KPoint *kp = g->kpts[k];
    cudaStream_t st = (cudaStream_t)stream;
    const size_t boxsz = (size_t)g->grid[0] * g->grid[1] * g->grid[2];
    rc = ensure_workspace(g, kp, nbands); if (rc) return rc;
    const int chunk = fft_chunk_bands(g, kp);
    CU_TRY(g->d_boxt.resize(boxsz * std::min(chunk, nbands)));
    for (int b0 = 0; b0 < nbands; b0 += chunk) {
        const int n = std::min(chunk, nbands - b0);
        k_box_relayout<true><<<g->sm_count * 8, 256, 0, st>>>(reinterpret_cast<const c128 *>(box_r_dev) + (size_t)b0 * boxsz, g->d_boxt.p,
                                                             g->ax[0], g->ax[1], g->ax[2], n);
        g->launches++;
        PlaneArgs a; a.box = g->d_boxt.p;
        rc = dispatch_plane<2>(g, kp, kp->d_W.p, n, a, st); if (rc) return rc;
        rc = dispatch_zfwd<GM_PLAIN>(g, kp, kp->d_W.p, nullptr, reinterpret_cast<c128 *>(psi_g_dev) + (size_t)b0 * kp->ng, n, 1.0, st);
        if (rc) return rc;
    }
    CU_TRY(cudaGetLastError());
    return QM_OK;
}

QM_API int qm_get_launch_count(const qm_gspace *g, unsigned long long *count) {
    if (!g || !count) return fail(QM_EINVAL, "null argument");
    *count = g->launches; return QM_OK;
}

QM_API int qm_profile_enable(qm_gspace *g, int on) {
    if (!g) return fail(QM_EINVAL, "null handle");
    g->prof.collect();
    g->prof.on = on != 0;
    return QM_OK;
}
QM_API int qm_profile_reset(qm_gspace *g) {
    if (!g) return fail(QM_EINVAL, "null handle");
    g->prof.reset();
    return QM_OK;
}
QM_API int qm_profile_read(qm_gspace *g, int kind, double *total_ms, unsigned long long *launches) {
    if (!g || kind < 0 || kind >= QM_K_COUNT) return fail(QM_EINVAL, "qm_profile_read: bad argument");
    g->prof.collect();
    if (total_ms) *total_ms = g->prof.total_ms[kind];
    if (launches) *launches = g->prof.count[kind];
    return QM_OK;
}
QM_API const char *qm_kernel_name(int kind) {
    static const char *names[QM_K_COUNT] = {"k_zinv", "k_plane", "k_zfwd", "k_proj1", "k_reduce_p", "k_dmul",
                                            "k_proj2", "k_sub_gemm", "k_sub_reduce", "k_gen_y", "k_gen_x"};
    return (kind >= 0 && kind < QM_K_COUNT) ? names[kind] : "?";
}

QM_API int qm_probe_fp64_tensor_peak(double *tflops_dmma, double *tflops_dfma) {
    int dev = 0, sms = 0, count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || count == 0) return fail(QM_ECUDA, "no CUDA device");
    CU_TRY(cudaGetDevice(&dev));
    CU_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double *sink = nullptr;
    CU_TRY(cudaMalloc(&sink, sizeof(double)));
    cudaEvent_t e0, e1;
    CU_TRY(cudaEventCreate(&e0)); CU_TRY(cudaEventCreate(&e1));
    const int iters = 1 << 15, threads = 512, blocks = sms * 4;
    float ms = 0.f;
    double best_mma = 0.0, best_fma = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        CU_TRY(cudaEventRecord(e0));
        k_probe_dmma<<<blocks, threads>>>(sink, iters);
        CU_TRY(cudaEventRecord(e1)); CU_TRY(cudaEventSynchronize(e1));
        CU_TRY(cudaEventElapsedTime(&ms, e0, e1));
        // one DMMA m8n8k4 = 8*8*4 FMA = 512 flop per warp instruction
        const double fl = (double)blocks * (threads / 32) * (double)iters * 8.0 * 512.0;
        best_mma = std::max(best_mma, fl / (ms * 1e-3) * 1e-12);
        CU_TRY(cudaEventRecord(e0));
        k_probe_dfma<<<blocks, threads>>>(sink, iters);
        CU_TRY(cudaEventRecord(e1)); CU_TRY(cudaEventSynchronize(e1));
        CU_TRY(cudaEventElapsedTime(&ms, e0, e1));
        const double fl2 = (double)blocks * threads * (double)iters * 16.0 * 2.0;
        best_fma = std::max(best_fma, fl2 / (ms * 1e-3) * 1e-12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    if (tflops_dmma) *tflops_dmma = best_mma;
    if (tflops_dfma) *tflops_dfma = best_fma;
    return QM_OK;
}

}  // extern "C"
