// Internal declarations shared by the translation units of libqm_hpsi (not part of the C ABI).
//   qm_api.cu          the C ABI, host-side set-up, projector / subspace launches
//   qm_z.cu            launches of the z-stick kernels (k_zinv, k_zfwd), every supported length
//   qm_plane<M>.cu     launches of the fused xy-plane kernel, one translation unit per MODE (compiled in parallel)
//   qm_geny.cu, qm_genx<M>.cu   the unfused y / x passes for boxes the fused kernel cannot take (n1 != n2, large planes)
#pragma once
#include <cuda_runtime.h>
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <utility>
#include <vector>

#include "../../include/qm_hpsi.h"
#include "fft_kernels.cuh"
#include "qm_plan.h"
#include "gspace_host.h"

extern thread_local std::string qm_g_err;            // defined in qm_api.cu
inline int fail(int code, const std::string &msg) { qm_g_err = msg; return code; }

#define CU_TRY(expr)                                                                        \
    do {                                                                                    \
        cudaError_t _e = (expr);                                                            \
        if (_e != cudaSuccess)                                                              \
            return fail(_e == cudaErrorMemoryAllocation ? QM_ENOMEM : QM_ECUDA,             \
                        std::string(#expr) + ": " + cudaGetErrorString(_e));                \
    } while (0)

template <class T> struct DevBuf {
    T *p = nullptr; size_t n = 0;
    unsigned long long *moved = nullptr;    // counter to bump when a live block is freed and re-allocated (KPoint::ws_gen)
    ~DevBuf() { if (p) cudaFree(p); }
    cudaError_t resize(size_t m) {
        if (m <= n) return cudaSuccess;
        if (p) { cudaFree(p); p = nullptr; n = 0; if (moved) ++*moved; }
        cudaError_t e = cudaMalloc(&p, m * sizeof(T));
        if (e == cudaSuccess) n = m;
        return e;
    }
    cudaError_t upload(const std::vector<T> &h) {
        cudaError_t e = resize(h.size() ? h.size() : 1);
        if (e != cudaSuccess) return e;
        if (h.empty()) return cudaSuccess;
        return cudaMemcpy(p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice);
    }
};

struct KPoint : QmKTables {
    DevBuf<int4> d_rowinfo, d_stickinfo;
    DevBuf<double> d_g2;
    // non-local
    bool nl_set = false;
    int nproj = 0, dblock = 0;
    int nmblk = 0, nkc = 0, ngt = 0, nic = 0;          // tile counts of the two beta copies
    DevBuf<c128> d_beta1, d_beta2;
    DevBuf<double> d_D;
    // workspaces of this k-point (calls on different k-points may run on different streams)
    DevBuf<c128> d_W, d_Ppart, d_P, d_part;
    DevBuf<c128> d_slab;                                // unfused path: half-transformed planes (gen_kernels.cuh)
    DevBuf<double> d_qt;
    DevBuf<int> d_pdesc;
    DevBuf<c128> d_sophase;                             // split-operator: exp(-i dt |k+G|^2 / 4)
    cudaStream_t side_stream = nullptr;                 // GEMM 1 of an apply runs here, beside the FFT path (qm_api.cu run_apply)
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    // Work-space generation: goes up whenever one of the blocks above is moved by a growing resize, or qm_set_nonlocal
    // changes the projector shape.  A qm_batch_plan holds these addresses and shapes inside its graph; it records the
    // generation of every k-point it uses and qm_batch_plan_launch refuses to run a stale graph.
    unsigned long long ws_gen = 0;
    KPoint() {
        d_beta1.moved = d_beta2.moved = d_W.moved = d_Ppart.moved = d_P.moved = d_part.moved = d_slab.moved = &ws_gen;
        d_D.moved = d_qt.moved = &ws_gen;
        d_pdesc.moved = &ws_gen;
    }
    KPoint(const KPoint &) = delete;
    KPoint &operator=(const KPoint &) = delete;
    ~KPoint() {
        if (ev_fork) cudaEventDestroy(ev_fork);
        if (ev_join) cudaEventDestroy(ev_join);
        if (side_stream) cudaStreamDestroy(side_stream);
    }
    // unfused passes: resident CTAs per SM of k_gen_y (forward / backward) and of k_gen_x per MODE for this k-point's x
    // tile; 0 = not asked yet.  Filled by qm_prepare_gen_* at qm_gspace_create (and at the first launch for the sphere
    // of a qm_mtxel handle), so that no launch on the hot path or under stream capture queries the occupancy.
    int gen_y_per_sm[2] = {0, 0};
    int gen_x_per_sm[5] = {0, 0, 0, 0, 0};
    double ecut_override = 0.0;                         // epsilon spheres (qm_mtxel) carry their own cut-off
    QmKPlanDev plan() const {
        QmKPlanDev p;
        p.ng = ng; p.nsticks = nsticks; p.nx = nx; p.rowpitch = rowpitch;
        p.g2 = d_g2.p;
        p.row_info = d_rowinfo.p; p.x_iv = xiv; p.stick_info = d_stickinfo.p;
        return p;
    }
};

struct Profiler {
    bool on = false;
    std::vector<cudaEvent_t> pool;
    size_t used = 0;
    struct Rec { int kind; size_t e0, e1; };
    std::vector<Rec> recs;
    double total_ms[QM_K_COUNT] = {0};
    unsigned long long count[QM_K_COUNT] = {0};
    ~Profiler() { for (auto e : pool) cudaEventDestroy(e); }
    size_t next() {
        if (used == pool.size()) { cudaEvent_t e; cudaEventCreate(&e); pool.push_back(e); }
        return used++;
    }
    void begin(int kind, cudaStream_t st) {
        if (!on) return;
        Rec r; r.kind = kind; r.e0 = next(); r.e1 = next();
        cudaEventRecord(pool[r.e0], st);
        recs.push_back(r);
    }
    void end(cudaStream_t st) { if (on) cudaEventRecord(pool[recs.back().e1], st); }
    void collect() {
        for (const Rec &r : recs) {
            cudaEventSynchronize(pool[r.e1]);
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, pool[r.e0], pool[r.e1]) == cudaSuccess) {
                total_ms[r.kind] += ms; count[r.kind]++;
            }
        }
        recs.clear(); used = 0;
    }
    void reset() { collect(); for (int i = 0; i < QM_K_COUNT; ++i) { total_ms[i] = 0; count[i] = 0; } }
};

struct HostPipe {       // two-slot staging pipeline behind qm_apply_h_host(_async)
    bool init = false;
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaEvent_t in_ready[2], compute_done[2], out_done[2];
    bool used[2] = {false, false};
    DevBuf<c128> in[2], out[2];
    int slot = 0;
    ~HostPipe() {
        if (!init) return;
        for (int i = 0; i < 2; ++i) { cudaEventDestroy(in_ready[i]); cudaEventDestroy(compute_done[i]); cudaEventDestroy(out_done[i]); }
        cudaStreamDestroy(s_in); cudaStreamDestroy(s_out);
    }
};

struct qm_gspace {
    Profiler prof;
    HostPipe pipe;
    double lattice[9], recip[9];
    double ecut;
    int grid[3];
    QmAxis ax[3];
    std::vector<KPoint *> kpts;
    DevBuf<c128> d_tw[3];
    DevBuf<double> d_vt, d_rhot;
    bool rho_open = false;
    bool v_set = false;
    DevBuf<c128> d_subpart, d_tay_h, d_tay_t;
    DevBuf<c128> d_boxt;            // transposed boxes of the debug hooks
    DevBuf<c128> d_sofield;         // split-operator: exp(-i dt V(r)) / N in the transposed-box layout
    bool so_set = false;
    double so_dt = 0.0;
    unsigned long long launches = 0;
    bool pdl = true;                // programmatic dependent launch between the kernels of an apply (QM_PDL=0: off)
    bool nl_overlap = true;         // projection GEMM of an apply on a side stream beside the FFT path (QM_NL_OVERLAP=0: off)
    bool fused = true;              // the fused plane kernel takes this box (else: the unfused passes, gen_kernels.cuh)
    int device = 0;                 // the CUDA device the handle was created on (every call checks it)
    int sm_count = 148;
    int max_smem = 0;
    size_t l2_bytes = 0;
    int fft_chunk = 0;              // bands per internal pass of the FFT path (0: derived from the L2 size; QM_FFT_CHUNK)
    int z_cta_per_sm = 2;           // resident z-kernel CTAs per SM the grid is sized for (QM_Z_CTA_PER_SM)
    int plane_ctas_per_sm = 0;      // resident plane-kernel CTAs per SM (0: two when two plane arrays fit, else one; QM_PLANE_CTAS)
    ~qm_gspace() { for (auto *k : kpts) delete k; }
};

// GW plane-wave matrix elements for one (k+q, k) pair of k-points: the epsilon sphere |q+G|^2 < ecut_eps on the
// handle's FFT box, with its own stick tables, and the workspaces of qm_matrix_elements.
struct qm_mtxel {
    qm_gspace *g = nullptr;
    int k_bra = 0, k_ket = 0;
    KPoint sph;
    DevBuf<c128> d_ketbox, d_brabox, d_Wp;
};

// A fixed list of qm_apply_h calls captured as one CUDA graph (qm_batch_plan_*).
struct qm_batch_plan {
    qm_gspace *g = nullptr;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    unsigned long long launches = 0;        // kernels per graph launch
    std::vector<std::pair<int, unsigned long long>> gens;   // (k, KPoint::ws_gen at capture) of every k-point in the graph
    ~qm_batch_plan() {
        if (exec) cudaGraphExecDestroy(exec);
        if (graph) cudaGraphDestroy(graph);
    }
};

constexpr int PLANE_GROUP = QM_GROUP;
inline size_t plane_rowtab_bytes(const qm_gspace *g, const KPoint *kp) {
    return (size_t)kp->nx * std::max(g->ax[0].r1, g->ax[0].r2) * sizeof(int4);
}
inline size_t plane_smem(const qm_gspace *g, const KPoint *kp, int ngroups) {
    const QmAxis &ax = g->ax[0];
    const int tt = std::max(ax.r1, ax.r2);
    const size_t sl = (size_t)qm_scratch_pitch(ax.len, tt);
    // scratch lines per group: one per team, plus a sink line when some lanes of a group have no butterfly in a pass
    // (fft_kernels.cuh PlaneGeom)
    const int lpg = PLANE_GROUP / tt + ((ax.r1 != ax.r2 || PLANE_GROUP % tt != 0) ? 1 : 0);
    const size_t a_elems = ((size_t)kp->nx * kp->rowpitch + 7) & ~(size_t)7;
    return (a_elems + (size_t)ngroups * lpg * sl) * sizeof(c128) + (size_t)kp->nx * sizeof(int4) + 16;
}

// number of independent groups of the plane kernel: the fewest groups that reach the
// minimum number of column rounds within the shared-memory and thread limits
inline int plane_groups(const qm_gspace *g, const KPoint *kp, int ctas_per_sm = 1) {
    const QmAxis &ax = g->ax[0];
    const int tpg = PLANE_GROUP / std::max(ax.r1, ax.r2);
    const int nchunks = (ax.n + tpg - 1) / tpg;
    int gmax = std::min(QM_PLANE_MAX_THREADS / PLANE_GROUP / ctas_per_sm, nchunks);
    if (gmax < 1) return 0;
    // the SM's shared memory (max_smem + 1 KB reserved per CTA) is shared by the resident CTAs
    const size_t budget = ctas_per_sm == 1 ? (size_t)g->max_smem : ((size_t)g->max_smem + 1024) / ctas_per_sm - 1024;
    while (gmax > 1 && plane_smem(g, kp, gmax) > budget) --gmax;
    if (plane_smem(g, kp, gmax) > budget) return 0;
    const int rounds = (nchunks + gmax - 1) / gmax;
    int best = gmax;
    for (int c = gmax; c >= 1; --c)
        if ((nchunks + c - 1) / c == rounds) best = c;
    return best;
}

// z kernels: grid.x tiles-in-flight per band chosen so that the whole grid is close to a whole number of
// resident CTAs per SM (each CTA then loops over ~ntiles / grid.x tiles)
inline int z_grid_x(const qm_gspace *g, int ntiles, int nb, int cta_per_sm) {
    const int slots = g->sm_count * cta_per_sm;
    int gx = std::max(1, slots / std::max(1, nb));
    if (gx >= ntiles) return ntiles;
    const int rounds = (ntiles + gx - 1) / gx;          // fewest CTAs that keep the same number of rounds
    return (ntiles + rounds - 1) / rounds;
}

// Kernel launch with the programmatic-serialisation attribute (async_copy.cuh pdl_wait): only for kernels that call
// pdl_wait() before they touch global memory.
template <class... KArgs, class... Args>
inline cudaError_t qm_launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl,
                                 Args &&...args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(std::forward<Args>(args))...);
}

struct PlaneArgs {          // operands of the plane kernel beyond the stick planes W
    c128 *box = nullptr;            // MODE 1 output / MODE 2 first operand (transposed boxes, one per state)
    const c128 *box2 = nullptr;     // MODE 2 second operand (conjugated) / MODE 4 complex field
    int npair2 = 0;                 // MODE 2 with a second operand: states in box2 (plane index counts pairs a * npair2 + b)
    double scale = 1.0;
    const double *occ = nullptr;    // MODE 3
    double *rhot = nullptr;
};

// dispatch on FFT length ---------------------------------------------------------------------
// QM_FOR_SIZES: the lengths the fused plane kernel is compiled for; QM_FOR_SIZES_ALL adds the lengths above 144 that only the
// z kernels and the unfused passes take (gspace_host.h kQmSizes lists them all).
#ifdef QM_DEV_SIZES      /* developer builds: only the lengths of the five BASELINE.json configs (fast compile) */
#define QM_FOR_SIZES(X) X(12, 3, 4) X(24, 4, 6) X(32, 4, 8) X(48, 6, 8) X(96, 12, 8) X(144, 12, 12)
#define QM_FOR_SIZES_ALL(X) QM_FOR_SIZES(X) X(36, 6, 6) X(192, 12, 16)
#else
#define QM_FOR_SIZES(X)                                                                              \
    X(8, 2, 4) X(12, 3, 4) X(16, 4, 4) X(18, 3, 6) X(20, 4, 5) X(24, 4, 6) X(30, 5, 6) X(32, 4, 8)   \
    X(36, 6, 6) X(40, 5, 8) X(48, 6, 8) X(60, 6, 10) X(64, 8, 8) X(72, 8, 9) X(80, 8, 10)            \
    X(96, 12, 8) X(100, 10, 10) X(108, 9, 12) X(120, 10, 12) X(128, 8, 16) X(144, 12, 12)
#define QM_FOR_SIZES_ALL(X) QM_FOR_SIZES(X) X(160, 10, 16) X(180, 12, 15) X(192, 12, 16) X(225, 15, 15) X(240, 15, 16) X(256, 16, 16)
#endif

// ---- launches implemented in the other translation units ------------------------------------------------------
// phase == nullptr: plain scatter; else psi(G) * phase[g] on the way in (split-operator half-step)
int qm_launch_zinv(qm_gspace *g, KPoint *kp, const c128 *psi, const c128 *phase, c128 *W, int nb, cudaStream_t st);
// gm: fft_phases.cuh GM_*
int qm_launch_zfwd(qm_gspace *g, KPoint *kp, int gm, const c128 *W, const c128 *aux, c128 *out, int nb, double scale,
                   cudaStream_t st);
int qm_prepare_z(qm_gspace *g);
// fused xy-plane kernel, MODE 0..4 (one translation unit each)
int qm_launch_plane_m0(qm_gspace *g, KPoint *kp, c128 *W, int nb, const PlaneArgs &a, cudaStream_t st);
int qm_launch_plane_m1(qm_gspace *g, KPoint *kp, c128 *W, int nb, const PlaneArgs &a, cudaStream_t st);
int qm_launch_plane_m2(qm_gspace *g, KPoint *kp, c128 *W, int nb, const PlaneArgs &a, cudaStream_t st);
int qm_launch_plane_m3(qm_gspace *g, KPoint *kp, c128 *W, int nb, const PlaneArgs &a, cudaStream_t st);
int qm_launch_plane_m4(qm_gspace *g, KPoint *kp, c128 *W, int nb, const PlaneArgs &a, cudaStream_t st);
int qm_prepare_plane_m0(qm_gspace *g);
int qm_prepare_plane_m1(qm_gspace *g);
int qm_prepare_plane_m2(qm_gspace *g);
int qm_prepare_plane_m3(qm_gspace *g);
int qm_prepare_plane_m4(qm_gspace *g);
// unfused passes (qm_geny.cu, qm_genx<M>.cu): one slab pass over the planes [bp0, bp0 + nbp) of a launch
int qm_launch_gen_y(qm_gspace *g, KPoint *kp, bool back, c128 *W, c128 *slab, int bp0, int nbp, cudaStream_t st);
int qm_launch_gen_x_m0(qm_gspace *g, KPoint *kp, c128 *slab, int bp0, int nbp, const PlaneArgs &a, cudaStream_t st);
int qm_launch_gen_x_m1(qm_gspace *g, KPoint *kp, c128 *slab, int bp0, int nbp, const PlaneArgs &a, cudaStream_t st);
int qm_launch_gen_x_m2(qm_gspace *g, KPoint *kp, c128 *slab, int bp0, int nbp, const PlaneArgs &a, cudaStream_t st);
int qm_launch_gen_x_m3(qm_gspace *g, KPoint *kp, c128 *slab, int bp0, int nbp, const PlaneArgs &a, cudaStream_t st);
int qm_launch_gen_x_m4(qm_gspace *g, KPoint *kp, c128 *slab, int bp0, int nbp, const PlaneArgs &a, cudaStream_t st);
int qm_prepare_gen_y(qm_gspace *g);
int qm_prepare_gen_x_m0(qm_gspace *g);
int qm_prepare_gen_x_m1(qm_gspace *g);
int qm_prepare_gen_x_m2(qm_gspace *g);
int qm_prepare_gen_x_m3(qm_gspace *g);
int qm_prepare_gen_x_m4(qm_gspace *g);
