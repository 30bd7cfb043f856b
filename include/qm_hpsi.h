/*
 * qm_hpsi.h -- C ABI of the B200-native plane-wave Kohn-Sham Hamiltonian apply.
 *
 *   H|psi_nk>(G) = 1/2 |k+G|^2 psi(G)                                   PAPER.md:146 (eq. 12), 668-674 (eqs. 49-51)
 *                + [ FFT( V_loc(r) * IFFT(psi) ) ](G)                    PAPER.md:652-666 (eqs. 46-48), 725-730
 *                + sum_ij beta_i(G) D_ij <beta_j|psi>                    PAPER.md:153-161 (eq. 14), 1019-1024
 *
 * The operator is the paper's KSHam.h_psi(): a black-box
 * Hermitian apply on a block of trial vectors in complex128.
 *
 * Conventions (readings A1-A8 of DESIGN.md section 3):
 *  - Hartree / bohr inside; ecutwfc given in Ry; sphere = { m : |k+G_m|^2 [bohr^-2] <= ecutwfc [Ry] }.
 *  - lattice rows are a_i; b_i = rows of 2 pi (A^-1)^T; k in fractions of b_i.
 *  - sphere order = ascending C-order flat box index
 *        idx = ((m1 mod n1)*n2 + (m2 mod n2))*n3 + (m3 mod n3)
 *  - V_r is flat C order over (n1,n2,n3), r_j = sum_i (j_i/n_i) a_i.
 *  - wavefunction blocks are [nbands][ng(k)] row-major complex128 (last axis = G,
 *    PAPER.md:783-784), interleaved (re,im), 16-byte aligned.
 *
 * Pointer kinds are stated per argument: HOST or DEVICE.  No torch types, no
 * exceptions, no printing.  Every function returns QM_OK (0) or a negative
 * qm_status; qm_last_error() gives thread-local text for the last failure.
 * Hot-path calls (qm_apply_h) only enqueue work on `stream` (a cudaStream_t
 * passed as void*): no device synchronisation, no host<->device copy, no
 * allocation after the first call with a given nbands (none at all after
 * qm_reserve).
 * There is no CPU fallback: without a CUDA device every compute call fails
 * with QM_ECUDA.
 *
 * Devices and streams.  A handle belongs to the CUDA device that was current in
 * qm_gspace_create; every call that touches the device returns QM_EINVAL if
 * another device is current.  Work spaces are owned per k-point: calls for
 * DIFFERENT k-points of one handle may be in flight on different streams at the
 * same time (e.g. the ten k-points of a band x k batch); calls for the SAME
 * k-point, and qm_set_vloc / qm_split_operator_set / the density calls (shared
 * tables), must be stream-ordered with respect to each other -- the library
 * cannot detect a violation.  Host-side state (qm_last_error is thread-local;
 * the handle is not locked) allows one calling thread per handle at a time.
 */
#ifndef QM_HPSI_H
#define QM_HPSI_H

#include <stdint.h>

#if defined(__GNUC__)
#define QM_API __attribute__((visibility("default")))
#else
#define QM_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qm_gspace qm_gspace;                 /* opaque, owned by the library */
typedef struct { double re, im; } qm_c128;          /* interleaved complex128 */

typedef enum {
    QM_OK = 0,
    QM_EINVAL = -1,      /* bad argument (null pointer, k out of range, nbands <= 0, overlap ...) */
    QM_ENOTSET = -2,     /* qm_apply_h before qm_set_vloc / qm_set_nonlocal for that k */
    QM_EGRID = -3,       /* sphere does not fit the FFT grid (2|m_i|+1 > n_i) or grid size unsupported */
    QM_ECUDA = -4,       /* CUDA runtime error (text in qm_last_error) */
    QM_ENOMEM = -5       /* host or device allocation failed */
} qm_status;

/* Build the G-sphere, its sphere->box index map and the stick tables for nk k-points.
 * (GSpace(recilat, ecut) and the per-k gkspc.)
 *  lattice_bohr  HOST  9 doubles, rows a1,a2,a3
 *  ecutwfc_ry          cut-off in Rydberg
 *  fft_grid      HOST  3 ints n1,n2,n3; each must be a supported FFT length (see qm_fft_size_supported: products of two
 *                      radices <= 16 with factors 2, 3, 5, from 8 to 256) and hold the sphere (2|m_i|+1 <= n_i), else
 *                      QM_EGRID.  The three lengths are independent.  Boxes with n1 == n2 <= 144 whose xy-plane working set
 *                      fits one SM's shared memory (up to the 216-atom cell at 30 Ry) run the fused xy-plane kernel; every
 *                      other legal box (n1 != n2, longer axes, larger planes: PAPER.md:689-712, 1490, 1666) runs the same
 *                      transforms as separate y | x | y passes through HBM -- same results, same entry points.
 *  kpts_cryst    HOST  nk*3 doubles (may be NULL iff nk==1 => Gamma)
 *  out                 receives the handle; destroy with qm_gspace_destroy.
 * Uploads the tables to the current CUDA device (synchronously; this is set-up, not hot path). */
QM_API int qm_gspace_create(const double *lattice_bohr, double ecutwfc_ry, const int *fft_grid,
                     const double *kpts_cryst, int nk, qm_gspace **out);
QM_API int qm_gspace_destroy(qm_gspace *g);

/* Queries (HOST outputs). */
QM_API int qm_gspace_num_k(const qm_gspace *g, int *nk);
QM_API int qm_gspace_num_g(const qm_gspace *g, int k, int *ng);
QM_API int qm_gspace_num_sticks(const qm_gspace *g, int k, int *nsticks, int *nxcols);
QM_API int qm_gspace_get_index_map(const qm_gspace *g, int k, int32_t *idx_host);   /* ng */
QM_API int qm_gspace_get_miller(const qm_gspace *g, int k, int32_t *miller_host);   /* ng*3 */
QM_API int qm_gspace_get_g2(const qm_gspace *g, int k, double *g2_host);            /* |k+G|^2, bohr^-2 */
/* *flag = 1 if n_i >= 4 max|m_i| + 1 on every axis (the product V*psi is alias free) */
QM_API int qm_gspace_alias_free(const qm_gspace *g, int k, int *flag);
/* 1 if `n` is a supported FFT length, else 0. */
QM_API int qm_fft_size_supported(int n);

/* Set the local potential (eq. 47).
 *  V_r_dev  DEVICE  n1*n2*n3 doubles, C order, Hartree.
 * The library copies (and re-lays-out) V on `stream`; the caller may free its buffer once the
 * stream reaches that point. */
QM_API int qm_set_vloc(qm_gspace *g, const double *V_r_dev, void *stream);

/* Set the non-local projectors for k-point k.
 *  beta_kG_dev  DEVICE  [nproj][ng(k)] row-major complex128
 *  D_dev        DEVICE  (nproj/d_block) real symmetric blocks [d_block][d_block], Hartree;
 *                       d_block == nproj => one dense matrix.  nproj % d_block == 0.
 *  nproj == 0 (pointers may be NULL) selects a local-only Hamiltonian.
 * The library copies both on `stream`. */
QM_API int qm_set_nonlocal(qm_gspace *g, int k, const qm_c128 *beta_kG_dev, int nproj,
                    const double *D_dev, int d_block, void *stream);

/* Grow the per-k-point work spaces (stick planes, unfused slabs, projector partials) that qm_apply_h,
 * qm_split_operator_propagate and qm_density_accumulate need for blocks of up to `nbands` wavefunctions at k-point k, so
 * that none of those calls allocates later (projector work spaces are sized by qm_set_nonlocal as well).  NOT covered, and
 * still grown on first use by their own calls: the density running sum (qm_density_reset), the two Taylor blocks
 * (qm_taylor_propagate), the box of the debug hooks (qm_debug_g2r / r2g), the split-K partials of qm_subspace and the
 * work spaces of a qm_mtxel handle.  May synchronise the device (cudaMalloc); not a hot-path call. */
QM_API int qm_reserve(qm_gspace *g, int k, int nbands);

/* psi_out = H psi_in for a block of nbands wavefunctions at k-point k.
 *  psi_in_dev, psi_out_dev  DEVICE  [nbands][ng(k)] row-major complex128; must not overlap;
 *                           psi_out is overwritten.
 * Only enqueues work; everything is ordered on `stream`.  (With projectors set, the first projection GEMM, which reads
 * psi_in only, is placed on a library-owned side stream that forks from and joins `stream` by events, so that it may
 * run beside the FFT kernels; to the caller the call behaves like work on `stream`, also under stream capture.) */
QM_API int qm_apply_h(qm_gspace *g, const qm_c128 *psi_in_dev, qm_c128 *psi_out_dev,
               int nbands, int k, void *stream);

/* A fixed batch of qm_apply_h calls as ONE submission (north_star: "batched over (band,k)"; the paper's band and
 * k-point independence).  The items -- (k[i], psi_in_dev[i], psi_out_dev[i], nbands[i]), every pointer
 * DEVICE and fixed for the life of the plan -- are captured once into a CUDA graph: items of different k-points sit on
 * parallel branches (k-points own their work spaces), items of one k-point run in list order.  qm_batch_plan_launch
 * enqueues the whole graph on `stream`; it replaces the per-call launch latency that dominates the small configs.
 * qm_set_vloc / qm_set_nonlocal must have been called for every k used; creation reserves the work spaces
 * (qm_reserve) and may synchronise.  The graph holds the addresses and shapes of the k-points' work spaces, so two
 * things make a plan STALE: a later call on one of its k-points that needs a larger work space than the plan
 * reserved (qm_apply_h, qm_reserve, density, Taylor, debug calls with more bands: the block is freed and re-allocated),
 * and a later qm_set_nonlocal with a different nproj or d_block for one of its k-points.  The library counts both per
 * k-point; qm_batch_plan_launch on a stale plan launches nothing and returns QM_EINVAL -- destroy the plan and create
 * it again (or call qm_reserve with the largest band count you will use BEFORE creating plans).  The plan borrows
 * the handle: destroy it before qm_gspace_destroy. */
typedef struct qm_batch_plan qm_batch_plan;
QM_API int qm_batch_plan_create(qm_gspace *g, int nitems, const int *k, const qm_c128 *const *psi_in_dev,
                                qm_c128 *const *psi_out_dev, const int *nbands, qm_batch_plan **out);
QM_API int qm_batch_plan_launch(qm_batch_plan *p, void *stream);
QM_API int qm_batch_plan_destroy(qm_batch_plan *p);

/* Electron density from Bloch states (eq. 2, 1008):  n(r_j) = sum_i f_i |psi_i(r_j)|^2 with
 * psi_i(r_j) = sum_{G in sphere(k)} psi_i(G) exp(+i G.r_j) (unnormalised synthesis, reading A5/A20; the Bloch phase
 * exp(i k.r) drops out of |psi|^2), r_j = sum_a (j_a/n_a) a_a.  Scatter, pruned backward FFT and |.|^2 are fused; the
 * full box of psi(r) is never written.  The running sum lives in library memory between calls:
 *   qm_density_reset      zero it (allocates on first use);
 *   qm_density_accumulate add weight * occ[i] * |psi_i(r)|^2 for a block of nbands states at k-point k
 *                         (call it once per band batch and k-point; weight = the k-point weight);
 *   qm_density_get        rho[j] = scale * running sum, flat C order over (n1,n2,n3), overwritten.
 *  psi_dev  DEVICE [nbands][ng(k)] complex128    occ_dev  DEVICE [nbands] doubles    rho_dev  DEVICE [n1*n2*n3] doubles
 * Every z-plane of the sum is accumulated by one thread block in band order: bitwise reproducible, no atomics.
 * QM_ENOTSET if accumulate / get come before reset.  All three only enqueue on `stream`. */
QM_API int qm_density_reset(qm_gspace *g, void *stream);
QM_API int qm_density_accumulate(qm_gspace *g, int k, const qm_c128 *psi_dev, int nbands, const double *occ_dev,
                          double weight, void *stream);
QM_API int qm_density_get(qm_gspace *g, double *rho_dev, double scale, void *stream);

/* Taylor-series propagator of the TDKS equation (eq. 52; the paper's prop_psi()):
 *   psi_out = sum_{r=0}^{order} (-i dt)^r / r!  H^r psi_in          (dt in atomic units of time, H in Hartree)
 * as `order` chained qm_apply_h calls with a fused scale-and-accumulate kernel between them; needs qm_set_vloc /
 * qm_set_nonlocal like qm_apply_h.  psi_in_dev, psi_out_dev DEVICE [nbands][ng(k)] complex128, must not overlap;
 * psi_out is overwritten.  order == 0 copies.  Two library-owned blocks of the same size are grown on first use. */
QM_API int qm_taylor_propagate(qm_gspace *g, int k, const qm_c128 *psi_in_dev, qm_c128 *psi_out_dev, int nbands, double dt,
                        int order, void *stream);

/* Split-operator exponential of the TDKS propagator (eq. 53; the paper's second expoper form):
 *   psi_out = exp(-i dt T/2) exp(-i dt V) exp(-i dt T/2) psi_in
 * T(G) = 1/2 |k+G|^2 is diagonal on the sphere: its half-steps are the phases exp(-i dt |k+G|^2 / 4), applied as psi
 * is scattered and as the result is gathered.  V is the LOCAL potential (reading A22 of DESIGN.md: the paper does not say
 * what V holds when projectors are present; they are not part of this propagator -- use qm_taylor_propagate): the
 * middle factor is the multiplication by exp(-i dt V(r_j)) on the FFT grid between the backward and the forward
 * transform, i.e. on the sphere  sum_G' Ehat(G - G') psi(G'),  Ehat = (1/N) DFT[exp(-i dt V)].  One pass, three kernels.
 *   qm_split_operator_set        builds exp(-i dt V(r)) / N and the kinetic phases of every k-point on `stream`
 *                                V_r_dev DEVICE n1*n2*n3 doubles, C order, Hartree (copied); dt in atomic units of time
 *   qm_split_operator_propagate  psi_in_dev, psi_out_dev DEVICE [nbands][ng(k)] complex128, must not overlap;
 *                                QM_ENOTSET before qm_split_operator_set. */
QM_API int qm_split_operator_set(qm_gspace *g, const double *V_r_dev, double dt, void *stream);
QM_API int qm_split_operator_propagate(qm_gspace *g, int k, const qm_c128 *psi_in_dev, qm_c128 *psi_out_dev, int nbands,
                                       void *stream);

/* GW plane-wave matrix elements (eqs. 56-57; the paper's matrix_elements):
 *   M_{nn'}(k, q, G) = < n k+q | exp(i (q+G).r) | n' k > = sum_G'' conj(c_{n,k+q}(G''+G)) c_{n'k}(G'')
 * for the G of the epsilon sphere |q+G|^2 < ecut_eps (strict, as printed in eq. 56), q = kpts[k_bra] - kpts[k_ket]
 * in crystal coordinates.  Reading A21 of DESIGN.md: eq. 56 is the definition (eq. 57 names the FFT directions the
 * other way round from eq. 9); G''+G is looked up modulo the FFT box (reading A8), so on a box with
 * n_i >= 2 m_wfn + m_eps + 1 nothing wraps.  No cell-volume factor.  Computed as the paper describes: both states are
 * synthesised on the grid (scatter + pruned backward FFT), multiplied, and analysed (forward FFT pruned to the
 * epsilon sphere); the ket boxes are synthesised once per call.
 *   qm_mtxel_create     builds the epsilon sphere (sorted like the wavefunction spheres: ascending C-order box index) and
 *                       its stick tables on the handle's FFT box; QM_EGRID if it does not fit (2|m_i|+1 > n_i).
 *                       The qm_mtxel borrows the handle: destroy it before qm_gspace_destroy.
 *   qm_mtxel_num_g / _get_miller / _get_index_map   HOST outputs, ng_eps / ng_eps*3 / ng_eps entries
 *   qm_matrix_elements  bra_dev DEVICE [nbra][ng(k_bra)], ket_dev DEVICE [nket][ng(k_ket)] complex128;
 *                       out_dev DEVICE [nbra][nket][ng_eps] complex128, overwritten.  Only enqueues on `stream`
 *                       after its work spaces ((nket + a few) boxes of n1*n2*n3 complex128) exist. */
typedef struct qm_mtxel qm_mtxel;
QM_API int qm_mtxel_create(qm_gspace *g, int k_bra, int k_ket, double ecut_eps_ry, qm_mtxel **out);
QM_API int qm_mtxel_destroy(qm_mtxel *m);
QM_API int qm_mtxel_num_g(const qm_mtxel *m, int *ng);
QM_API int qm_mtxel_get_miller(const qm_mtxel *m, int32_t *miller_host);
QM_API int qm_mtxel_get_index_map(const qm_mtxel *m, int32_t *idx_host);
QM_API int qm_matrix_elements(qm_mtxel *m, const qm_c128 *bra_dev, int nbra, const qm_c128 *ket_dev, int nket,
                              qm_c128 *out_dev, void *stream);

/* Subspace products S[i][j] = <a_i|b_j> = sum_G conj(a_i(G)) b_j(G) over the sphere of k-point k: the step right
 * after h_psi in the Davidson solver, the paper's WavefunG.vdot(psi, phi) = ZGEMM.
 * With b = H a this is the subspace Hamiltonian, with b = a the overlap matrix.  Plain sum, no volume factor.
 *  a_dev  DEVICE  [na][ng(k)] row-major complex128     b_dev  DEVICE  [nb][ng(k)] row-major complex128
 *  s_dev  DEVICE  [na][nb] row-major complex128, overwritten; must not overlap a or b.  a == b is allowed.
 * FP64 tensor cores (DMMA), split-K with a fixed-order reduction (bitwise reproducible).  Only enqueues on `stream`;
 * the split-K workspace is library owned and grown on first use. */
QM_API int qm_subspace(qm_gspace *g, int k, const qm_c128 *a_dev, int na, const qm_c128 *b_dev, int nb,
                qm_c128 *s_dev, void *stream);

/* qm_subspace for callers that are not allowed to allocate device memory: the same product, the same kernels, the same
 * summation order (hence the same bits as qm_subspace on the same device), but no handle and no cudaMalloc anywhere.
 *
 * Who needs this.  qm_subspace keeps its split-K partial sums in a buffer it cudaMallocs on first use.  That is not
 * possible for (1) a host application whose own memory pool (a framework's caching allocator, a DFT code's arena) has
 * already claimed almost the whole device, so a cudaMalloc from inside this library fails with out-of-memory although
 * the caller has buffers to hand out; (2) a solver iteration that keeps several streams busy: cudaMalloc and cudaFree
 * synchronise the whole device, so one growing work space stalls every stream, not just the caller's; (3) a job that
 * runs under a fixed memory budget and must know the footprint of this library when it is loaded, not when a larger
 * block first arrives.  For them the partial sums live in ONE fixed array that is part of the library image
 * (static __device__, QM_SUBSPACE_STATIC_MAX_ELEMS complex128 = 16 MiB): every GPU on which the library's kernels are
 * loaded carries these 16 MiB until the process exits, whether or not this function is ever called.
 *
 *  a_dev  DEVICE  [na][ng] row-major complex128     b_dev  DEVICE  [nb][ng] row-major complex128     (16-byte aligned)
 *  s_dev  DEVICE  [na][nb] row-major complex128, overwritten; must not overlap a or b.  a == b is allowed.
 *  ng             row length = number of plane waves of the sphere (what qm_gspace_num_g reports); no handle is needed.
 * The caller owns all three buffers; the call allocates no device memory (no cudaMalloc, cudaMallocAsync, cudaFree,
 * and no library routine that would) -- not on the first call either.  It runs on the current device.
 *
 * Limit.  The partial sums of one call need  ceil(na/64)*64 * ceil(nb/64)*64  elements per K split and must fit the
 * array: blocks up to 1024 x 1024 states (or 512 x 2048, ...) are taken; beyond that the call returns QM_EINVAL and
 * touches nothing -- use qm_subspace there.  Inside the limit the split count is the one qm_subspace would choose.
 *
 * First call on a device.  It looks up the device address of the array (cudaGetSymbolAddress), reads the SM count and
 * opts the GEMM kernel into its shared-memory size; these are synchronous set-up calls, remembered per device.  Make
 * that first call during start-up, outside any stream capture; later calls on that device only enqueue two kernels on
 * `stream`.
 *
 * Sharing.  There is one array per device and every call uses it.  Nothing in it has to start at zero: each call
 * writes every partial sum it later reads, so whatever the previous call left behind is ignored.  But two calls whose
 * kernels can run at the same time on one GPU (different streams without an ordering between them, or two host
 * threads) overwrite each other's partial sums and both results are garbage -- the library cannot see this.  Order such
 * calls on one stream or with events.  Different GPUs have different copies and do not interfere. */
#define QM_SUBSPACE_STATIC_MAX_ELEMS (1u << 20)
QM_API int qm_subspace_static(const qm_c128 *a_dev, int na, const qm_c128 *b_dev, int nb, int ng, qm_c128 *s_dev,
                              void *stream);

/* Same operation with HOST buffers (pinned memory recommended): the library copies psi_in to
 * a library-owned device buffer, applies H, copies the result back, all on `stream`, then
 * synchronises the stream.  This is the end-to-end entry bench.py times. */
QM_API int qm_apply_h_host(qm_gspace *g, const qm_c128 *psi_in_host, qm_c128 *psi_out_host,
                    int nbands, int k, void *stream);

/* Asynchronous form of qm_apply_h_host for streaming many blocks: the call only enqueues
 * (H2D on an internal copy stream, the apply on `stream`, D2H on a second internal copy stream,
 * chained by events, two staging slots) and returns; consecutive calls therefore overlap the
 * copies of one block with the compute of its neighbours.  psi_out_host is valid, and
 * psi_in_host may be reused, after qm_host_synchronize (or after the matching block's D2H has
 * completed).  Host buffers should be pinned, otherwise the copies are synchronous. */
QM_API int qm_apply_h_host_async(qm_gspace *g, const qm_c128 *psi_in_host, qm_c128 *psi_out_host,
                                 int nbands, int k, void *stream);
QM_API int qm_host_synchronize(qm_gspace *g);

/* Test hooks (not hot path) exercising the same kernels (A5):
 *  qm_debug_g2r : box_r[b][n1*n2*n3] = (1/N) sum_G psi_g[b][G] e^{+iG.r}   (scatter + backward FFT)
 *  qm_debug_r2g : psi_g[b][ng]       = sum_r box_r[b][r] e^{-iG.r}, taken on the sphere (unnormalised)
 * all buffers DEVICE. */
QM_API int qm_debug_g2r(qm_gspace *g, const qm_c128 *psi_g_dev, qm_c128 *box_r_dev, int nbands, int k, void *stream);
QM_API int qm_debug_r2g(qm_gspace *g, const qm_c128 *box_r_dev, qm_c128 *psi_g_dev, int nbands, int k, void *stream);

/* Number of CUDA kernels this handle has launched so far (for bench.py's gpu_launches). */
QM_API int qm_get_launch_count(const qm_gspace *g, unsigned long long *count);

/* Per-kernel device timing (measurement aid for bench.py's roofline block; off by default).
 * When enabled every hot-path kernel launch is bracketed by CUDA events on its own stream.
 * qm_profile_read synchronises those events and returns the accumulated device time (ms) and
 * the number of launches of one kernel kind since the last reset. */
typedef enum {
    QM_K_ZINV = 0,      /* scatter + backward z-FFT on sticks           (a1, a2) */
    QM_K_PLANE = 1,     /* fused xy-plane kernel incl. V_loc multiply   (a2, a3, a4) */
    QM_K_ZFWD = 2,      /* forward z-FFT + gather + kinetic             (a4, a5) */
    QM_K_PROJ1 = 3,     /* P = beta^H psi   (DMMA)                      (a6) */
    QM_K_PREDUCE = 4,   /* split-K reduction of P; with D blocks that divide 16 also Q = D P, fused  (a7) */
    QM_K_DMUL = 5,      /* Q = D P, general block size (separate launch)  (a7) */
    QM_K_PROJ2 = 6,     /* out += beta Q    (DMMA)                      (a8) */
    QM_K_SUBGEMM = 7,   /* S = A^H B (DMMA, split-K)                     (8(f) rank 1) */
    QM_K_SUBREDUCE = 8, /* split-K reduction of S */
    QM_K_GENY = 9,      /* unfused y pass (backward or forward) of boxes the fused plane kernel does not take */
    QM_K_GENX = 10,     /* unfused x round trip incl. V_loc multiply of such boxes */
    QM_K_COUNT = 11
} qm_kernel_kind;
QM_API int qm_profile_enable(qm_gspace *g, int on);
QM_API int qm_profile_reset(qm_gspace *g);
QM_API int qm_profile_read(qm_gspace *g, int kind, double *total_ms, unsigned long long *launches);
QM_API const char *qm_kernel_name(int kind);

/* FP64 tensor-core (DMMA m8n8k4) peak probe: runs a register-resident DMMA loop on every SM
 * and returns the measured TFLOP/s (HOST output).  Used as the roofline denominator for the
 * projector GEMMs (MEASURED_PEAKS.json has no FP64 entry). Synchronous. */
QM_API int qm_probe_fp64_tensor_peak(double *tflops_dmma, double *tflops_dfma);

QM_API const char *qm_last_error(void);                    /* thread-local text */
QM_API const char *qm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* QM_HPSI_H */
