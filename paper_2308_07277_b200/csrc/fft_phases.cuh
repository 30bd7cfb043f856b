// Phase functions of the pruned 3-D FFT pipeline ("sticks").
//
// A length-N line (N = R1*R2) lives in shared memory as a padded 2-D array [R1][R2P], R2P = R2|1
// (odd pitch => the strided accesses of the second four-step pass are bank-conflict free).
//   natural index i      <-> pos(i) = (i / R2) * R2P + i % R2
//   transposed label p   <-> same pos(p); label p = k1*R2 + k2 stands for index k1 + R1*k2
// Backward transform "A": natural in  -> transposed out, in place, one barrier between its two steps.
// Forward  transform "B": transposed in -> natural out,  in place, one barrier between its two steps.
// So G -> r -> G never needs a transpose or a digit-reversal pass: the r-space data simply lives in
// transposed order and V_loc is re-laid-out once (qm_set_vloc) to match.
//
// Every function here is one "phase": it is executed by all threads of a CTA between two barriers.
// They are __host__ __device__ so tests/test_host_emulation.py can run the identical index logic
// on the CPU with a loop over thread ids.
#pragma once
#include "fft_reg.cuh"

template <int R1_, int R2_> struct LineCfg {
    static constexpr int R1 = R1_, R2 = R2_;
    static constexpr int N = R1 * R2;
    static constexpr int R2P = R2 | 1;
    static constexpr int L = R1 * R2P;                  // padded line length
    static constexpr int TT = R1 > R2 ? R1 : R2;        // team size (threads per line)
    static QM_HD int pos(int i) { return (i / R2) * R2P + (i % R2); }
};

// Per-thread twiddle rows held in registers: TW[j] = exp(-2 pi i u j / N) for the thread's fixed u.
// (Looking them up in shared memory at stride j costs up to 8-way bank conflicts; every thread keeps
//  the same u for the whole kernel, so the row is loaded once.)
template <int R> struct TwRow {
    c128 w[R];
    template <int J> QM_HD c128 get() const { return w[J]; }
};
// Same interface, but looked up in a table on every use (kernels that use each twiddle only once).
struct TwTable {
    const c128 *tw; int u;
    template <int J> QM_HD c128 get() const { return tw[u * J]; }
};
template <int R> QM_HD void load_twrow(TwRow<R> &t, const c128 *tw, int u, int limit) {
    static_for<R>([&](auto I) { constexpr int j = decltype(I)::value; t.w[j] = (u < limit) ? tw[u * j] : c128{1.0, 0.0}; });
}

// One plane row of the stick buffer: the occupied i2 indices are the intervals [a1,b1] and [a2,b2]
// (convex sphere), stored back to back starting at stick index sbase.
struct RowInfo {
    int a1, b1, a2, b2, sbase;
    QM_HD int stick(int i) const {      // stick index of natural index i, or -1 if the row has no stick there
        return (i >= a1 && i <= b1) ? sbase + i - a1
                                    : ((i >= a2 && i <= b2) ? sbase + (b1 - a1 + 1) + i - a2 : -1);
    }
};
// Backward step 1 reading its (pruned) input straight from the stick plane in global memory:
// the plane array needs neither a load pass nor a zero fill.
template <class C, class TW> QM_HD void lineA_step1_gin(c128 *line, const c128 *Wp, const RowInfo ri, int u, const TW &tw) {
    if (u >= C::R2) return;
    c128 t[C::R1];
    static_for<C::R1>([&](auto I) {
        constexpr int n1 = decltype(I)::value;
        const int s = ri.stick(n1 * C::R2 + u);
        t[n1] = (s >= 0) ? Wp[s] : c128{0.0, 0.0};
    });
    Dft<C::R1, +1>::run(t);
    static_for<C::R1>([&](auto I) {
        constexpr int k1 = decltype(I)::value;
        line[k1 * C::R2P + u] = (k1 == 0) ? t[k1] : cmul_conj(t[k1], tw.template get<k1>());
    });
}
// Forward step 2 writing only the occupied outputs straight to the stick plane in global memory.
template <class C> QM_HD void lineB_step2_gout(const c128 *line, c128 *Wp, const RowInfo ri, int u) {
    if (u >= C::R2) return;
    c128 t[C::R1];
    static_for<C::R1>([&](auto I) { constexpr int a = decltype(I)::value; t[a] = line[a * C::R2P + u]; });
    Dft<C::R1, -1>::run(t);
    static_for<C::R1>([&](auto I) {
        constexpr int c = decltype(I)::value;
        const int s = ri.stick(c * C::R2 + u);
        if (s >= 0) Wp[s] = t[c];
    });
}

// ---- pruned passes with hoisted addressing ---------------------------------------------------------
// A thread with fixed u touches the line elements i = n*R2 + u (n = 0..R1-1).  When only two index
// intervals [a1,b1], [a2,b2] of the line exist (stored back to back with element stride `stride`), the
// elements that exist and their addresses depend on (u, intervals) only: they are worked out once
// (per kernel for the x direction, per row for the y direction) instead of once per access.
struct Pruned {
    unsigned m1, m2;      // bit n set: i = n*R2+u lies in interval 1 / interval 2
    int c1, c2;           // element offset of i: n*R2*stride + c1 (interval 1), + c2 (interval 2)
};
QM_HD unsigned qm_range_mask(int a, int b, int u, int r2, int r1) {   // { n : a <= n*r2 + u <= b }
    int lo = a - u, hi = b - u;
    if (hi < 0 || b < a) return 0u;
    lo = lo <= 0 ? 0 : (lo + r2 - 1) / r2;
    hi = hi / r2;
    if (hi > r1 - 1) hi = r1 - 1;
    return lo > hi ? 0u : ((2u << hi) - (1u << lo));
}
template <class C> QM_HD Pruned make_pruned(int a1, int b1, int a2, int b2, int u, int stride) {
    const int cnt1 = b1 >= a1 ? b1 - a1 + 1 : 0;
    return Pruned{qm_range_mask(a1, b1, u, C::R2, C::R1), qm_range_mask(a2, b2, u, C::R2, C::R1),
                  (u - a1) * stride, (u - a2 + cnt1) * stride};
}
// Stick-plane workspace W of one band, blocked by tiles of QM_ZT sticks: element (plane label p, stick s) lives at
// base[((s / QM_ZT) * n3 + p) * QM_ZT + s % QM_ZT].  A tile's N3 x QM_ZT block is contiguous (what the z kernels move
// with one bulk copy); the plane kernel addresses single elements through this pointer-like view (p fixed).
constexpr int QM_ZT = 16;
struct WView {
    c128 *base;            // element (p, stick 0) of the band: band base + p * QM_ZT
    unsigned tstride;      // elements between consecutive tiles: n3 * QM_ZT
    int s;                 // stick
    QM_HD WView operator+(int e) const { return WView{base, tstride, s + e}; }
    QM_HD c128 *ptr() const { const unsigned us = (unsigned)s; return base + ((us / QM_ZT) * tstride + (us % QM_ZT)); }
};
QM_HD WView qm_wview(c128 *band_base, int p, int n3) { return WView{band_base + p * QM_ZT, (unsigned)(n3 * QM_ZT), 0}; }
QM_HD const c128 *qm_ptr(const c128 *p) { return p; }
QM_HD c128 *qm_ptr(c128 *p) { return p; }
QM_HD c128 *qm_ptr(const WView &w) { return w.ptr(); }

// predicated 16-byte accesses (no branch, no address arithmetic beyond base + immediate)
struct SpaceShared {}; struct SpaceGlobal {};
QM_HD c128 ld_pred(SpaceShared, const c128 *p, bool pred) {
#ifdef __CUDA_ARCH__
    c128 v;
    asm volatile("{ .reg .pred q; setp.ne.u32 q, %3, 0; mov.f64 %0, 0d0000000000000000; mov.f64 %1, 0d0000000000000000;\n"
                 "  @q ld.shared.v2.f64 {%0, %1}, [%2]; }"
                 : "=d"(v.x), "=d"(v.y) : "r"((unsigned)__cvta_generic_to_shared(p)), "r"((unsigned)pred) : "memory");
    return v;
#else
    return pred ? *p : c128{0.0, 0.0};
#endif
}
QM_HD c128 ld_pred(SpaceGlobal, const c128 *p, bool pred) {
#ifdef __CUDA_ARCH__
    c128 v;
    asm volatile("{ .reg .pred q; setp.ne.u32 q, %3, 0; mov.f64 %0, 0d0000000000000000; mov.f64 %1, 0d0000000000000000;\n"
                 "  @q ld.global.v2.f64 {%0, %1}, [%2]; }"
                 : "=d"(v.x), "=d"(v.y) : "l"(p), "r"((unsigned)pred) : "memory");
    return v;
#else
    return pred ? *p : c128{0.0, 0.0};
#endif
}
QM_HD void st_pred(SpaceShared, c128 *p, c128 v, bool pred) {
#ifdef __CUDA_ARCH__
    asm volatile("{ .reg .pred q; setp.ne.u32 q, %3, 0; @q st.shared.v2.f64 [%0], {%1, %2}; }"
                 :: "r"((unsigned)__cvta_generic_to_shared(p)), "d"(v.x), "d"(v.y), "r"((unsigned)pred) : "memory");
#else
    if (pred) *p = v;
#endif
}
QM_HD void st_pred(SpaceGlobal, c128 *p, c128 v, bool pred) {
#ifdef __CUDA_ARCH__
    asm volatile("{ .reg .pred q; setp.ne.u32 q, %3, 0; @q st.global.v2.f64 [%0], {%1, %2}; }"
                 :: "l"(p), "d"(v.x), "d"(v.y), "r"((unsigned)pred) : "memory");
#else
    if (pred) *p = v;
#endif
}
// Backward step 1 with pruned input: src = first stored element of the line, estride = R2*stride (elements
// between n and n+1); writes the full padded line `dst`.
template <class C, class SP, class P, class TW>
QM_HD void prunedA_step1(SP sp, const P src, int estride, const Pruned pr, c128 *dst, int u, const TW &tw) {
    if (u >= C::R2) return;
    c128 t[C::R1];
    // interval 1 lies below N/2 and interval 2 at or above it (host tables), so for most n1 the interval is
    // known at compile time and the access is base + immediate under one mask-bit test
    const P p1 = src + pr.c1, p2 = src + pr.c2;
    const unsigned mm = pr.m1 | pr.m2;
    static_for<C::R1>([&](auto I) {
        constexpr int n1 = decltype(I)::value;
        if constexpr (2 * (n1 + 1) * C::R2 <= C::N) t[n1] = ld_pred(sp, qm_ptr(p1 + n1 * estride), (mm & (1u << n1)) != 0u);
        else if constexpr (2 * n1 * C::R2 >= C::N) t[n1] = ld_pred(sp, qm_ptr(p2 + n1 * estride), (mm & (1u << n1)) != 0u);
        else {
            const bool in2 = (pr.m2 >> n1) & 1u;
            t[n1] = ld_pred(sp, qm_ptr((in2 ? p2 : p1) + n1 * estride), (mm & (1u << n1)) != 0u);
        }
    });
    Dft<C::R1, +1>::run(t);
    static_for<C::R1>([&](auto I) {
        constexpr int k1 = decltype(I)::value;
        dst[k1 * C::R2P + u] = (k1 == 0) ? t[k1] : cmul_conj(t[k1], tw.template get<k1>());
    });
}
// "Quarter" form of the pruned backward step 1: when every occupied index lies below N/4 or at/above 3N/4
// (true for every alias-free grid, 4 m + 1 <= n), only the first Q and the last Q first-pass inputs of a thread
// can exist, Q = ceil(R1 / 4).  They are fetched ahead of time into 2Q registers (prefetch_quarter) and the
// transform is started later from those registers (prunedA_step1_pre).
template <class C> struct Quarter { static constexpr int Q = (C::R1 + 3) / 4; };
template <class C, class SP, class P>
QM_HD void prefetch_quarter(SP sp, const P src, int estride, const Pruned pr, c128 (&pre)[2 * Quarter<C>::Q]) {
    constexpr int Q = Quarter<C>::Q;
    const P p1 = src + pr.c1, p2 = src + pr.c2;
    static_for<Q>([&](auto I) {
        constexpr int j = decltype(I)::value;
        pre[j] = ld_pred(sp, qm_ptr(p1 + j * estride), (pr.m1 >> j) & 1u);
        pre[Q + j] = ld_pred(sp, qm_ptr(p2 + (C::R1 - Q + j) * estride), (pr.m2 >> (C::R1 - Q + j)) & 1u);
    });
}
template <class C, class TW>
QM_HD void prunedA_step1_pre(const c128 (&pre)[2 * Quarter<C>::Q], c128 *dst, int u, const TW &tw) {
    if (u >= C::R2) return;
    constexpr int Q = Quarter<C>::Q;
    c128 t[C::R1];
    static_for<C::R1>([&](auto I) {
        constexpr int n1 = decltype(I)::value;
        if constexpr (n1 < Q) t[n1] = pre[n1];
        else if constexpr (n1 >= C::R1 - Q) t[n1] = pre[Q + n1 - (C::R1 - Q)];
        else t[n1] = c128{0.0, 0.0};
    });
    Dft<C::R1, +1>::run(t);
    static_for<C::R1>([&](auto I) {
        constexpr int k1 = decltype(I)::value;
        dst[k1 * C::R2P + u] = (k1 == 0) ? t[k1] : cmul_conj(t[k1], tw.template get<k1>());
    });
}
// Forward step 2 with pruned output: reads the full padded line `srcline`, stores only what exists.
template <class C, class SP, class P>
QM_HD void prunedB_step2(SP sp, const c128 *srcline, const P dst, int estride, const Pruned pr, int u) {
    if (u >= C::R2) return;
    c128 t[C::R1];
    static_for<C::R1>([&](auto I) { constexpr int a = decltype(I)::value; t[a] = srcline[a * C::R2P + u]; });
    Dft<C::R1, -1>::run(t);
    const P p1 = dst + pr.c1, p2 = dst + pr.c2;
    const unsigned mm = pr.m1 | pr.m2;
    static_for<C::R1>([&](auto I) {
        constexpr int c = decltype(I)::value;
        if constexpr (2 * (c + 1) * C::R2 <= C::N) st_pred(sp, qm_ptr(p1 + c * estride), t[c], (mm & (1u << c)) != 0u);
        else if constexpr (2 * c * C::R2 >= C::N) st_pred(sp, qm_ptr(p2 + c * estride), t[c], (mm & (1u << c)) != 0u);
        else {
            const bool in2 = (pr.m2 >> c) & 1u;
            st_pred(sp, qm_ptr((in2 ? p2 : p1) + c * estride), t[c], (mm & (1u << c)) != 0u);
        }
    });
}
// Quarter-rule form of the pruned forward step 2: only the first Q and last Q outputs of a thread can exist.
template <class C, class SP, class P>
QM_HD void prunedB_step2_quarter(SP sp, const c128 *srcline, const P dst, int estride, const Pruned pr, int u) {
    if (u >= C::R2) return;
    constexpr int Q = Quarter<C>::Q;
    c128 t[C::R1];
    static_for<C::R1>([&](auto I) { constexpr int a = decltype(I)::value; t[a] = srcline[a * C::R2P + u]; });
    Dft<C::R1, -1>::run(t);
    const P p1 = dst + pr.c1, p2 = dst + pr.c2;
    static_for<Q>([&](auto I) {
        constexpr int j = decltype(I)::value;
        constexpr int c2 = C::R1 - Q + j;
        st_pred(sp, qm_ptr(p1 + j * estride), t[j], (pr.m1 >> j) & 1u);
        st_pred(sp, qm_ptr(p2 + c2 * estride), t[c2], (pr.m2 >> c2) & 1u);
    });
}

template <class C, class TW> QM_HD void lineA_step1(c128 *line, int u, const TW &tw) {
    if (u >= C::R2) return;
    c128 t[C::R1];
    static_for<C::R1>([&](auto I) { constexpr int n1 = decltype(I)::value; t[n1] = line[n1 * C::R2P + u]; });
    Dft<C::R1, +1>::run(t);
    static_for<C::R1>([&](auto I) {
        constexpr int k1 = decltype(I)::value;
        line[k1 * C::R2P + u] = (k1 == 0) ? t[k1] : cmul_conj(t[k1], tw.template get<k1>());
    });
}
template <class C> QM_HD void lineA_step2(c128 *line, int u) {
    if (u >= C::R1) return;
    c128 t[C::R2];
    static_for<C::R2>([&](auto I) { constexpr int n2 = decltype(I)::value; t[n2] = line[u * C::R2P + n2]; });
    Dft<C::R2, +1>::run(t);
    static_for<C::R2>([&](auto I) { constexpr int k2 = decltype(I)::value; line[u * C::R2P + k2] = t[k2]; });
}
template <class C, class TW> QM_HD void lineB_step1(c128 *line, int u, const TW &tw) {
    if (u >= C::R1) return;
    c128 t[C::R2];
    static_for<C::R2>([&](auto I) { constexpr int b = decltype(I)::value; t[b] = line[u * C::R2P + b]; });
    Dft<C::R2, -1>::run(t);
    static_for<C::R2>([&](auto I) {
        constexpr int d = decltype(I)::value;
        line[u * C::R2P + d] = (d == 0) ? t[d] : cmul(t[d], tw.template get<d>());
    });
}
template <class C> QM_HD void lineB_step2(c128 *line, int u) {
    if (u >= C::R2) return;
    c128 t[C::R1];
    static_for<C::R1>([&](auto I) { constexpr int a = decltype(I)::value; t[a] = line[a * C::R2P + u]; });
    Dft<C::R1, -1>::run(t);
    static_for<C::R1>([&](auto I) { constexpr int c = decltype(I)::value; line[c * C::R2P + u] = t[c]; });
}

// ---- z kernels: one shared-memory round trip per stick ------------------------------------------------
// zinv pass 2: thread (stick t, row u) finishes the backward transform and writes the stick planes
// W[p = u*R2 + k2][s] straight from registers (lanes run over sticks => contiguous 16-byte stores).
template <class C> QM_HD void zinv_step2_store(const c128 *line, c128 *Wcol, long pstride, int u) {
    if (u >= C::R1) return;
    c128 t[C::R2];
    static_for<C::R2>([&](auto I) { constexpr int n2 = decltype(I)::value; t[n2] = line[u * C::R2P + n2]; });
    Dft<C::R2, +1>::run(t);
    static_for<C::R2>([&](auto I) { constexpr int k2 = decltype(I)::value; Wcol[(long)(u * C::R2 + k2) * pstride] = t[k2]; });
}
// zfwd pass 1: thread (stick t, row u) reads W[p = u*R2 + b][s] into registers and starts the forward transform.
template <class C, class TW> QM_HD void zfwd_step1_load(const c128 *Wcol, long pstride, c128 *line, int u, const TW &tw) {
    if (u >= C::R1) return;
    c128 t[C::R2];
    static_for<C::R2>([&](auto I) { constexpr int b = decltype(I)::value; t[b] = Wcol[(long)(u * C::R2 + b) * pstride]; });
    Dft<C::R2, -1>::run(t);
    static_for<C::R2>([&](auto I) {
        constexpr int d = decltype(I)::value;
        line[u * C::R2P + d] = (d == 0) ? t[d] : cmul(t[d], tw.template get<d>());
    });
}
// zfwd pass 2: finishes the forward transform and gathers to the sphere with the kinetic term fused
// (PAPER.md:668-674): out[g] = (V psi)(G) + 1/2 |k+G|^2 psi_in[g] for the G of this stick only.
template <class C> QM_HD void zfwd_step2_gather(const c128 *line, c128 *out, const c128 *psi_in, const double *g2,
                                                 const Pruned pr, int u, bool kinetic) {
    if (u >= C::R2) return;
    c128 t[C::R1];
    static_for<C::R1>([&](auto I) { constexpr int a = decltype(I)::value; t[a] = line[a * C::R2P + u]; });
    Dft<C::R1, -1>::run(t);
    static_for<C::R1>([&](auto I) {
        constexpr int c = decltype(I)::value;
        const bool in2 = (pr.m2 >> c) & 1u, in1 = (pr.m1 >> c) & 1u;
        const int off = (in2 ? pr.c2 : pr.c1) + c * C::R2;
        if (in1 || in2) {
            c128 v = t[c];
            if (kinetic) { const double h = 0.5 * g2[off]; const c128 x = psi_in[off]; v.x = fma(h, x.x, v.x); v.y = fma(h, x.y, v.y); }
            out[off] = v;
        }
    });
}

// Quarter-rule forms of the gather (see Quarter): the 1/2|k+G|^2 psi_in terms of the <= 2Q outputs a thread can
// own are fetched ahead of the transform (prefetch_kin) and added when the outputs are stored.
template <class C> QM_HD void prefetch_kin(const c128 *psi_in, const double *g2, const Pruned pr, bool kinetic,
                                            c128 (&kin)[2 * Quarter<C>::Q]) {
    constexpr int Q = Quarter<C>::Q;
    static_for<Q>([&](auto I) {
        constexpr int j = decltype(I)::value;
        const int o1 = pr.c1 + j * C::R2, o2 = pr.c2 + (C::R1 - Q + j) * C::R2;
        const bool q1 = kinetic && ((pr.m1 >> j) & 1u), q2 = kinetic && ((pr.m2 >> (C::R1 - Q + j)) & 1u);
        const c128 x1 = ld_pred(SpaceGlobal{}, psi_in + o1, q1), x2 = ld_pred(SpaceGlobal{}, psi_in + o2, q2);
        const double h1 = q1 ? 0.5 * g2[o1] : 0.0, h2 = q2 ? 0.5 * g2[o2] : 0.0;
        kin[j] = c128{h1 * x1.x, h1 * x1.y};
        kin[Q + j] = c128{h2 * x2.x, h2 * x2.y};
    });
}
template <class C> QM_HD void zfwd_step2_gather_pre(const c128 *line, c128 *out, const Pruned pr, int u,
                                                     const c128 (&kin)[2 * Quarter<C>::Q]) {
    if (u >= C::R2) return;
    constexpr int Q = Quarter<C>::Q;
    c128 t[C::R1];
    static_for<C::R1>([&](auto I) { constexpr int a = decltype(I)::value; t[a] = line[a * C::R2P + u]; });
    Dft<C::R1, -1>::run(t);
    static_for<Q>([&](auto I) {
        constexpr int j = decltype(I)::value;
        constexpr int c2 = C::R1 - Q + j;
        st_pred(SpaceGlobal{}, out + pr.c1 + j * C::R2, t[j] + kin[j], (pr.m1 >> j) & 1u);
        st_pred(SpaceGlobal{}, out + pr.c2 + c2 * C::R2, t[c2] + kin[Q + j], (pr.m2 >> c2) & 1u);
    });
}

// ---- x direction of the plane kernel: X compact rows <-> full length-N1 line in scratch -------------
// A: plane array [X][rowpitch].  The occupied box indices i1 form two intervals (the sphere is convex):
// [a1,b1] -> rows 0.., [a2,b2] -> rows (b1-a1+1)..; everything else is not stored (zero).
struct XRows {
    int a1, b1, a2, b2;
    QM_HD int row(int i1) const {
        return (i1 >= a1 && i1 <= b1) ? i1 - a1 : ((i1 >= a2 && i1 <= b2) ? i1 - a2 + (b1 - a1 + 1) : -1);
    }
};
template <class C, class TW> QM_HD void xcol_step1(const c128 *A, int rowpitch, int colpos, const XRows xr,
                                                   c128 *scr, int u, const TW &tw) {
    if (u >= C::R2) return;
    c128 t[C::R1];
    static_for<C::R1>([&](auto I) {
        constexpr int n1 = decltype(I)::value;
        const int r = xr.row(n1 * C::R2 + u);
        t[n1] = (r >= 0) ? A[r * rowpitch + colpos] : c128{0.0, 0.0};
    });
    Dft<C::R1, +1>::run(t);
    static_for<C::R1>([&](auto I) {
        constexpr int k1 = decltype(I)::value;
        scr[k1 * C::R2P + u] = (k1 == 0) ? t[k1] : cmul_conj(t[k1], tw.template get<k1>());
    });
}
// MODE 0: apply  (backward step 2, multiply by v[x], forward step 1)      PAPER.md:659-662 (eq. 47)
// MODE 1: g2r    (backward step 2, write psi(r)*scale to box, stop)
// MODE 2: r2g    (read box, forward step 1)
// v: this thread's R2 potential values V(x = u + R1*k2), already in registers (prefetched by the caller).
// box: pointer to element x=0 of this column in a natural-order box, xstride = n2*n3.
template <int R> struct VRow { double v[R]; };
// V of one plane column is stored in pairs: vcol[(j * R1 + u) * 2 + e] = V(x = u + R1*(2j + e)), j < R2E/2
// (R2E = R2 rounded up to even, the pad is zero), so a thread reads its R2 values with 16-byte loads and the
// lanes of a team read contiguous 16-byte words.
template <class C> struct VLayout { static constexpr int R2E = C::R2 + (C::R2 & 1), COL = C::R1 * R2E; };
template <class C> QM_HD void load_vrow(VRow<C::R2> &vr, const double *vcol, int u) {
    if (u >= C::R1) return;
#ifdef QM_ABLATE_V        /* timing experiment only */
    static_for<C::R2>([&](auto I) { vr.v[decltype(I)::value] = 1.0; });
    return;
#endif
    const double2 *q = reinterpret_cast<const double2 *>(vcol) + u;
    static_for<VLayout<C>::R2E / 2>([&](auto I) {
        constexpr int j = decltype(I)::value;
        const double2 d = q[j * C::R1];
        vr.v[2 * j] = d.x;
        if constexpr (2 * j + 1 < C::R2) vr.v[2 * j + 1] = d.y;
    });
}
template <class C, int MODE, class TW> QM_HD void xcol_step2(c128 *scr, int u, const TW &tw, const VRow<C::R2> &vr,
                                                             c128 *box, long xstride, double scale) {
    if (u >= C::R1) return;
    c128 t[C::R2];
    if constexpr (MODE == 2) {
        static_for<C::R2>([&](auto I) { constexpr int k2 = decltype(I)::value; t[k2] = box[(long)(u + C::R1 * k2) * xstride]; });
    } else {
        static_for<C::R2>([&](auto I) { constexpr int n2 = decltype(I)::value; t[n2] = scr[u * C::R2P + n2]; });
        Dft<C::R2, +1>::run(t);                      // t[k2] = psi(x = u + R1*k2)
        if constexpr (MODE == 1) {
            static_for<C::R2>([&](auto I) { constexpr int k2 = decltype(I)::value; box[(long)(u + C::R1 * k2) * xstride] = cscale(t[k2], scale); });
            return;
        } else {
            static_for<C::R2>([&](auto I) { constexpr int k2 = decltype(I)::value; t[k2] = cscale(t[k2], vr.v[k2]); });
        }
    }
    Dft<C::R2, -1>::run(t);
    static_for<C::R2>([&](auto I) {
        constexpr int d = decltype(I)::value;
        scr[u * C::R2P + d] = (d == 0) ? t[d] : cmul(t[d], tw.template get<d>());
    });
}
template <class C> QM_HD void xcol_step3(c128 *A, int rowpitch, int colpos, const XRows xr,
                                         const c128 *scr, int u) {
    if (u >= C::R2) return;
    c128 t[C::R1];
    static_for<C::R1>([&](auto I) { constexpr int a = decltype(I)::value; t[a] = scr[a * C::R2P + u]; });
    Dft<C::R1, -1>::run(t);
    static_for<C::R1>([&](auto I) {
        constexpr int c = decltype(I)::value;
        const int r = xr.row(u + C::R2 * c);
        if (r >= 0) A[r * rowpitch + colpos] = t[c];
    });
}
