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
//  the same u for a whole phase, so the row is loaded once per phase.)
template <int R> struct TwRow {
    c128 w[R];
    template <int J> QM_HD c128 get() const { return w[J]; }
};
template <int R> QM_HD void load_twrow(TwRow<R> &t, const c128 *tw, int u, int limit) {
    static_for<R>([&](auto I) { constexpr int j = decltype(I)::value; t.w[j] = (u < limit) ? tw[u * j] : c128{1.0, 0.0}; });
}

// ---- shared-memory lines -----------------------------------------------------------------------------
// A line in shared memory as its own pointer-like type, so that the pruned passes can tell it from a global
// pointer (predicated accesses need the state space).  Plain accesses go through the generic pointer: explicit
// ld/st.shared asm for them was measured 4 % slower in the plane kernel (it pins the instruction order).
struct SLine {
    c128 *p;
    QM_HD c128 &operator[](int i) const { return p[i]; }
    QM_HD SLine operator+(int e) const { return SLine{p + e}; }
};
QM_HD SLine qm_sline(const c128 *p) { return SLine{const_cast<c128 *>(p)}; }

// Stick-plane workspace W of one band, blocked by tiles of QM_ZT sticks: element (plane label p, stick s) lives at
// band_base[((s / QM_ZT) * n3 + p) * QM_ZT + s % QM_ZT].  A tile's N3 x QM_ZT block is contiguous (what the z kernels
// move with one bulk copy); the plane kernel addresses single elements through this pointer-like view (p fixed).
#ifndef QM_ZT_STICKS
#define QM_ZT_STICKS 16
#endif
constexpr int QM_ZT = QM_ZT_STICKS;
struct WView {
    c128 *base;            // element (p, stick 0) of the band: band base + p * QM_ZT
    unsigned tstride;      // elements between consecutive tiles: n3 * QM_ZT
    int s;                 // stick
    QM_HD WView operator+(int e) const { return WView{base, tstride, s + e}; }
    QM_HD c128 *ptr() const { const unsigned us = (unsigned)s; return base + ((us / QM_ZT) * tstride + (us % QM_ZT)); }
};
QM_HD WView qm_wview(c128 *band_base, int p, int n3) { return WView{band_base + p * QM_ZT, (unsigned)(n3 * QM_ZT), 0}; }

// ---- predicated 16-byte accesses (no branch) ------------------------------------------------------------
QM_HD c128 ld_pred(const c128 *p, bool pred) {
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
QM_HD c128 ld_pred(const WView &w, bool pred) { return ld_pred((const c128 *)w.ptr(), pred); }
QM_HD c128 ld_pred(const SLine &l, bool pred) {
#ifdef __CUDA_ARCH__
    c128 v;
    asm volatile("{ .reg .pred q; setp.ne.u32 q, %3, 0; mov.f64 %0, 0d0000000000000000; mov.f64 %1, 0d0000000000000000;\n"
                 "  @q ld.shared.v2.f64 {%0, %1}, [%2]; }"
                 : "=d"(v.x), "=d"(v.y) : "r"((unsigned)__cvta_generic_to_shared(l.p)), "r"((unsigned)pred) : "memory");
    return v;
#else
    return pred ? *l.p : c128{0.0, 0.0};
#endif
}
QM_HD void st_pred(c128 *p, c128 v, bool pred) {
#ifdef __CUDA_ARCH__
    asm volatile("{ .reg .pred q; setp.ne.u32 q, %3, 0; @q st.global.v2.f64 [%0], {%1, %2}; }"
                 :: "l"(p), "d"(v.x), "d"(v.y), "r"((unsigned)pred) : "memory");
#else
    if (pred) *p = v;
#endif
}
QM_HD void st_pred(const WView &w, c128 v, bool pred) { st_pred(w.ptr(), v, pred); }
QM_HD void st_pred(const SLine &l, c128 v, bool pred) {
#ifdef __CUDA_ARCH__
    asm volatile("{ .reg .pred q; setp.ne.u32 q, %3, 0; @q st.shared.v2.f64 [%0], {%1, %2}; }"
                 :: "r"((unsigned)__cvta_generic_to_shared(l.p)), "d"(v.x), "d"(v.y), "r"((unsigned)pred) : "memory");
#else
    if (pred) *l.p = v;
#endif
}

// A sphere-side operand that is multiplied by a per-G phase as it is loaded (split-operator propagator,
// PAPER.md:1137-1139 eq. 53: psi(G) exp(-i dt |k+G|^2 / 4) on the way into the backward transform).  Pointer-like, so
// the pruned passes below take it in place of a plain pointer; `ph` is indexed like the first band of `a`.
struct PhasedPtr {
    const c128 *a, *ph;
    QM_HD PhasedPtr operator+(int e) const { return PhasedPtr{a + e, ph + e}; }
};
QM_HD c128 ld_pred(const PhasedPtr &p, bool pred) {
    const c128 x = ld_pred(p.a, pred), w = ld_pred(p.ph, pred);
    return cmul(x, w);
}

// ---- pruned passes with hoisted addressing ---------------------------------------------------------
// A thread with fixed u touches the line elements i = n*R2 + u (n = 0..R1-1).  When only two index
// intervals [a1,b1], [a2,b2] of the line exist (stored back to back with element stride `stride`), the
// elements that exist and their addresses depend on (u, intervals) only: they are worked out once
// (per kernel for the x direction, per row / stick for the y and z directions) instead of once per access.
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
// intervals packed as in the host tables: x = a1 | b1 << 16, y = a2 | b2 << 16
template <class C> QM_HD Pruned make_pruned_packed(int x, int y, int u, int stride) {
    return make_pruned<C>((int)(short)(x & 0xffff), x >> 16, (int)(short)(y & 0xffff), y >> 16, u, stride);
}

// Backward step 1 with pruned input.  src: pointer-like (const c128 *, WView, SLine) to the first stored element
// of the line, estride = R2*stride (elements between n and n+1); writes the full padded line `dst`.
// Interval 1 lies below N/2 and interval 2 at or above it (host tables), so for most n the interval is known at
// compile time and the access is base + immediate under one mask-bit test.
// Every first pass is written as a head (loads + radix-R butterflies into t[]) and a tail (twiddle multiply + store), so
// that a caller may fetch the twiddle row between the two (tmem_rows.cuh); the one-call forms below do both.
// The tails take the factors j in [J0, J1) of the row at a time (TwChunk: a window of a row), so that a row that is not
// held in registers can be brought in piecewise.
template <int J0, int J1> struct TwChunk {
    c128 w[J1 - J0];
    template <int J> QM_HD c128 get() const { static_assert(J >= J0 && J < J1, "factor outside the chunk"); return w[J - J0]; }
};
template <class C, int J0, int J1, bool GUARD = true, class L, class TW>
QM_HD void stepA1_tail_range(const c128 (&t)[C::R1], const L dst, int u, const TW &tw) {
    if constexpr (GUARD) if (u >= C::R2) return;
    static_for<J1 - J0>([&](auto I) {
        constexpr int k1 = J0 + decltype(I)::value;
        if constexpr (k1 == 0) dst[u] = t[0];
        else dst[k1 * C::R2P + u] = cmul_conj(t[k1], tw.template get<k1>());
    });
}
template <class C, int J0, int J1, bool GUARD = true, class L, class TW>
QM_HD void stepB1_tail_range(const c128 (&t)[C::R2], const L line, int u, const TW &tw) {
    if constexpr (GUARD) if (u >= C::R1) return;
    static_for<J1 - J0>([&](auto I) {
        constexpr int d = J0 + decltype(I)::value;
        if constexpr (d == 0) line[u * C::R2P] = t[0];
        else line[u * C::R2P + d] = cmul(t[d], tw.template get<d>());
    });
}
template <class C, class L, class TW>
QM_HD void stepA1_tail(const c128 (&t)[C::R1], const L dst, int u, const TW &tw) { stepA1_tail_range<C, 0, C::R1>(t, dst, u, tw); }
template <class C, class L, class TW>
QM_HD void stepB1_tail(const c128 (&t)[C::R2], const L line, int u, const TW &tw) { stepB1_tail_range<C, 0, C::R2>(t, line, u, tw); }
template <class C, bool GUARD = true, class P>
QM_HD void prunedA_step1_head(const P src, int estride, const Pruned pr, c128 (&t)[C::R1], int u) {
    if constexpr (GUARD) if (u >= C::R2) return;
    const P p1 = src + pr.c1, p2 = src + pr.c2;
    const unsigned mm = pr.m1 | pr.m2;
    static_for<C::R1>([&](auto I) {
        constexpr int n1 = decltype(I)::value;
        if constexpr (2 * (n1 + 1) * C::R2 <= C::N) t[n1] = ld_pred(p1 + n1 * estride, (mm & (1u << n1)) != 0u);
        else if constexpr (2 * n1 * C::R2 >= C::N) t[n1] = ld_pred(p2 + n1 * estride, (mm & (1u << n1)) != 0u);
        else {
            const bool in2 = (pr.m2 >> n1) & 1u;
            t[n1] = ld_pred((in2 ? p2 : p1) + n1 * estride, (mm & (1u << n1)) != 0u);
        }
    });
    Dft<C::R1, +1>::run(t);
}
template <class C, class P, class L, class TW>
QM_HD void prunedA_step1(const P src, int estride, const Pruned pr, const L dst, int u, const TW &tw) {
    c128 t[C::R1];
    prunedA_step1_head<C>(src, estride, pr, t, u);
    stepA1_tail<C>(t, dst, u, tw);
}
// "Quarter" form of the pruned backward step 1: when every occupied index lies below N/4 or at/above 3N/4
// (true for every alias-free grid, 4 m + 1 <= n), only the first Q and the last Q first-pass inputs of a thread
// can exist, Q = ceil(R1 / 4).  They are fetched ahead of time into 2Q registers (prefetch_quarter) and the
// transform is started later from those registers (prunedA_step1_pre).
template <class C> struct Quarter { static constexpr int Q = (C::R1 + 3) / 4; };
template <class C, class P>
QM_HD void prefetch_quarter(const P src, int estride, const Pruned pr, c128 (&pre)[2 * Quarter<C>::Q]) {
    constexpr int Q = Quarter<C>::Q;
    const P p1 = src + pr.c1, p2 = src + pr.c2;
    static_for<Q>([&](auto I) {
        constexpr int j = decltype(I)::value;
        pre[j] = ld_pred(p1 + j * estride, (pr.m1 >> j) & 1u);
        pre[Q + j] = ld_pred(p2 + (C::R1 - Q + j) * estride, (pr.m2 >> (C::R1 - Q + j)) & 1u);
    });
}
template <class C, bool GUARD = true>
QM_HD void prunedA_step1_pre_head(const c128 (&pre)[2 * Quarter<C>::Q], c128 (&t)[C::R1], int u) {
    if constexpr (GUARD) if (u >= C::R2) return;
    constexpr int Q = Quarter<C>::Q;
    static_for<C::R1>([&](auto I) {
        constexpr int n1 = decltype(I)::value;
        if constexpr (n1 < Q) t[n1] = pre[n1];
        else if constexpr (n1 >= C::R1 - Q) t[n1] = pre[Q + n1 - (C::R1 - Q)];
        else t[n1] = c128{0.0, 0.0};
    });
    DftQuarterIn<C::R1, +1>::run(t);
}
template <class C, class L, class TW>
QM_HD void prunedA_step1_pre(const c128 (&pre)[2 * Quarter<C>::Q], const L dst, int u, const TW &tw) {
    c128 t[C::R1];
    prunedA_step1_pre_head<C>(pre, t, u);
    stepA1_tail<C>(t, dst, u, tw);
}
template <class C, class P, class L, class TW>
QM_HD void prunedA_step1_quarter(const P src, int estride, const Pruned pr, const L dst, int u, const TW &tw) {
    if (u >= C::R2) return;
    c128 pre[2 * Quarter<C>::Q];
    prefetch_quarter<C>(src, estride, pr, pre);
    prunedA_step1_pre<C>(pre, dst, u, tw);
}
// Forward step 2 with pruned output: reads the full padded line `srcline`, stores only what exists.
template <class C, bool GUARD = true, class L, class P>
QM_HD void prunedB_step2(const L srcline, const P dst, int estride, const Pruned pr, int u) {
    if constexpr (GUARD) if (u >= C::R2) return;
    c128 t[C::R1];
    static_for<C::R1>([&](auto I) { constexpr int a = decltype(I)::value; t[a] = srcline[a * C::R2P + u]; });
    Dft<C::R1, -1>::run(t);
    const P p1 = dst + pr.c1, p2 = dst + pr.c2;
    const unsigned mm = pr.m1 | pr.m2;
    static_for<C::R1>([&](auto I) {
        constexpr int c = decltype(I)::value;
        if constexpr (2 * (c + 1) * C::R2 <= C::N) st_pred(p1 + c * estride, t[c], (mm & (1u << c)) != 0u);
        else if constexpr (2 * c * C::R2 >= C::N) st_pred(p2 + c * estride, t[c], (mm & (1u << c)) != 0u);
        else {
            const bool in2 = (pr.m2 >> c) & 1u;
            st_pred((in2 ? p2 : p1) + c * estride, t[c], (mm & (1u << c)) != 0u);
        }
    });
}
// Quarter-rule form of the pruned forward step 2: only the first Q and last Q outputs of a thread can exist.
template <class C, bool GUARD = true, class L, class P>
QM_HD void prunedB_step2_quarter(const L srcline, const P dst, int estride, const Pruned pr, int u) {
    if constexpr (GUARD) if (u >= C::R2) return;
    constexpr int Q = Quarter<C>::Q;
    c128 t[C::R1];
    static_for<C::R1>([&](auto I) { constexpr int a = decltype(I)::value; t[a] = srcline[a * C::R2P + u]; });
    DftQuarterOut<C::R1, -1>::run(t);
    const P p1 = dst + pr.c1, p2 = dst + pr.c2;
    static_for<Q>([&](auto I) {
        constexpr int j = decltype(I)::value;
        constexpr int c2 = C::R1 - Q + j;
        st_pred(p1 + j * estride, t[j], (pr.m1 >> j) & 1u);
        st_pred(p2 + c2 * estride, t[c2], (pr.m2 >> c2) & 1u);
    });
}

// ---- full (unpruned) in-place passes ---------------------------------------------------------------------
template <class C, bool GUARD = true, class L> QM_HD void lineA_step2(const L line, int u) {
    if constexpr (GUARD) if (u >= C::R1) return;
    c128 t[C::R2];
    static_for<C::R2>([&](auto I) { constexpr int n2 = decltype(I)::value; t[n2] = line[u * C::R2P + n2]; });
    Dft<C::R2, +1>::run(t);
    static_for<C::R2>([&](auto I) { constexpr int k2 = decltype(I)::value; line[u * C::R2P + k2] = t[k2]; });
}
template <class C, bool GUARD = true, class L> QM_HD void lineB_step1_head(const L line, int u, c128 (&t)[C::R2]) {
    if constexpr (GUARD) if (u >= C::R1) return;
    static_for<C::R2>([&](auto I) { constexpr int b = decltype(I)::value; t[b] = line[u * C::R2P + b]; });
    Dft<C::R2, -1>::run(t);
}
template <class C, class L, class TW> QM_HD void lineB_step1(const L line, int u, const TW &tw) {
    c128 t[C::R2];
    lineB_step1_head<C>(line, u, t);
    stepB1_tail<C>(t, line, u, tw);
}

// ---- z kernels: one shared-memory round trip per stick ------------------------------------------------
// zinv pass 2: thread (stick t, row u) finishes the backward transform and writes plane labels p = u*R2 + k2
// of its stick into the staging block [N][QM_ZT] (lanes run over sticks => contiguous 16-byte stores).
template <class C, class L> QM_HD void zinv_step2_store(const L line, const L stagecol, int pstride, int u) {
    if (u >= C::R1) return;
    c128 t[C::R2];
    static_for<C::R2>([&](auto I) { constexpr int n2 = decltype(I)::value; t[n2] = line[u * C::R2P + n2]; });
    Dft<C::R2, +1>::run(t);
    static_for<C::R2>([&](auto I) { constexpr int k2 = decltype(I)::value; stagecol[(u * C::R2 + k2) * pstride] = t[k2]; });
}
// zfwd pass 1: thread (stick t, row u) reads plane labels p = u*R2 + b of its stick from the staging block and
// starts the forward transform.
template <class C, class L, class TW> QM_HD void zfwd_step1_load(const L stagecol, int pstride, const L line, int u, const TW &tw) {
    if (u >= C::R1) return;
    c128 t[C::R2];
    static_for<C::R2>([&](auto I) { constexpr int b = decltype(I)::value; t[b] = stagecol[(u * C::R2 + b) * pstride]; });
    Dft<C::R2, -1>::run(t);
    static_for<C::R2>([&](auto I) {
        constexpr int d = decltype(I)::value;
        line[u * C::R2P + d] = (d == 0) ? t[d] : cmul(t[d], tw.template get<d>());
    });
}
// zfwd pass 2: finishes the forward transform and gathers to the sphere.  What is stored for a G of this stick (GM):
//   GM_PLAIN    out[g] = F(G)                                                   (debug r2g)
//   GM_KINETIC  out[g] = F(G) + 1/2 |k+G|^2 psi_in[g]       kinetic term fused
//   GM_PHASE    out[g] = F(G) * aux[g]                      split-operator half-step, PAPER.md:1137-1139 (eq. 53)
//   GM_CONJ     out[g] = conj(F(G)) * scale                 GW matrix elements, PAPER.md:1319-1328 (eq. 56; A21)
// The per-G operand is fetched ahead of the transform (`kin`: the term to add, or the factor to multiply by).
enum { GM_PLAIN = 0, GM_KINETIC = 1, GM_PHASE = 2, GM_CONJ = 3 };
template <int GM> QM_HD c128 gather_fetch(const c128 *aux, const double *g2, int off, bool pred) {
    if constexpr (GM == GM_KINETIC) {
        const c128 x = ld_pred(aux + off, pred);
        const double h = pred ? 0.5 * g2[off] : 0.0;
        return c128{h * x.x, h * x.y};
    } else if constexpr (GM == GM_PHASE) {
        return ld_pred(aux + off, pred);
    } else {
        return c128{0.0, 0.0};
    }
}
template <int GM> QM_HD c128 gather_combine(c128 f, c128 kin, double scale) {
    if constexpr (GM == GM_KINETIC) return f + kin;
    else if constexpr (GM == GM_PHASE) return cmul(f, kin);
    else if constexpr (GM == GM_CONJ) return c128{f.x * scale, -f.y * scale};
    else return f;
}
template <class C, int GM, class L> QM_HD void zfwd_step2_gather(const L line, c128 *out, const c128 *aux, const double *g2,
                                                                  const Pruned pr, int u, double scale) {
    if (u >= C::R2) return;
    c128 t[C::R1];
    static_for<C::R1>([&](auto I) { constexpr int a = decltype(I)::value; t[a] = line[a * C::R2P + u]; });
    Dft<C::R1, -1>::run(t);
    static_for<C::R1>([&](auto I) {
        constexpr int c = decltype(I)::value;
        const bool in2 = (pr.m2 >> c) & 1u, in1 = (pr.m1 >> c) & 1u;
        const int off = (in2 ? pr.c2 : pr.c1) + c * C::R2;
        if (in1 || in2) out[off] = gather_combine<GM>(t[c], gather_fetch<GM>(aux, g2, off, true), scale);
    });
}
// Quarter-rule forms of the gather (see Quarter): the per-G operands of the <= 2Q outputs a thread can own are
// fetched ahead of the transform (prefetch_kin) and combined when the outputs are stored.
template <class C, int GM> QM_HD void prefetch_kin(const c128 *aux, const double *g2, const Pruned pr, bool active,
                                                    c128 (&kin)[2 * Quarter<C>::Q]) {
    constexpr int Q = Quarter<C>::Q;
    static_for<Q>([&](auto I) {
        constexpr int j = decltype(I)::value;
        const int o1 = pr.c1 + j * C::R2, o2 = pr.c2 + (C::R1 - Q + j) * C::R2;
        const bool q1 = active && ((pr.m1 >> j) & 1u), q2 = active && ((pr.m2 >> (C::R1 - Q + j)) & 1u);
        kin[j] = gather_fetch<GM>(aux, g2, o1, q1);
        kin[Q + j] = gather_fetch<GM>(aux, g2, o2, q2);
    });
}
template <class C, int GM, class L> QM_HD void zfwd_step2_gather_pre(const L line, c128 *out, const Pruned pr, int u,
                                                                      const c128 (&kin)[2 * Quarter<C>::Q], double scale) {
    if (u >= C::R2) return;
    constexpr int Q = Quarter<C>::Q;
    c128 t[C::R1];
    static_for<C::R1>([&](auto I) { constexpr int a = decltype(I)::value; t[a] = line[a * C::R2P + u]; });
    DftQuarterOut<C::R1, -1>::run(t);
    static_for<Q>([&](auto I) {
        constexpr int j = decltype(I)::value;
        constexpr int c2 = C::R1 - Q + j;
        st_pred(out + pr.c1 + j * C::R2, gather_combine<GM>(t[j], kin[j], scale), (pr.m1 >> j) & 1u);
        st_pred(out + pr.c2 + c2 * C::R2, gather_combine<GM>(t[c2], kin[Q + j], scale), (pr.m2 >> c2) & 1u);
    });
}

// ---- x direction of the plane kernel -----------------------------------------------------------------------
// The occupied box indices i1 form two intervals (the sphere is convex): [a1,b1] -> plane rows 0..,
// [a2,b2] -> the following rows; everything else is not stored (zero).  Steps 1 and 3 of a column are
// prunedA_step1 / prunedB_step2 on the plane array with stride = row pitch; step 2 works on the scratch line:
// MODE 0: apply  (backward step 2, multiply by v[x], forward step 1)      PAPER.md:659-662 (eq. 47)
// MODE 1: g2r    (backward step 2, write psi(r)*scale to the column of a transposed box, stop)
// MODE 2: r2g    (read the column of a transposed box -- optionally times the conjugate of a second one: the pair
//                 product phi_a(r) conj(phi_b(r)) of the GW matrix elements, PAPER.md:1319-1328 -- , forward step 1)
// MODE 4: apply with a complex field (backward step 2, multiply by f[x], forward step 1): the middle factor
//                 exp(-i dt V(r)) of the split-operator propagator, PAPER.md:1137-1139 (eq. 53)
// v: this thread's R2 potential values V(x = u + R1*k2), already in registers (prefetched by the caller).
// Transposed box ("BoxT"): element (x, y, z) at [(p * N2 + col) * N1 + x], p / col = transposed z / y labels, x natural;
// a thread's x = u + R1*k2 make the lanes of a team read contiguous 16-byte words.  box / box2 / the field point at
// element x = 0 of this column.
template <int R> struct VRow { double v[R]; };
// V of one plane column is stored in pairs: vcol[(j * R1 + u) * 2 + e] = V(x = u + R1*(2j + e)), j < R2E/2
// (R2E = R2 rounded up to even, the pad is zero), so a thread reads its R2 values with 16-byte loads and the
// lanes of a team read contiguous 16-byte words.
template <class C> struct VLayout { static constexpr int R2E = C::R2 + (C::R2 & 1), COL = C::R1 * R2E; };
template <class C> QM_HD void load_vrow(VRow<C::R2> &vr, const double *vcol, int u) {
    if (u >= C::R1) return;
    const double2 *q = reinterpret_cast<const double2 *>(vcol) + u;
    static_for<VLayout<C>::R2E / 2>([&](auto I) {
        constexpr int j = decltype(I)::value;
        const double2 d = q[j * C::R1];
        vr.v[2 * j] = d.x;
        if constexpr (2 * j + 1 < C::R2) vr.v[2 * j + 1] = d.y;
    });
}
// head: everything up to the forward radix pass (returns false in MODE 1, which stops after the backward transform);
// tail: stepB1_tail on the scratch line.
// `act` = false: a lane that stands in for nothing (GUARD = false callers): it computes on whatever it was pointed at and
// must not store to global memory.
template <class C, int MODE, bool GUARD = true, class L>
QM_HD void xcol_step2_head(const L scr, int u, const VRow<C::R2> &vr, c128 *box, const c128 *box2, double scale, c128 (&t)[C::R2],
                           bool act = true) {
    if constexpr (GUARD) if (u >= C::R1) return;
    if constexpr (MODE == 2) {
        static_for<C::R2>([&](auto I) { constexpr int k2 = decltype(I)::value; t[k2] = box[u + C::R1 * k2]; });
        if (box2) static_for<C::R2>([&](auto I) { constexpr int k2 = decltype(I)::value; t[k2] = cmul_conj(t[k2], box2[u + C::R1 * k2]); });
    } else {
        c128 f[MODE == 4 ? C::R2 : 1];
        if constexpr (MODE == 4) static_for<C::R2>([&](auto I) { constexpr int k2 = decltype(I)::value; f[k2] = box2[u + C::R1 * k2]; });
        static_for<C::R2>([&](auto I) { constexpr int n2 = decltype(I)::value; t[n2] = scr[u * C::R2P + n2]; });
        Dft<C::R2, +1>::run(t);                      // t[k2] = psi(x = u + R1*k2)
        if constexpr (MODE == 1) {
            if (act) static_for<C::R2>([&](auto I) { constexpr int k2 = decltype(I)::value; box[u + C::R1 * k2] = cscale(t[k2], scale); });
            return;
        } else if constexpr (MODE == 4) {
            static_for<C::R2>([&](auto I) { constexpr int k2 = decltype(I)::value; t[k2] = cmul(t[k2], f[k2]); });
        } else {
            static_for<C::R2>([&](auto I) { constexpr int k2 = decltype(I)::value; t[k2] = cscale(t[k2], vr.v[k2]); });
        }
    }
    Dft<C::R2, -1>::run(t);
}
template <class C, int MODE, class L, class TW>
QM_HD void xcol_step2(const L scr, int u, const TW &tw, const VRow<C::R2> &vr, c128 *box, const c128 *box2, double scale) {
    c128 t[C::R2];
    xcol_step2_head<C, MODE>(scr, u, vr, box, box2, scale, t);
    if constexpr (MODE != 1) stepB1_tail<C>(t, scr, u, tw);
}
// MODE 3 of the plane kernel (density, eq. 2): backward step 2, then rho(x) += w |psi(x)|^2 on this
// thread's R2 points.  The running density of a plane column is kept in the V layout (VLayout), so the read-modify-
// write is 16-byte and lane-contiguous; one CTA owns a plane for all bands, so the order of the sums is fixed.
template <class C, class L> QM_HD void xcol_density(const L scr, int u, double *rhocol, double w) {
    if (u >= C::R1) return;
    c128 t[C::R2];
    static_for<C::R2>([&](auto I) { constexpr int n2 = decltype(I)::value; t[n2] = scr[u * C::R2P + n2]; });
    Dft<C::R2, +1>::run(t);                          // t[k2] = psi(x = u + R1*k2)
    double2 *q = reinterpret_cast<double2 *>(rhocol) + u;
    static_for<VLayout<C>::R2E / 2>([&](auto I) {
        constexpr int j = decltype(I)::value;
        double2 d = q[j * C::R1];
        d.x = fma(w, t[2 * j].x * t[2 * j].x + t[2 * j].y * t[2 * j].y, d.x);
        if constexpr (2 * j + 1 < C::R2) d.y = fma(w, t[2 * j + 1].x * t[2 * j + 1].x + t[2 * j + 1].y * t[2 * j + 1].y, d.y);
        q[j * C::R1] = d;
    });
}
