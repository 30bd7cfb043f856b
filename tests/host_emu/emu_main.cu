// CPU thread-emulation of the FFT-path kernels (TEST ONLY; never linked into libqm_hpsi.so).
// Runs the very same __host__ __device__ phase functions and host-built stick tables that the CUDA
// kernels use, with "for (tid ...)" loops standing in for the threads between two barriers, so the
// index logic of the pipeline can be checked against numpy on a machine without a GPU.
//
// usage: emu_main <n> <lat9.bin> <ecut> <k1> <k2> <k3> <nb> <psi.bin> <v.bin> <out_prefix>
// writes <out_prefix>.idx (int32), .g2 (the library's host |k+G|^2 table), .hloc (T+L apply, c128 [nb][ng]), .g2r (c128 [nb][n^3]), .r2g
#include <cstdio>
#include <cstdlib>
#include <string>
#include <vector>
#include "../../paper_2308_07277_b200/csrc/fft_phases.cuh"
#include "../../paper_2308_07277_b200/csrc/gspace_host.h"

template <class T> std::vector<T> slurp(const char *path) {
    FILE *f = fopen(path, "rb"); if (!f) { perror(path); exit(2); }
    fseek(f, 0, SEEK_END); long n = ftell(f); fseek(f, 0, SEEK_SET);
    std::vector<T> v(n / sizeof(T));
    if (fread(v.data(), 1, n, f) != (size_t)n) exit(2);
    fclose(f); return v;
}
template <class T> void dump(const std::string &path, const std::vector<T> &v) {
    FILE *f = fopen(path.c_str(), "wb"); fwrite(v.data(), sizeof(T), v.size(), f); fclose(f);
}

struct RowInfo { int a1, b1, a2, b2, sbase; };
struct XRows { int a1, b1, a2, b2; };

template <class C> struct Emu {
    static constexpr int LP = C::L | 1, SL = C::L | 1, TS = QM_ZT;
    const QmKTables &kp; QmAxis ax; std::vector<c128> tw;
    Emu(const QmKTables &k, QmAxis a) : kp(k), ax(a), tw(C::N) {
        for (int j = 0; j < C::N; ++j) {
            long double ang = -2.0L * 3.14159265358979323846264338327950288L * j / C::N;
            tw[j] = c128{(double)cosl(ang), (double)sinl(ang)};
        }
    }
    TwRow<C::R1> rowA(int u) { TwRow<C::R1> t; load_twrow(t, tw.data(), u, C::R2); return t; }
    TwRow<C::R2> rowB(int u) { TwRow<C::R2> t; load_twrow(t, tw.data(), u, C::R1); return t; }
    static Pruned stick_pruned(const int4 q, int u) {
        return make_pruned<C>((int)(short)(q.x & 0xffff), q.x >> 16, (int)(short)(q.y & 0xffff), q.y >> 16, u, 1);
    }
    // k_zinv for one band: psi[ng] -> W[N][S]   (same thread mappings as the kernel)
    void zinv(const c128 *psi, c128 *W) {
        const int S = kp.nsticks, nthr = TS * C::TT;
        for (int s0 = 0; s0 < S; s0 += TS) {
            const int ns = std::min(TS, S - s0);
            std::vector<c128> lines(TS * LP, c128{1e300, -1e300});
            for (int tid = 0; tid < nthr; ++tid) {
                int t = tid / C::TT, u = tid % C::TT;
                if (t < ns) {
                    const int4 q = kp.stickinfo[s0 + t];
                    if (kp.z_quarter) {
                        c128 pre[2 * Quarter<C>::Q];
                        prefetch_quarter<C>(psi + q.z, C::R2, stick_pruned(q, u), pre);
                        prunedA_step1_pre<C>(pre, qm_sline(&lines[t * LP]), u, rowA(u));
                    } else prunedA_step1<C>(psi + q.z, C::R2, stick_pruned(q, u), qm_sline(&lines[t * LP]), u, rowA(u));
                }
            }
            for (int tid = 0; tid < nthr; ++tid) {
                int t = tid % TS, u = tid / TS;
                if (t < ns) zinv_step2_store<C>(qm_sline(&lines[t * LP]), qm_sline(W + (size_t)(s0 / TS) * C::N * QM_ZT + t), QM_ZT, u);
            }
        }
    }
    void zfwd(const c128 *W, const c128 *psi_in, c128 *out, bool kinetic) {
        const int S = kp.nsticks, nthr = TS * C::TT;
        for (int s0 = 0; s0 < S; s0 += TS) {
            const int ns = std::min(TS, S - s0);
            std::vector<c128> lines(TS * LP, c128{1e300, -1e300});
            for (int tid = 0; tid < nthr; ++tid) {
                int t = tid % TS, u = tid / TS;
                if (t < ns) zfwd_step1_load<C>(qm_sline(W + (size_t)(s0 / TS) * C::N * QM_ZT + t), QM_ZT, qm_sline(&lines[t * LP]), u, rowB(u));
            }
            for (int tid = 0; tid < nthr; ++tid) {
                int t = tid / C::TT, u = tid % C::TT;
                if (t < ns) {
                    const int4 q = kp.stickinfo[s0 + t];
                    if (kp.z_quarter) {
                        c128 kin[2 * Quarter<C>::Q];
                        if (kinetic) {
                            prefetch_kin<C, GM_KINETIC>(psi_in + q.z, kp.g2.data() + q.z, stick_pruned(q, u), true, kin);
                            zfwd_step2_gather_pre<C, GM_KINETIC>(qm_sline(&lines[t * LP]), out + q.z, stick_pruned(q, u), u, kin, 1.0);
                        } else {
                            prefetch_kin<C, GM_PLAIN>(nullptr, nullptr, stick_pruned(q, u), true, kin);
                            zfwd_step2_gather_pre<C, GM_PLAIN>(qm_sline(&lines[t * LP]), out + q.z, stick_pruned(q, u), u, kin, 1.0);
                        }
                    } else if (kinetic) zfwd_step2_gather<C, GM_KINETIC>(qm_sline(&lines[t * LP]), out + q.z, psi_in + q.z, kp.g2.data() + q.z, stick_pruned(q, u), u, 1.0);
                    else zfwd_step2_gather<C, GM_PLAIN>(qm_sline(&lines[t * LP]), out + q.z, nullptr, nullptr, stick_pruned(q, u), u, 1.0);
                }
            }
        }
    }
    // k_plane for one (band, p).  vt: relaid potential; box: transposed box (fft_phases.cuh BoxT) of this band
    template <int MODE> void plane(int p, c128 *W, const double *vt, c128 *box, double scale, int ncol) {
        const int X = kp.nx, rp = kp.rowpitch, S = kp.nsticks, n3 = ax.n, nthr = ncol * C::TT;
        // A is deliberately filled with garbage: every position must be written before it is read
        std::vector<c128> A((size_t)X * rp, c128{1e300, -1e300}), scr((size_t)ncol * SL);
        auto row_info = [&](int r) {
            const int4 q = kp.rowinfo[r];
            return RowInfo{(int)(short)(q.x & 0xffff), q.x >> 16, (int)(short)(q.y & 0xffff), q.y >> 16, q.z};
        };
        const WView Wp = qm_wview(W, p, n3);
        if (MODE != 2) {
            for (int task = 0; task < X * C::TT; ++task) {
                const RowInfo ri = row_info(task / C::TT);
                const int u = task % C::TT;
                const Pruned pr = make_pruned<C>(ri.a1, ri.b1, ri.a2, ri.b2, u, 1);
                if (kp.y_quarter) prunedA_step1_quarter<C>(Wp + ri.sbase, C::R2, pr, qm_sline(&A[(task / C::TT) * rp]), u, rowA(u));
                else prunedA_step1<C>(Wp + ri.sbase, C::R2, pr, qm_sline(&A[(task / C::TT) * rp]), u, rowA(u));
            }
            for (int task = 0; task < X * C::TT; ++task) lineA_step2<C>(qm_sline(&A[(task / C::TT) * rp]), task % C::TT);
        }
        const XRows xr{kp.xiv.x, kp.xiv.y, kp.xiv.z, kp.xiv.w};
        for (int cbase = 0; cbase < C::N; cbase += ncol) {
            if (MODE != 2)
                for (int tid = 0; tid < nthr; ++tid) {
                    int c = tid / C::TT, u = tid % C::TT, col = cbase + c;
                    if (col < C::N) {
                        if (kp.x_quarter) prunedA_step1_quarter<C>(qm_sline(A.data() + C::pos(col)), C::R2 * rp, make_pruned<C>(xr.a1, xr.b1, xr.a2, xr.b2, u, rp), qm_sline(&scr[(size_t)c * SL]), u, rowA(u));
                        else prunedA_step1<C>(qm_sline(A.data() + C::pos(col)), C::R2 * rp, make_pruned<C>(xr.a1, xr.b1, xr.a2, xr.b2, u, rp), qm_sline(&scr[(size_t)c * SL]), u, rowA(u));
                    }
                }
            for (int tid = 0; tid < nthr; ++tid) {
                int c = tid / C::TT, u = tid % C::TT, col = cbase + c;
                if (col >= C::N) continue;
                VRow<C::R2> vr;
                if (MODE == 0) load_vrow<C>(vr, vt + ((size_t)p * C::N + col) * VLayout<C>::COL, u);
                c128 *bx = MODE == 0 ? nullptr : box + ((size_t)p * C::N + col) * C::N;
                xcol_step2<C, MODE>(qm_sline(&scr[(size_t)c * SL]), u, rowB(u), vr, bx, nullptr, scale);
            }
            if (MODE != 1)
                for (int tid = 0; tid < nthr; ++tid) {
                    int c = tid / C::TT, u = tid % C::TT, col = cbase + c;
                    if (col < C::N) {
                        if (kp.x_quarter) prunedB_step2_quarter<C>(qm_sline(&scr[(size_t)c * SL]), qm_sline(A.data() + C::pos(col)), C::R2 * rp, make_pruned<C>(xr.a1, xr.b1, xr.a2, xr.b2, u, rp), u);
                        else prunedB_step2<C>(qm_sline(&scr[(size_t)c * SL]), qm_sline(A.data() + C::pos(col)), C::R2 * rp, make_pruned<C>(xr.a1, xr.b1, xr.a2, xr.b2, u, rp), u);
                    }
                }
        }
        if (MODE != 1) {
            for (int task = 0; task < X * C::TT; ++task) lineB_step1<C>(qm_sline(&A[(task / C::TT) * rp]), task % C::TT, rowB(task % C::TT));
            for (int task = 0; task < X * C::TT; ++task) {
                const RowInfo ri = row_info(task / C::TT);
                const int u = task % C::TT;
                if (kp.y_quarter) prunedB_step2_quarter<C>(qm_sline(&A[(task / C::TT) * rp]), Wp + ri.sbase, C::R2, make_pruned<C>(ri.a1, ri.b1, ri.a2, ri.b2, u, 1), u);
                else prunedB_step2<C>(qm_sline(&A[(task / C::TT) * rp]), Wp + ri.sbase, C::R2, make_pruned<C>(ri.a1, ri.b1, ri.a2, ri.b2, u, 1), u);
            }
        }
    }
};

template <class C> int run(int n, const double *lat, double ecut, const double *k, int nb, const char *psi_path,
                           const char *v_path, const std::string &prefix)
{
    int grid[3] = {n, n, n};
    QmAxis ax[3];
    for (int i = 0; i < 3; ++i) ax[i] = qm_make_axis(*qm_find_size(n));
    double recip[9]; qm_reciprocal(lat, recip);
    QmKTables kp; for (int i = 0; i < 3; ++i) kp.k[i] = k[i];
    std::string msg;
    if (qm_build_tables(lat, recip, ecut, grid, ax, &kp, &msg)) { fprintf(stderr, "%s\n", msg.c_str()); return 3; }
    auto psi = slurp<c128>(psi_path);
    auto v = slurp<double>(v_path);
    if ((int)psi.size() != nb * kp.ng || (int)v.size() != n * n * n) { fprintf(stderr, "size mismatch ng=%d\n", kp.ng); return 4; }
    const size_t n3 = (size_t)n * n * n;
    const int r2e = VLayout<C>::R2E, colsz = VLayout<C>::COL;
    std::vector<double> vt((size_t)n * n * colsz, 0.0);
    for (size_t i = 0; i < vt.size(); ++i) {
        int e = i % colsz, u = (e >> 1) % ax[0].r1, k2 = 2 * ((e >> 1) / ax[0].r1) + (e & 1), col = (i / colsz) % n, p = i / ((size_t)colsz * n);
        int x = u + ax[0].r1 * k2;
        int y = (col / ax[1].r2) + ax[1].r1 * (col % ax[1].r2), z = (p / ax[2].r2) + ax[2].r1 * (p % ax[2].r2);
        if (k2 < ax[0].r2) vt[i] = v[((size_t)x * n + y) * n + z] / (double)n3;
    }
    Emu<C> emu(kp, ax[2]);
    const int S = kp.nsticks, ncol = 5;     // odd column count on purpose: exercises the ragged last pass
    std::vector<c128> hloc((size_t)nb * kp.ng), g2r(nb * n3), r2g((size_t)nb * kp.ng), W((size_t)n * ((S + QM_ZT - 1) / QM_ZT) * QM_ZT);
    for (int b = 0; b < nb; ++b) {
        emu.zinv(&psi[(size_t)b * kp.ng], W.data());
        for (int p = 0; p < n; ++p) emu.template plane<0>(p, W.data(), vt.data(), nullptr, 1.0, ncol);
        emu.zfwd(W.data(), &psi[(size_t)b * kp.ng], &hloc[(size_t)b * kp.ng], true);
        emu.zinv(&psi[(size_t)b * kp.ng], W.data());
        for (int p = 0; p < n; ++p) emu.template plane<1>(p, W.data(), nullptr, &g2r[b * n3], 1.0 / (double)n3, ncol);
        for (int p = 0; p < n; ++p) emu.template plane<2>(p, W.data(), nullptr, &g2r[b * n3], 1.0, ncol);
        emu.zfwd(W.data(), nullptr, &r2g[(size_t)b * kp.ng], false);
    }
    {   // the emulated planes wrote / read transposed boxes: bring g2r back to natural C order for the comparison
        std::vector<c128> nat(g2r.size());
        for (int b = 0; b < nb; ++b)
            for (int p = 0; p < n; ++p)
                for (int col = 0; col < n; ++col)
                    for (int x = 0; x < n; ++x) {
                        const int y = (col / ax[1].r2) + ax[1].r1 * (col % ax[1].r2), z = (p / ax[2].r2) + ax[2].r1 * (p % ax[2].r2);
                        nat[b * n3 + ((size_t)x * n + y) * n + z] = g2r[b * n3 + ((size_t)p * n + col) * n + x];
                    }
        g2r.swap(nat);
    }
    dump(prefix + ".idx", kp.idx); dump(prefix + ".g2", kp.g2); dump(prefix + ".hloc", hloc); dump(prefix + ".g2r", g2r); dump(prefix + ".r2g", r2g);
    printf("ng %d sticks %d nx %d quarter x%d y%d z%d\n", kp.ng, kp.nsticks, kp.nx, (int)kp.x_quarter, (int)kp.y_quarter, (int)kp.z_quarter);
    return 0;
}

int main(int argc, char **argv) {
    if (argc != 11) { fprintf(stderr, "usage\n"); return 1; }
    const int n = atoi(argv[1]);
    auto lat = slurp<double>(argv[2]);
    const double ecut = atof(argv[3]);
    const double k[3] = {atof(argv[4]), atof(argv[5]), atof(argv[6])};
    const int nb = atoi(argv[7]);
    switch (n) {
#define X(N, A, B) case N: return run<LineCfg<A, B>>(n, lat.data(), ecut, k, nb, argv[8], argv[9], argv[10]);
        X(8, 2, 4) X(12, 3, 4) X(16, 4, 4) X(18, 3, 6) X(20, 4, 5) X(24, 4, 6) X(30, 5, 6) X(32, 4, 8)
        X(36, 6, 6) X(40, 5, 8) X(48, 6, 8) X(60, 6, 10) X(64, 8, 8) X(72, 8, 9) X(80, 8, 10)
        X(96, 12, 8) X(100, 10, 10) X(108, 9, 12) X(120, 10, 12) X(128, 8, 16) X(144, 12, 12)
        X(160, 10, 16) X(180, 12, 15) X(192, 12, 16) X(225, 15, 15) X(240, 15, 16) X(256, 16, 16)
#undef X
    }
    fprintf(stderr, "unsupported n\n");
    return 1;
}
