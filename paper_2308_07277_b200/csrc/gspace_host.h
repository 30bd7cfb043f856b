// Host-side set-up of one k-point: G-sphere enumeration, sphere->box index map, stick tables.
// Pure C++ (no CUDA): used by qm_api.cu and by the CPU thread-emulation test (tests/host_emu).
//   sphere:  all integer m with |k + G_m|^2 [bohr^-2] <= ecutwfc [Ry]
//   order:   ascending idx = ((m1 mod n1)*n2 + (m2 mod n2))*n3 + (m3 mod n3)
//   sticks:  the (i1,i2) lines of the box that hold at least one G
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <string>
#include <vector>
#include "qm_plan.h"

struct FftSize { int n, r1, r2; };
// supported FFT lengths and their two-pass factorisation n = r1 * r2
static const FftSize kQmSizes[] = {
    {8, 2, 4},   {12, 3, 4},  {16, 4, 4},  {18, 3, 6},  {20, 4, 5},   {24, 4, 6},   {30, 5, 6},
    {32, 4, 8},  {36, 6, 6},  {40, 5, 8},  {48, 6, 8},  {60, 6, 10},  {64, 8, 8},   {72, 8, 9},
    {80, 8, 10}, {96, 12, 8}, {100, 10, 10}, {108, 9, 12}, {120, 10, 12}, {128, 8, 16}, {144, 12, 12},
    // above 144: z kernels and the unfused xy passes only (the fused plane kernel is not compiled for them)
    {160, 10, 16}, {180, 12, 15}, {192, 12, 16}, {225, 15, 15}, {240, 15, 16}, {256, 16, 16},
};
static const int kQmFusedMax = 144;
static inline const FftSize *qm_find_size(int n) {
    for (const auto &s : kQmSizes) if (s.n == n) return &s;
    return nullptr;
}
static inline QmAxis qm_make_axis(const FftSize &s) {
    QmAxis a; a.n = s.n; a.r1 = s.r1; a.r2 = s.r2; a.r2p = s.r2 | 1; a.len = s.r1 * a.r2p; return a;
}

static inline void qm_reciprocal(const double *a, double *b) {
    // b_i = rows of 2 pi (A^-1)^T; (A^-1)^T = cofactor matrix / det
    const double c00 = a[4] * a[8] - a[5] * a[7], c01 = a[5] * a[6] - a[3] * a[8], c02 = a[3] * a[7] - a[4] * a[6];
    const double c10 = a[2] * a[7] - a[1] * a[8], c11 = a[0] * a[8] - a[2] * a[6], c12 = a[1] * a[6] - a[0] * a[7];
    const double c20 = a[1] * a[5] - a[2] * a[4], c21 = a[2] * a[3] - a[0] * a[5], c22 = a[0] * a[4] - a[1] * a[3];
    const double det = a[0] * c00 + a[1] * c01 + a[2] * c02;
    const double f = 2.0 * M_PI / det;
    b[0] = f * c00; b[1] = f * c01; b[2] = f * c02;
    b[3] = f * c10; b[4] = f * c11; b[5] = f * c12;
    b[6] = f * c20; b[7] = f * c21; b[8] = f * c22;
}

struct QmKTables {
    double k[3] = {0, 0, 0};
    int ng = 0, nsticks = 0, nx = 0, rowpitch = 0;
    int mmax[3] = {0, 0, 0};
    std::vector<int32_t> idx, miller;          // miller: ng*3
    std::vector<double> g2;
    std::vector<int32_t> stickoff;             // [S+1] first G of each stick
    std::vector<int16_t> xrow;
    std::vector<short4> rowiv;                 // per plane row: occupied i2 intervals
    std::vector<int4> rowinfo;                 // packed (a1|b1<<16, a2|b2<<16, first stick of the row, 0)
    std::vector<int4> stickinfo;               // per stick: packed occupied i3 intervals (a1|b1<<16, a2|b2<<16), first G, 0
    short4 xiv = {1, 0, 1, 0};                 // occupied i1 intervals (rows 0.. and following)
    bool x_contiguous = true;
    bool x_quarter = false;                    // the same rule for the occupied i1 (x rows of the plane kernel)
    bool z_quarter = false;                    // same rule for the occupied i3 of every stick (z kernels)
    bool y_quarter = false;                    // every occupied i2 of every row lies in the first / last quarter-block (fft_phases.cuh Quarter)
};

// returns 0, or -1 (sphere does not fit the grid) / -2 (empty sphere); msg gets the reason
// strict: keep |k+G|^2 < ecut instead of <= (the epsilon sphere of the GW matrix elements, eq. 56)
static inline int qm_build_tables(const double *lattice, const double *recip, double ecut, const int *grid,
                                  const QmAxis *ax, QmKTables *kp, std::string *msg, bool strict = false)
{
    const double *b = recip, *a = lattice;
    const int n1 = grid[0], n2 = grid[1], n3 = grid[2];
    const double qmax = std::sqrt(ecut);
    int bound[3];
    for (int i = 0; i < 3; ++i) {
        const double an = std::sqrt(a[3 * i] * a[3 * i] + a[3 * i + 1] * a[3 * i + 1] + a[3 * i + 2] * a[3 * i + 2]);
        bound[i] = (int)std::floor(qmax * an / (2.0 * M_PI) + std::fabs(kp->k[i])) + 1;
    }
    struct Ent { int64_t idx; int m[3]; double g2; };
    std::vector<Ent> ents;
    for (int m1 = -bound[0]; m1 <= bound[0]; ++m1)
        for (int m2 = -bound[1]; m2 <= bound[1]; ++m2)
            for (int m3 = -bound[2]; m3 <= bound[2]; ++m3) {
                const double f1 = m1 + kp->k[0], f2 = m2 + kp->k[1], f3 = m3 + kp->k[2];
                const double qx = f1 * b[0] + f2 * b[3] + f3 * b[6];
                const double qy = f1 * b[1] + f2 * b[4] + f3 * b[7];
                const double qz = f1 * b[2] + f2 * b[5] + f3 * b[8];
                const double q2 = qx * qx + qy * qy + qz * qz;
                if (strict ? q2 < ecut : q2 <= ecut) {
                    Ent e; e.m[0] = m1; e.m[1] = m2; e.m[2] = m3; e.g2 = q2; e.idx = 0;
                    ents.push_back(e);
                    kp->mmax[0] = std::max(kp->mmax[0], std::abs(m1));
                    kp->mmax[1] = std::max(kp->mmax[1], std::abs(m2));
                    kp->mmax[2] = std::max(kp->mmax[2], std::abs(m3));
                }
            }
    for (int i = 0; i < 3; ++i)
        if (2 * kp->mmax[i] + 1 > grid[i]) { *msg = "G-sphere does not fit the FFT grid (2|m|+1 > n)"; return -1; }
    if (ents.empty()) { *msg = "empty G-sphere"; return -2; }
    auto wrapi = [](int m, int n) { int r = m % n; return r < 0 ? r + n : r; };
    for (auto &e : ents)
        e.idx = ((int64_t)wrapi(e.m[0], n1) * n2 + wrapi(e.m[1], n2)) * n3 + wrapi(e.m[2], n3);
    std::sort(ents.begin(), ents.end(), [](const Ent &x, const Ent &y) { return x.idx < y.idx; });
    const int ng = (int)ents.size();
    kp->ng = ng;
    kp->idx.resize(ng); kp->miller.resize((size_t)ng * 3); kp->g2.resize(ng);
    kp->stickoff.clear();
    std::vector<int32_t> stick_i1, stick_i2;
    int64_t cur = -1;
    for (int i = 0; i < ng; ++i) {
        const Ent &e = ents[i];
        kp->idx[i] = (int32_t)e.idx;
        kp->miller[3 * i] = e.m[0]; kp->miller[3 * i + 1] = e.m[1]; kp->miller[3 * i + 2] = e.m[2];
        kp->g2[i] = e.g2;
        const int64_t line = e.idx / n3;
        if (line != cur) {
            cur = line;
            kp->stickoff.push_back(i);
            stick_i1.push_back((int)(line / n2));
            stick_i2.push_back((int)(line % n2));
        }
    }
    const int S = (int)kp->stickoff.size();
    kp->stickoff.push_back(ng);
    kp->nsticks = S;
    kp->xrow.assign(n1, -1);
    int nx = 0;
    for (int s = 0; s < S; ++s)
        if (kp->xrow[stick_i1[s]] < 0) kp->xrow[stick_i1[s]] = (int16_t)nx++;   // sticks ascend in i1
    kp->nx = nx;
    {   // occupied i1 intervals; rows must follow them in order (true for a convex sphere)
        short4 iv = {1, 0, 1, 0};
        for (int i1 = 0; i1 < n1; ++i1) {
            if (kp->xrow[i1] < 0) continue;
            if (2 * i1 < n1) { if (iv.x > iv.y) iv.x = (short)i1; iv.y = (short)i1; }
            else { if (iv.z > iv.w) iv.z = (short)i1; iv.w = (short)i1; }
        }
        kp->xiv = iv;
        kp->x_contiguous = true;
        const int c1 = iv.x <= iv.y ? iv.y - iv.x + 1 : 0;
        for (int i1 = 0; i1 < n1; ++i1) {
            const int want = (i1 >= iv.x && i1 <= iv.y) ? i1 - iv.x
                             : ((i1 >= iv.z && i1 <= iv.w) ? i1 - iv.z + c1 : -1);
            if (want != kp->xrow[i1]) kp->x_contiguous = false;
        }
        if (!kp->x_contiguous) { *msg = "occupied x columns are not two contiguous intervals"; return -1; }
    }
    kp->rowpitch = ax[1].len | 1;
    // occupied i2 intervals of every plane row: [0..m2max] and [n2+m2min..n2-1] (the sphere is convex, so
    // the sticks of a row are contiguous in m2); verified below, else the plane kernel zero-fills.
    kp->rowiv.assign(nx, short4{1, 0, 1, 0});
    std::vector<int> rowcount(nx, 0);
    for (int s = 0; s < S; ++s) {
        short4 &iv = kp->rowiv[kp->xrow[stick_i1[s]]];
        const int i2 = stick_i2[s];
        rowcount[kp->xrow[stick_i1[s]]]++;
        if (2 * i2 < n2) {        // non-negative m2
            if (iv.x > iv.y) { iv.x = (short)i2; iv.y = (short)i2; }
            else { iv.x = std::min<short>(iv.x, (short)i2); iv.y = std::max<short>(iv.y, (short)i2); }
        } else {
            if (iv.z > iv.w) { iv.z = (short)i2; iv.w = (short)i2; }
            else { iv.z = std::min<short>(iv.z, (short)i2); iv.w = std::max<short>(iv.w, (short)i2); }
        }
    }
    kp->rowinfo.resize(nx);
    {
        int s = 0;
        for (int r = 0; r < nx; ++r) {
            const short4 iv = kp->rowiv[r];
            const int span = (iv.x <= iv.y ? iv.y - iv.x + 1 : 0) + (iv.z <= iv.w ? iv.w - iv.z + 1 : 0);
            if (span != rowcount[r]) { *msg = "sticks of a plane row are not two contiguous intervals"; return -1; }
            kp->rowinfo[r] = int4{(int)(unsigned short)iv.x | ((int)iv.y << 16), (int)(unsigned short)iv.z | ((int)iv.w << 16), s, 0};
            s += span;      // sticks ascend in (i1, i2): the row's sticks are [s, s + span)
        }
    }
    // occupied i3 intervals of every stick: [0..m3max] and [n3+m3min..n3-1]; the G of a stick are stored in
    // ascending i3, i.e. interval 1 then interval 2 back to back (what the z kernels' pruned passes assume)
    kp->stickinfo.resize(S);
    kp->z_quarter = true;
    const int zq = (ax[2].r1 + 3) / 4;
    for (int s = 0; s < S; ++s) {
        short4 iv = {1, 0, 1, 0};
        for (int g = kp->stickoff[s]; g < kp->stickoff[s + 1]; ++g) {
            const int i3 = kp->idx[g] % n3;
            if (2 * i3 < n3) { if (iv.x > iv.y) iv.x = (short)i3; iv.y = (short)i3; }
            else { if (iv.z > iv.w) iv.z = (short)i3; iv.w = (short)i3; }
        }
        const int span = (iv.x <= iv.y ? iv.y - iv.x + 1 : 0) + (iv.z <= iv.w ? iv.w - iv.z + 1 : 0);
        if (span != kp->stickoff[s + 1] - kp->stickoff[s]) { *msg = "G of a stick are not two contiguous intervals"; return -1; }
        if (iv.x <= iv.y && iv.y >= zq * ax[2].r2) kp->z_quarter = false;
        if (iv.z <= iv.w && iv.z < (ax[2].r1 - zq) * ax[2].r2) kp->z_quarter = false;
        kp->stickinfo[s] = int4{(int)(unsigned short)iv.x | ((int)iv.y << 16), (int)(unsigned short)iv.z | ((int)iv.w << 16),
                                kp->stickoff[s], 0};
    }
    {
        const int q = (ax[0].r1 + 3) / 4;
        const short4 iv = kp->xiv;
        kp->x_quarter = !(iv.x <= iv.y && iv.y >= q * ax[0].r2) && !(iv.z <= iv.w && iv.z < (ax[0].r1 - q) * ax[0].r2);
    }
    {   // quarter rule for the plane kernel's register prefetch: i2 < Q*r2 or i2 >= (r1-Q)*r2, Q = ceil(r1/4)
        const int q = (ax[1].r1 + 3) / 4;
        kp->y_quarter = true;
        for (int r = 0; r < nx; ++r) {
            const short4 iv = kp->rowiv[r];
            if (iv.x <= iv.y && iv.y >= q * ax[1].r2) kp->y_quarter = false;
            if (iv.z <= iv.w && iv.z < (ax[1].r1 - q) * ax[1].r2) kp->y_quarter = false;
        }
    }
    return 0;
}
