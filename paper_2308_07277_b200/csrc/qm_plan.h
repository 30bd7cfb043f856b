// Plain-old-data plans handed to the kernels (device pointers inside).
#pragma once
#include <stdint.h>
#include <vector_types.h>

struct c128;

struct QmAxis {            // one FFT axis: n = r1 * r2
    int n, r1, r2, r2p, len;   // len = r1 * r2p (padded line length)
};

struct QmKPlanDev {        // per k-point tables on the device
    int ng;                // plane waves in the sphere
    int nsticks;           // S: (i1,i2) lines that intersect the sphere
    int nx;                // X: distinct i1 among the sticks
    int rowpitch;          // pitch of one plane row (odd, >= axis2.len)
    short4 x_iv;                 //        occupied i1 intervals [x,y] -> rows 0.., [z,w] -> following rows
    const int4 *row_info;        // [X]    per plane row: (a1 | b1<<16, a2 | b2<<16, first stick, 0): occupied i2 intervals
    const int4 *stick_info;      // [S]    per stick: (a1 | b1<<16, a2 | b2<<16, first G, 0): occupied i3 intervals
    const double *g2;            // [ng]   |k+G|^2
};

struct QmGridDev {
    QmAxis ax[3];
    const c128 *tw[3];     // tw[a][j] = exp(-2 pi i j / n_a)
    const double *vt;      // re-laid-out potential (fft_phases.cuh VLayout) * 1/(n1 n2 n3), or nullptr
};

// transposed label p -> natural index (p / r2) + r1 * (p % r2)
static inline int qm_label_to_index(const QmAxis &a, int p) { return (p / a.r2) + a.r1 * (p % a.r2); }
static inline int qm_pos(const QmAxis &a, int i) { return (i / a.r2) * a.r2p + (i % a.r2); }
