// In-register complex128 DFT codelets (radix 2,3,4,5 and their composites) for sm_100a.
// Sign convention: DIR = -1 forward  e^{-2 pi i jk/R}  (r -> G),
//                  DIR = +1 backward e^{+2 pi i jk/R}  (G -> r, eq. 9).
// Everything is resolved at compile time (static indices only) so the arrays live in registers.
#pragma once
#include <utility>
#include "roots_gen.cuh"

#ifndef QM_HD
#define QM_HD __host__ __device__ __forceinline__
#endif

struct __align__(16) c128 { double x, y; };

QM_HD c128 operator+(c128 a, c128 b) { return {a.x + b.x, a.y + b.y}; }
QM_HD c128 operator-(c128 a, c128 b) { return {a.x - b.x, a.y - b.y}; }
QM_HD c128 cmul(c128 a, c128 b) {
    return {a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x};
}
QM_HD c128 cmul_conj(c128 a, c128 b) {   // a * conj(b)
    return {a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y};
}
QM_HD c128 cscale(c128 a, double s) { return {a.x * s, a.y * s}; }

// multiply by (DIR * i)
template <int DIR> QM_HD c128 mul_i(c128 a) {
    if constexpr (DIR > 0) return {-a.y, a.x};
    else return {a.y, -a.x};
}

template <class F, int... I>
QM_HD void static_for_impl(F &&f, std::integer_sequence<int, I...>) {
    (f(std::integral_constant<int, I>{}), ...);
}
template <int N, class F> QM_HD void static_for(F &&f) {
    static_for_impl(f, std::make_integer_sequence<int, N>{});
}

// a * exp(DIR * 2 pi i J / R), J and R compile-time
template <int R, int J, int DIR> QM_HD c128 mul_root(c128 a) {
    constexpr int j = ((J % R) + R) % R;
    if constexpr (j == 0) return a;
    else if constexpr (2 * j == R) return {-a.x, -a.y};
    else if constexpr (4 * j == R) return mul_i<DIR>(a);
    else if constexpr (4 * j == 3 * R) return mul_i<-DIR>(a);
    else {
        constexpr double c = qm_cos2pi(j, R);
        constexpr double s = (DIR > 0 ? 1.0 : -1.0) * qm_sin2pi(j, R);
        return {a.x * c - a.y * s, a.x * s + a.y * c};
    }
}

template <int R, int DIR> struct Dft;

template <int DIR> struct Dft<1, DIR> {
    static QM_HD void run(c128 (&)[1]) {}
};
template <int DIR> struct Dft<2, DIR> {
    static QM_HD void run(c128 (&x)[2]) {
        c128 a = x[0], b = x[1];
        x[0] = a + b; x[1] = a - b;
    }
};
template <int DIR> struct Dft<3, DIR> {
    static QM_HD void run(c128 (&x)[3]) {
        constexpr double s3 = 0.8660254037844386;   // sqrt(3)/2
        c128 t1 = x[1] + x[2];
        c128 t2 = {x[0].x - 0.5 * t1.x, x[0].y - 0.5 * t1.y};
        c128 d = x[1] - x[2];
        c128 t3 = mul_i<DIR>(c128{s3 * d.x, s3 * d.y});
        x[0] = x[0] + t1;
        x[1] = t2 + t3;
        x[2] = t2 - t3;
    }
};
template <int DIR> struct Dft<4, DIR> {
    static QM_HD void run(c128 (&x)[4]) {
        c128 s02 = x[0] + x[2], d02 = x[0] - x[2];
        c128 s13 = x[1] + x[3], d13 = mul_i<DIR>(x[1] - x[3]);
        x[0] = s02 + s13; x[2] = s02 - s13;
        x[1] = d02 + d13; x[3] = d02 - d13;
    }
};
template <int DIR> struct Dft<5, DIR> {
    static QM_HD void run(c128 (&x)[5]) {
        constexpr double c1 = qm_cos2pi(1, 5), c2 = qm_cos2pi(2, 5);
        constexpr double s1 = qm_sin2pi(1, 5), s2 = qm_sin2pi(2, 5);
        c128 a14 = x[1] + x[4], d14 = x[1] - x[4];
        c128 a23 = x[2] + x[3], d23 = x[2] - x[3];
        c128 p1 = {x[0].x + c1 * a14.x + c2 * a23.x, x[0].y + c1 * a14.y + c2 * a23.y};
        c128 p2 = {x[0].x + c2 * a14.x + c1 * a23.x, x[0].y + c2 * a14.y + c1 * a23.y};
        c128 q1 = mul_i<DIR>(c128{s1 * d14.x + s2 * d23.x, s1 * d14.y + s2 * d23.y});
        c128 q2 = mul_i<DIR>(c128{s2 * d14.x - s1 * d23.x, s2 * d14.y - s1 * d23.y});
        x[0] = x[0] + a14 + a23;
        x[1] = p1 + q1; x[4] = p1 - q1;
        x[2] = p2 + q2; x[3] = p2 - q2;
    }
};

// R = RA * RB, input index n = n1*RB + n2, output index k = k1 + RA*k2 (natural order in place).
template <int RA, int RB, int DIR> struct DftComposite {
    static constexpr int R = RA * RB;
    static QM_HD void run(c128 (&x)[R]) {
        c128 y[R];
        static_for<RB>([&](auto N2) {
            constexpr int n2 = decltype(N2)::value;
            c128 t[RA];
            static_for<RA>([&](auto N1) { constexpr int n1 = decltype(N1)::value; t[n1] = x[n1 * RB + n2]; });
            Dft<RA, DIR>::run(t);
            static_for<RA>([&](auto K1) {
                constexpr int k1 = decltype(K1)::value;
                y[k1 * RB + n2] = mul_root<R, n2 * k1, DIR>(t[k1]);
            });
        });
        static_for<RA>([&](auto K1) {
            constexpr int k1 = decltype(K1)::value;
            c128 t[RB];
            static_for<RB>([&](auto N2) { constexpr int n2 = decltype(N2)::value; t[n2] = y[k1 * RB + n2]; });
            Dft<RB, DIR>::run(t);
            static_for<RB>([&](auto K2) { constexpr int k2 = decltype(K2)::value; x[k1 + RA * k2] = t[k2]; });
        });
    }
};

// Good-Thomas prime-factor form for coprime RA, RB: no internal twiddles at all.
//   n = (RB*n1 + RA*n2) mod R,   k = (RB*(RB^-1 mod RA)*k1 + RA*(RA^-1 mod RB)*k2) mod R
//   => w_R^{nk} = w_RA^{n1 k1} * w_RB^{n2 k2}
__host__ __device__ constexpr int qm_modinv(int a, int m) { for (int x = 1; x < m; ++x) if ((a * x) % m == 1) return x; return 1; }
template <int RA, int RB, int DIR> struct DftPFA {
    static constexpr int R = RA * RB;
    static constexpr int EA = RB * qm_modinv(RB % RA, RA), EB = RA * qm_modinv(RA % RB, RB);
    static QM_HD void run(c128 (&x)[R]) {
        c128 y[R];
        static_for<RB>([&](auto N2) {
            constexpr int n2 = decltype(N2)::value;
            c128 t[RA];
            static_for<RA>([&](auto N1) { constexpr int n1 = decltype(N1)::value; t[n1] = x[(RB * n1 + RA * n2) % R]; });
            Dft<RA, DIR>::run(t);
            static_for<RA>([&](auto K1) { constexpr int k1 = decltype(K1)::value; y[k1 * RB + n2] = t[k1]; });
        });
        static_for<RA>([&](auto K1) {
            constexpr int k1 = decltype(K1)::value;
            c128 t[RB];
            static_for<RB>([&](auto N2) { constexpr int n2 = decltype(N2)::value; t[n2] = y[k1 * RB + n2]; });
            Dft<RB, DIR>::run(t);
            static_for<RB>([&](auto K2) { constexpr int k2 = decltype(K2)::value; x[(EA * k1 + EB * k2) % R] = t[k2]; });
        });
    }
};

template <int DIR> struct Dft<6, DIR> { static QM_HD void run(c128 (&x)[6]) { DftPFA<2, 3, DIR>::run(x); } };
template <int DIR> struct Dft<8, DIR> { static QM_HD void run(c128 (&x)[8]) { DftComposite<2, 4, DIR>::run(x); } };
template <int DIR> struct Dft<9, DIR> { static QM_HD void run(c128 (&x)[9]) { DftComposite<3, 3, DIR>::run(x); } };
template <int DIR> struct Dft<10, DIR> { static QM_HD void run(c128 (&x)[10]) { DftPFA<2, 5, DIR>::run(x); } };
template <int DIR> struct Dft<12, DIR> { static QM_HD void run(c128 (&x)[12]) { DftPFA<3, 4, DIR>::run(x); } };
template <int DIR> struct Dft<15, DIR> { static QM_HD void run(c128 (&x)[15]) { DftPFA<3, 5, DIR>::run(x); } };
template <int DIR> struct Dft<16, DIR> { static QM_HD void run(c128 (&x)[16]) { DftComposite<4, 4, DIR>::run(x); } };

// ---- quarter-pruned codelets -------------------------------------------------------------------------------
// On an alias-free grid only the first and last quarter of a line's first-pass inputs (backward) / last-pass
// outputs (forward) exist (fft_phases.cuh, Quarter).  For radix 12 that is indices {0,1,2,9,10,11}: the six middle
// inputs are exact zeros, the six middle outputs are never stored.  The prime-factor forms below skip the work on
// them (72 and 80 FP64 instructions instead of 96); other radices fall back to the full codelet.
template <int R, int DIR> struct DftQuarterIn  { static QM_HD void run(c128 (&x)[R]) { Dft<R, DIR>::run(x); } };
template <int R, int DIR> struct DftQuarterOut { static QM_HD void run(c128 (&x)[R]) { Dft<R, DIR>::run(x); } };

// x[3..8] are zero on entry (their values are ignored); all 12 outputs are produced.
template <int DIR> struct DftQuarterIn<12, DIR> {
    static QM_HD void run(c128 (&x)[12]) {
        constexpr double s3 = (DIR > 0 ? 1.0 : -1.0) * 0.8660254037844386;     // Im w, w = exp(DIR 2 pi i / 3)
        // PFA 3x4, stage 1: DFT3 over n1 of x[(4 n1 + 3 n2) % 12]; y[k1][n2]
        c128 y[3][4];
        // n2 = 0: (x0, 0, 0)
        y[0][0] = x[0]; y[1][0] = x[0]; y[2][0] = x[0];
        {   // n2 = 1: (0, 0, c = x11):  X0 = c, X1 = c w^2, X2 = c w
            const c128 c = x[11];
            const c128 h = {-0.5 * c.x, -0.5 * c.y};
            y[0][1] = c;
            y[1][1] = {h.x + s3 * c.y, h.y - s3 * c.x};
            y[2][1] = {h.x - s3 * c.y, h.y + s3 * c.x};
        }
        {   // n2 = 2: (0, b = x10, c = x2):  X0 = b + c, X1 = b w + c w^2, X2 = b w^2 + c w
            const c128 s = x[10] + x[2], d = x[10] - x[2];
            const c128 h = {-0.5 * s.x, -0.5 * s.y};
            y[0][2] = s;
            y[1][2] = {h.x - s3 * d.y, h.y + s3 * d.x};
            y[2][2] = {h.x + s3 * d.y, h.y - s3 * d.x};
        }
        {   // n2 = 3: (a = x9, b = x1, 0):  X0 = a + b, X1 = a + b w, X2 = a + b w^2
            const c128 a = x[9], b = x[1];
            const c128 h = {a.x - 0.5 * b.x, a.y - 0.5 * b.y};
            y[0][3] = a + b;
            y[1][3] = {h.x - s3 * b.y, h.y + s3 * b.x};
            y[2][3] = {h.x + s3 * b.y, h.y - s3 * b.x};
        }
        // stage 2: DFT4 over n2, output index (4 k1 + 9 k2) % 12
        static_for<3>([&](auto K1) {
            constexpr int k1 = decltype(K1)::value;
            c128 t[4] = {y[k1][0], y[k1][1], y[k1][2], y[k1][3]};
            Dft<4, DIR>::run(t);
            static_for<4>([&](auto K2) { constexpr int k2 = decltype(K2)::value; x[(4 * k1 + 9 * k2) % 12] = t[k2]; });
        });
    }
};

// all 12 inputs are used; only x[0,1,2,9,10,11] hold results on exit (the others are unspecified).
template <int DIR> struct DftQuarterOut<12, DIR> {
    static QM_HD void run(c128 (&x)[12]) {
        constexpr double s3 = (DIR > 0 ? 1.0 : -1.0) * 0.8660254037844386;
        // PFA 4x3, stage 1: DFT4 over n1 of x[(3 n1 + 4 n2) % 12]; y[k1][n2]
        c128 y[4][3];
        static_for<3>([&](auto N2) {
            constexpr int n2 = decltype(N2)::value;
            c128 t[4];
            static_for<4>([&](auto N1) { constexpr int n1 = decltype(N1)::value; t[n1] = x[(3 * n1 + 4 * n2) % 12]; });
            Dft<4, DIR>::run(t);
            static_for<4>([&](auto K1) { constexpr int k1 = decltype(K1)::value; y[k1][n2] = t[k1]; });
        });
        // stage 2: DFT3 over n2 for each k1, output index (9 k1 + 4 k2) % 12; needed (k1,k2):
        //   0:(0,0)  1:(1,1)  2:(2,2)  9:(1,0)  10:(2,1)  11:(3,2)
        x[0] = y[0][0] + y[0][1] + y[0][2];
        {   // k1 = 1: k2 = 0 -> 9, k2 = 1 -> 1
            const c128 a = y[1][0], s = y[1][1] + y[1][2], d = y[1][1] - y[1][2];
            const c128 h = {a.x - 0.5 * s.x, a.y - 0.5 * s.y};
            x[9] = a + s;
            x[1] = {h.x - s3 * d.y, h.y + s3 * d.x};
        }
        {   // k1 = 2: k2 = 1 -> 10, k2 = 2 -> 2
            const c128 a = y[2][0], s = y[2][1] + y[2][2], d = y[2][1] - y[2][2];
            const c128 h = {a.x - 0.5 * s.x, a.y - 0.5 * s.y};
            x[10] = {h.x - s3 * d.y, h.y + s3 * d.x};
            x[2] = {h.x + s3 * d.y, h.y - s3 * d.x};
        }
        {   // k1 = 3: k2 = 2 -> 11
            const c128 a = y[3][0], s = y[3][1] + y[3][2], d = y[3][1] - y[3][2];
            x[11] = {a.x - 0.5 * s.x + s3 * d.y, a.y - 0.5 * s.y - s3 * d.x};
        }
    }
};

// Radix 8 (grids 64, 72, 80, 96, 128): existing inputs / wanted outputs are {0,1,6,7}.  Composite 2x4 form of Dft<8>
// with the work on the zero inputs (40 instead of 56 FP64 instructions) or on the unwanted outputs (48) removed.
template <int DIR> struct DftQuarterIn<8, DIR> {
    static QM_HD void run(c128 (&x)[8]) {
        // stage 1: DFT2 over n1 of (x[n2], x[4+n2]) with one of the two zero, then the root w8^(n2*k1)
        c128 y[2][4];
        y[0][0] = x[0];                 y[1][0] = x[0];
        y[0][1] = x[1];                 y[1][1] = mul_root<8, 1, DIR>(x[1]);
        y[0][2] = x[6];                 y[1][2] = mul_root<8, 2, DIR>(c128{-x[6].x, -x[6].y});
        y[0][3] = x[7];                 y[1][3] = mul_root<8, 3, DIR>(c128{-x[7].x, -x[7].y});
        static_for<2>([&](auto K1) {
            constexpr int k1 = decltype(K1)::value;
            c128 t[4] = {y[k1][0], y[k1][1], y[k1][2], y[k1][3]};
            Dft<4, DIR>::run(t);
            static_for<4>([&](auto K2) { constexpr int k2 = decltype(K2)::value; x[k1 + 2 * k2] = t[k2]; });
        });
    }
};
template <int DIR> struct DftQuarterOut<8, DIR> {
    static QM_HD void run(c128 (&x)[8]) {
        c128 y[2][4];
        static_for<4>([&](auto N2) {
            constexpr int n2 = decltype(N2)::value;
            const c128 a = x[n2], b = x[4 + n2];
            y[0][n2] = a + b;
            y[1][n2] = mul_root<8, n2, DIR>(a - b);
        });
        // stage 2: DFT4 over n2, outputs k = k1 + 2 k2 wanted for k2 in {0, 3} only:  X0 = (a+c)+(b+d),  X3 = (a-c) - DIR i (b-d)
        static_for<2>([&](auto K1) {
            constexpr int k1 = decltype(K1)::value;
            const c128 s02 = y[k1][0] + y[k1][2], d02 = y[k1][0] - y[k1][2];
            const c128 s13 = y[k1][1] + y[k1][3], d13 = mul_i<DIR>(y[k1][1] - y[k1][3]);
            x[k1] = s02 + s13;
            x[k1 + 6] = d02 - d13;
        });
    }
};
