/* O2: H|psi> by direct G-space summation -- CPU oracle, TEST INFRASTRUCTURE.
 *
 * Written from /root/reference/PAPER.md; shares no code with the CUDA path.
 *
 *   out_n(G) = 1/2 |k+G|^2 psi_n(G)                                   (T)  PAPER.md:146 eq.12, 668-674 eq.49-51
 *            + sum_{G' in sphere} Vhat(G - G') psi_n(G')               (L)  PAPER.md:146 eq.12, 650
 *            + sum_i beta_i(G) sum_j D_ij sum_{G'} conj(beta_j(G')) psi_n(G')
 *                                                                     (NL) PAPER.md:153-161 eq.14 (multi-projector form, A10)
 *
 * Vhat(G - G') is looked up in the FFT box at ((m - m') mod n) per component
 * (reading A8).  Every sum over G' is accumulated in long double (reading
 * A12): N_G reaches 8e4 and the parity tolerance is 1e-11.
 * No blocking, no reordering beyond "bands innermost"; OpenMP over output rows.
 *
 * Layouts: psi [nb][ng], beta [nproj][ng], out [nb][nrows], all complex128
 * interleaved (re,im); miller int32 [ng][3]; vhat complex128 [n1*n2*n3] C order;
 * D dense real [nproj][nproj].
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

static inline int wrap(int m, int n) { int r = m % n; return r < 0 ? r + n : r; }

/* P[j][n] = sum_G conj(beta_j(G)) psi_n(G), then Q = D P.  q: [nproj][nb] complex (long double pairs -> double) */
static void projections(int ng, int nb, int nproj, const double *psi, const double *beta,
                        const double *D, double *q)
{
    long double *p = (long double *)calloc((size_t)nproj * nb * 2, sizeof(long double));
    #pragma omp parallel for schedule(static)
    for (int j = 0; j < nproj; ++j) {
        const double *bj = beta + (size_t)2 * j * ng;
        for (int n = 0; n < nb; ++n) {
            const double *pn = psi + (size_t)2 * n * ng;
            long double sr = 0.0L, si = 0.0L;
            for (int g = 0; g < ng; ++g) {
                long double br = bj[2 * g], bi = bj[2 * g + 1];
                long double xr = pn[2 * g], xi = pn[2 * g + 1];
                sr += br * xr + bi * xi;          /* conj(b) * x */
                si += br * xi - bi * xr;
            }
            p[2 * ((size_t)j * nb + n)] = sr;
            p[2 * ((size_t)j * nb + n) + 1] = si;
        }
    }
    #pragma omp parallel for schedule(static)
    for (int i = 0; i < nproj; ++i)
        for (int n = 0; n < nb; ++n) {
            long double sr = 0.0L, si = 0.0L;
            for (int j = 0; j < nproj; ++j) {
                long double d = D[(size_t)i * nproj + j];
                sr += d * p[2 * ((size_t)j * nb + n)];
                si += d * p[2 * ((size_t)j * nb + n) + 1];
            }
            q[2 * ((size_t)i * nb + n)] = (double)sr;
            q[2 * ((size_t)i * nb + n) + 1] = (double)si;
        }
    free(p);
}

/* Computes out[n][r] = (H psi_n)(G_rows[r]) for r < nrows.  Returns 0. */
int oracle_hpsi_rows(int ng, int nb, const int32_t *miller, const double *g2,
                     const double *psi, const int32_t *grid, const double *vhat,
                     int nproj, const double *beta, const double *D,
                     int nrows, const int32_t *rows, double *out)
{
    const int n1 = grid[0], n2 = grid[1], n3 = grid[2];
    double *q = NULL;
    if (nproj > 0) {
        q = (double *)malloc((size_t)nproj * nb * 2 * sizeof(double));
        projections(ng, nb, nproj, psi, beta, D, q);
    }
    /* psi transposed to [ng][nb] so that "bands innermost" reads contiguously */
    double *pt = (double *)malloc((size_t)ng * nb * 2 * sizeof(double));
    for (int n = 0; n < nb; ++n)
        for (int g = 0; g < ng; ++g) {
            pt[2 * ((size_t)g * nb + n)] = psi[2 * ((size_t)n * ng + g)];
            pt[2 * ((size_t)g * nb + n) + 1] = psi[2 * ((size_t)n * ng + g) + 1];
        }
    #pragma omp parallel
    {
        long double *acc = (long double *)malloc((size_t)nb * 2 * sizeof(long double));
        #pragma omp for schedule(dynamic, 4)
        for (int r = 0; r < nrows; ++r) {
            const int g = rows[r];
            const int m1 = miller[3 * g], m2 = miller[3 * g + 1], m3 = miller[3 * g + 2];
            /* (T) */
            for (int n = 0; n < nb; ++n) {
                acc[2 * n] = 0.5L * (long double)g2[g] * (long double)pt[2 * ((size_t)g * nb + n)];
                acc[2 * n + 1] = 0.5L * (long double)g2[g] * (long double)pt[2 * ((size_t)g * nb + n) + 1];
            }
            /* (L) */
            for (int gp = 0; gp < ng; ++gp) {
                const int d1 = wrap(m1 - miller[3 * gp], n1);
                const int d2 = wrap(m2 - miller[3 * gp + 1], n2);
                const int d3 = wrap(m3 - miller[3 * gp + 2], n3);
                const size_t vi = ((size_t)d1 * n2 + d2) * n3 + d3;
                const long double vr = vhat[2 * vi], vim = vhat[2 * vi + 1];
                const double *x = pt + 2 * (size_t)gp * nb;
                for (int n = 0; n < nb; ++n) {
                    const long double xr = x[2 * n], xi = x[2 * n + 1];
                    acc[2 * n] += vr * xr - vim * xi;
                    acc[2 * n + 1] += vr * xi + vim * xr;
                }
            }
            /* (NL) */
            for (int i = 0; i < nproj; ++i) {
                const long double br = beta[2 * ((size_t)i * ng + g)];
                const long double bi = beta[2 * ((size_t)i * ng + g) + 1];
                const double *qi = q + 2 * (size_t)i * nb;
                for (int n = 0; n < nb; ++n) {
                    const long double qr = qi[2 * n], qim = qi[2 * n + 1];
                    acc[2 * n] += br * qr - bi * qim;
                    acc[2 * n + 1] += br * qim + bi * qr;
                }
            }
            for (int n = 0; n < nb; ++n) {
                out[2 * ((size_t)n * nrows + r)] = (double)acc[2 * n];
                out[2 * ((size_t)n * nrows + r) + 1] = (double)acc[2 * n + 1];
            }
        }
        free(acc);
    }
    free(pt);
    free(q);
    return 0;
}
