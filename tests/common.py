"""Shared helpers for the GPU parity tests: build a config's inputs once and hand them to both sides."""
from __future__ import annotations

import functools

import numpy as np

from oracle import gsphere as og
from oracle import hpsi as oh
from workloads import CONFIGS, cell_for, make_beta, make_dmatrix, make_kpoints, make_psi, make_vloc

TOL = 1e-11   # BASELINE.json north_star: max relative error per band (A13)


@functools.lru_cache(maxsize=None)
def problem(name: str, ik: int = 0, nbands: int | None = None, orthonormalise: bool = True):
    cfg = CONFIGS[name]
    lat, pos = cell_for(cfg)
    kpts = make_kpoints(cfg)
    k = kpts[ik]
    miller, idx, g2 = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid, k)
    v = make_vloc(cfg, lat)
    beta = make_beta(cfg, lat, pos, k, miller)
    dblk = make_dmatrix(cfg)
    psi = make_psi(cfg, ik, idx.size, nbands=nbands, orthonormalise=orthonormalise)
    return dict(cfg=cfg, lat=lat, pos=pos, kpts=kpts, k=k, miller=miller, idx=idx, g2=g2, v=v,
                vhat=oh.vhat_box(v, cfg.grid), beta=beta, dblk=dblk, psi=psi)


def band_errors(got: np.ndarray, ref: np.ndarray):
    """A13: per band max|d|/max|ref| and ||d||2/||ref||2; returns the worst of each."""
    d = np.abs(got - ref)
    e_inf = np.max(d, axis=1) / np.max(np.abs(ref), axis=1)
    e_2 = np.linalg.norm(got - ref, axis=1) / np.linalg.norm(ref, axis=1)
    return float(np.max(e_inf)), float(np.max(e_2))


def exact_g2(lattice, k_cryst, miller):
    """|k + G_m|^2 evaluated exactly (independent of both the oracle and the library): the lattice entries and k
    are doubles, hence exact rationals; B / 2 pi = (A^-1)^T is inverted in rational arithmetic (fractions), the
    quadratic form is summed exactly, and only the final factor (2 pi)^2 is applied in 60-digit arithmetic
    (mpmath) before ONE rounding to double.  Returns (g2_exact float64[ng], scale float64[ng]) where
    scale = sum_j (sum_i |f_i| |b_ij|)^2 is the magnitude the rounding errors of any double evaluation of
    q_j = sum_i f_i b_ij scale with (it equals g2 when no cancellation occurs, e.g. for orthogonal cells)."""
    from fractions import Fraction
    import mpmath
    mpmath.mp.dps = 60
    a = [[Fraction(float(x)) for x in row] for row in np.asarray(lattice, dtype=np.float64).reshape(3, 3)]
    det = (a[0][0] * (a[1][1] * a[2][2] - a[1][2] * a[2][1]) - a[0][1] * (a[1][0] * a[2][2] - a[1][2] * a[2][0])
           + a[0][2] * (a[1][0] * a[2][1] - a[1][1] * a[2][0]))

    def cof(i, j):
        r = [x for x in range(3) if x != i]
        c = [x for x in range(3) if x != j]
        return (-1) ** (i + j) * (a[r[0]][c[0]] * a[r[1]][c[1]] - a[r[0]][c[1]] * a[r[1]][c[0]])

    binv = [[cof(i, j) / det for j in range(3)] for i in range(3)]      # (A^-1)^T = cofactor matrix / det
    kf = [Fraction(float(x)) for x in np.asarray(k_cryst, dtype=np.float64).reshape(3)]
    four_pi2 = 4 * mpmath.pi ** 2
    out = np.empty(len(miller))
    scale = np.empty(len(miller))
    for n, m in enumerate(np.asarray(miller)):
        f = [Fraction(int(m[i])) + kf[i] for i in range(3)]
        q = [sum(f[i] * binv[i][j] for i in range(3)) for j in range(3)]
        s = sum(x * x for x in q)
        out[n] = float(four_pi2 * mpmath.mpf(s.numerator) / mpmath.mpf(s.denominator))
        qa = [sum(abs(f[i]) * abs(binv[i][j]) for i in range(3)) for j in range(3)]
        sa = sum(x * x for x in qa)
        scale[n] = float(four_pi2 * mpmath.mpf(sa.numerator) / mpmath.mpf(sa.denominator))
    return out, scale


# A14: a double evaluation of |k+G|^2 = sum_j (sum_i f_i b_ij)^2 makes, per component j, <= 6 roundings in b_ij
# (cofactor, determinant, quotient, 2 pi), 3 products and 2 sums, then 3 squares and 2 sums: first-order bound
# (2 * 9 + 3) u * scale = 21 u * scale, u = 2^-53; G2_TOL_U = 32 leaves room for LAPACK's inverse and second-order terms.
G2_TOL_U = 32.0
UNIT_ROUNDOFF = 2.0 ** -53
