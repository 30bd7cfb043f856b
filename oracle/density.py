"""ORACLE (test infrastructure, never on the product path): electron density from Bloch states.

    n(r) = sum_i f_i |psi_i(r)|^2                                   PAPER.md:100 (eq. 2), 1008 ("computing the
                                                                     electron density from Bloch states")
with psi_i(r_j) = sum_{G in sphere} psi_i(G) exp(+i G.r_j)          PAPER.md:133-137 (eq. 9 sign, reading A5),
r_j = sum_a (j_a / n_a) a_a, so G.r_j = 2 pi sum_a m_a j_a / n_a (k = Gamma phase convention: the Bloch factor
exp(i k.r) has modulus one and drops out of |psi|^2).  No 1/Omega and no 1/N: the caller's `scale` carries the
normalisation (reading A20 in DESIGN.md: the paper does not fix it).

The synthesis is the plain O(N_G) sum per point, written out with explicit phases (no FFT); `points` selects which
grid points to evaluate (all of them for small grids).  Pins: tests/test_oracle_density.py.
"""
from __future__ import annotations

import numpy as np


def psi_at_points(psi: np.ndarray, miller: np.ndarray, grid, points: np.ndarray) -> np.ndarray:
    """psi [nb][ng], miller [ng][3], points [npts][3] integer grid indices -> psi(r) [nb][npts]."""
    n = np.asarray(grid, dtype=np.int64)
    m = np.asarray(miller, dtype=np.int64)
    pts = np.asarray(points, dtype=np.int64)
    out = np.empty((psi.shape[0], pts.shape[0]), dtype=np.complex128)
    for a, j in enumerate(pts):
        # phase exponent reduced exactly in integers before it becomes a float: m_a j_a mod n_a over n_a
        frac = ((m[:, 0] * j[0]) % n[0]) / n[0] + ((m[:, 1] * j[1]) % n[1]) / n[1] + ((m[:, 2] * j[2]) % n[2]) / n[2]
        ph = np.exp(2j * np.pi * frac)
        out[:, a] = (psi.astype(np.clongdouble) * ph.astype(np.clongdouble)).sum(axis=1).astype(np.complex128)
    return out


def density(psi: np.ndarray, miller: np.ndarray, occ: np.ndarray, grid, points: np.ndarray | None = None,
            scale: float = 1.0) -> np.ndarray:
    """n at `points` (default: every grid point, C order over (n1,n2,n3)) = scale * sum_i occ_i |psi_i(r)|^2."""
    if points is None:
        n1, n2, n3 = grid
        points = np.stack(np.meshgrid(np.arange(n1), np.arange(n2), np.arange(n3), indexing="ij"), axis=-1).reshape(-1, 3)
    pr = psi_at_points(psi, miller, grid, points)
    return scale * np.einsum("i,ia->a", np.asarray(occ, dtype=np.float64), np.abs(pr) ** 2)
