"""O1: reciprocal lattice, G-sphere, sphere->box index map (oracle; test infrastructure).

Follows PAPER.md:149 (|k+G|^2/2 <= E_cut), PAPER.md:625-631 (reciprocal axes
printed for the bcc example), PAPER.md:689-712 (GSpace attributes, printed
listing) and PAPER.md:725-730 (``fftn(...).take(idxgrid)``: C-order flat box
index).  Readings A1-A4, A7 of SURVEY.md 8(c) / DESIGN.md section 3.
"""
from __future__ import annotations

import math
import numpy as np


def reciprocal_lattice(lattice: np.ndarray) -> np.ndarray:
    """Rows b_i with a_i . b_j = 2 pi delta_ij, i.e. B = 2 pi (A^-1)^T  (PAPER.md:625-631 prints the
    three axes of the bcc example; the defining relation is the one above)."""
    a = np.asarray(lattice, dtype=np.float64).reshape(3, 3)
    return 2.0 * math.pi * np.linalg.inv(a).T


def gsphere(lattice, ecut_ry: float, grid, k_cryst=(0.0, 0.0, 0.0), strict: bool = False):
    """All integer m with |k + G_m|^2 [bohr^-2] <= ecut [Ry]  (== q^2/2 <= E_cut Ha); `strict` selects `<`
    (the epsilon sphere of PAPER.md:1319-1321, eq. 56, is printed with a strict inequality).

    Returns (miller int32[ng,3], idx int32[ng], g2 float64[ng]) sorted by
    ascending C-order flat box index
        idx = ((m1 mod n1)*n2 + (m2 mod n2))*n3 + (m3 mod n3)
    Raises ValueError if the sphere does not fit the grid (2|m_i|+1 > n_i).
    """
    a = np.asarray(lattice, dtype=np.float64).reshape(3, 3)
    b = reciprocal_lattice(a)
    k = np.asarray(k_cryst, dtype=np.float64).reshape(3)
    n1, n2, n3 = (int(x) for x in grid)
    qmax = math.sqrt(ecut_ry)
    # |m_i + k_i| = |q . a_i| / 2pi <= |q| |a_i| / 2pi
    bound = [int(math.floor(qmax * np.linalg.norm(a[i]) / (2 * math.pi) + abs(k[i]))) + 1
             for i in range(3)]
    r1 = np.arange(-bound[0], bound[0] + 1)
    r2 = np.arange(-bound[1], bound[1] + 1)
    r3 = np.arange(-bound[2], bound[2] + 1)
    M1, M2, M3 = np.meshgrid(r1, r2, r3, indexing="ij")
    m = np.stack([M1.ravel(), M2.ravel(), M3.ravel()], axis=1)
    q = (m.astype(np.float64) + k[None, :]) @ b          # Cartesian k + G_m, rows
    g2 = q[:, 0] * q[:, 0] + q[:, 1] * q[:, 1] + q[:, 2] * q[:, 2]
    keep = (g2 < ecut_ry) if strict else (g2 <= ecut_ry)
    m = m[keep]
    g2 = g2[keep]
    for i, n in enumerate((n1, n2, n3)):
        if m.shape[0] and 2 * int(np.max(np.abs(m[:, i]))) + 1 > n:
            raise ValueError(f"G-sphere does not fit FFT grid along axis {i}")
    idx = ((m[:, 0] % n1) * n2 + (m[:, 1] % n2)) * n3 + (m[:, 2] % n3)
    order = np.argsort(idx, kind="stable")
    return (m[order].astype(np.int32), idx[order].astype(np.int32), g2[order])


def min_grid(miller: np.ndarray):
    """Smallest n_i with 2*max|m_i|+1 <= n_i (the grid rule behind PAPER.md:700-701)."""
    return tuple(2 * int(np.max(np.abs(miller[:, i]))) + 1 for i in range(3))
