"""ORACLE (test infrastructure, never on the product path): subspace products <psi_i|phi_j>.

The step right after h_psi in the Davidson solver: the paper's `WavefunG.vdot(psi, phi)`,
"the dot product <psi_i|phi_j>" computed there with BLAS ZGEMM.  The plain definition, written out:

    S[i, j] = sum_G conj(psi_i(G)) * phi_j(G)          (plain sum over the sphere, no volume factor: reading A10)

Explicit loops over (i, j), each sum accumulated in extended precision (np.longdouble) in the storage order of G,
so the result does not depend on a library's blocking.  Pins: tests/test_oracle_subspace.py.
"""
from __future__ import annotations

import numpy as np


def vdot_matrix(psi: np.ndarray, phi: np.ndarray) -> np.ndarray:
    """psi [na][ng], phi [nb][ng] complex128  ->  S [na][nb] complex128."""
    psi = np.asarray(psi, dtype=np.complex128)
    phi = np.asarray(phi, dtype=np.complex128)
    assert psi.ndim == 2 and phi.ndim == 2 and psi.shape[1] == phi.shape[1]
    na, nb = psi.shape[0], phi.shape[0]
    out = np.zeros((na, nb), dtype=np.complex128)
    pr, pi = psi.real.astype(np.longdouble), psi.imag.astype(np.longdouble)
    qr, qi = phi.real.astype(np.longdouble), phi.imag.astype(np.longdouble)
    for i in range(na):
        for j in range(nb):
            # conj(a) * b = (ar*br + ai*bi) + i (ar*bi - ai*br)
            re = np.sum(pr[i] * qr[j] + pi[i] * qi[j], dtype=np.longdouble)
            im = np.sum(pr[i] * qi[j] - pi[i] * qr[j], dtype=np.longdouble)
            out[i, j] = complex(float(re), float(im))
    return out
