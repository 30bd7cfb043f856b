"""O3: naive discrete Fourier transforms written from the definition (oracle; test infrastructure).

Sign/scale convention (eq. 9; reading A5):
  r2g (forward):   F(m) = sum_j f(j) exp(-2 pi i sum_a m_a j_a / n_a)          (unnormalised)
  g2r (backward):  f(j) = (1/N) sum_m F(m) exp(+2 pi i sum_a m_a j_a / n_a)
Separable O(N^4) evaluation with explicit DFT matrices; used only on small boxes.
"""
from __future__ import annotations

import numpy as np


def dft_matrix(n: int, sign: int) -> np.ndarray:
    j = np.arange(n)
    # reduce j*m mod n in integers first so the phase argument stays exact
    jm = (j[:, None] * j[None, :]) % n
    return np.exp(sign * 2j * np.pi * jm / n)


def naive_dftn(f: np.ndarray, sign: int = -1) -> np.ndarray:
    """Unnormalised 3-D DFT by three explicit matrix products."""
    n1, n2, n3 = f.shape
    w1, w2, w3 = dft_matrix(n1, sign), dft_matrix(n2, sign), dft_matrix(n3, sign)
    return np.einsum("ai,bj,ck,ijk->abc", w1, w2, w3, f.astype(np.complex128), optimize=True)


def naive_dftn_pointwise(f: np.ndarray, m, sign: int = -1) -> complex:
    """One output coefficient of the 3-D DFT by the plain triple sum (pure loops)."""
    n1, n2, n3 = f.shape
    acc = 0.0 + 0.0j
    for i in range(n1):
        for j in range(n2):
            for k in range(n3):
                ph = (m[0] * i) / n1 + (m[1] * j) / n2 + (m[2] * k) / n3
                acc += f[i, j, k] * np.exp(sign * 2j * np.pi * ph)
    return acc
