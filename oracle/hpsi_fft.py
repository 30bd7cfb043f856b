"""The paper's own CPU method for the local term, with library FFTs (oracle side; test infrastructure).

  psi(G) --scatter, IFFT--> psi(r);  (V psi)(r) = V(r) psi(r);  --FFT, take(idx)--> (V psi)(G)
                                                    PAPER.md:652-666 (eqs. 46-48), 725-730
  kinetic 1/2|k+G|^2 psi(G); projectors as two matrix products
  ("directly calls ZGEMM").
By the circular convolution theorem this equals the direct sum of hpsi.py on any
grid that holds the sphere (reading A8); tests check the two agree to ~1e-13.
It is a second opinion for full-size outputs, not the definition.
"""
from __future__ import annotations

import numpy as np
import scipy.fft


def g2r(psi_g, idx, grid, workers=-1):
    """Backward transform with 1/N (reading A5): box[idx] = psi; ifftn."""
    nb = psi_g.shape[0]
    n = int(np.prod(grid))
    box = np.zeros((nb, n), dtype=np.complex128)
    box[:, idx] = psi_g
    return scipy.fft.ifftn(box.reshape((nb,) + tuple(grid)), axes=(1, 2, 3), workers=workers)


def r2g(box_r, idx, grid, workers=-1):
    """Unnormalised forward FFT then ``take(idx)``."""
    nb = box_r.shape[0]
    f = scipy.fft.fftn(box_r.reshape((nb,) + tuple(grid)), axes=(1, 2, 3), workers=workers)
    return f.reshape(nb, -1)[:, idx]


def apply_h_fft(psi, idx, g2, v_r, grid, beta=None, d_dense=None, workers=-1):
    psi_r = g2r(psi, idx, grid, workers)
    vpsi = r2g(psi_r * np.asarray(v_r).reshape((1,) + tuple(grid)), idx, grid, workers)
    out = 0.5 * np.asarray(g2)[None, :] * psi + vpsi
    if beta is not None and beta.shape[0] > 0:
        p = np.conj(beta) @ psi.T            # [nproj][nb]
        out = out + ((d_dense @ p).T @ beta)
    return out
