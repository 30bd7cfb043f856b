"""O2: H|psi> by direct G-space summation (oracle; test infrastructure).

  H_{G,G'}(k) = 1/2 |k+G|^2 delta_{GG'} + Vhat(G-G')            PAPER.md:146 (eq. 12)
              + sum_ij beta_i(G) D_ij conj(beta_j(G'))           PAPER.md:153-161 (eq. 14; A10)
  Vhat(G) = (1/N) sum_r V(r) exp(-i G.r)                         PAPER.md:650 (matrix element of V)

Two spellings of the same definition:
  * ``h_matrix`` / ``apply_h_dense``: builds the dense N_G x N_G matrix with
    numpy and multiplies (small N_G only);
  * ``apply_h_rows``: the explicit triple loop of ``hpsi_direct.c`` (long-double
    accumulation), for any N_G, optionally on a subset of output rows.
"""
from __future__ import annotations

import ctypes
import numpy as np

from . import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(_build.build())
        lib.oracle_hpsi_rows.restype = ctypes.c_int
        lib.oracle_hpsi_rows.argtypes = [
            ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
        _lib = lib
    return _lib


def vhat_box(v_r: np.ndarray, grid) -> np.ndarray:
    """Vhat on the whole box: (1/N) * forward DFT of V(r) (library FFT as one step;
    pinned against the naive DFT in tests/test_oracle_dft.py)."""
    n = int(np.prod(grid))
    return np.fft.fftn(np.asarray(v_r, dtype=np.float64).reshape(grid)) / n


def expand_d(d_blocks: np.ndarray) -> np.ndarray:
    """Per-atom blocks [nat][b][b] -> dense block-diagonal [nproj][nproj]."""
    nat, b, _ = d_blocks.shape
    d = np.zeros((nat * b, nat * b))
    for a in range(nat):
        d[a * b:(a + 1) * b, a * b:(a + 1) * b] = d_blocks[a]
    return d


def h_matrix(miller, g2, vhat, grid, beta=None, d_dense=None) -> np.ndarray:
    """Dense H (eq. 12 plus the projector term).  O(N_G^2) memory: small spheres only."""
    m = np.asarray(miller, dtype=np.int64)
    n = np.asarray(grid, dtype=np.int64)
    diff = (m[:, None, :] - m[None, :, :]) % n[None, None, :]
    h = vhat.reshape(tuple(grid))[diff[..., 0], diff[..., 1], diff[..., 2]].astype(np.complex128)
    h[np.diag_indices_from(h)] += 0.5 * np.asarray(g2)
    if beta is not None and beta.shape[0] > 0:
        h += beta.T @ (d_dense.astype(np.complex128) @ np.conj(beta))
    return h


def apply_h_dense(psi, miller, g2, vhat, grid, beta=None, d_dense=None) -> np.ndarray:
    """psi [nb][ng] -> (H psi) [nb][ng] through the dense matrix."""
    h = h_matrix(miller, g2, vhat, grid, beta, d_dense)
    return np.ascontiguousarray((h @ psi.T).T)


def apply_h_rows(psi, miller, g2, vhat, grid, beta=None, d_dense=None, rows=None) -> np.ndarray:
    """psi [nb][ng] -> out [nb][len(rows)] by the explicit loops in hpsi_direct.c."""
    lib = _load()
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    nb, ng = psi.shape
    miller = np.ascontiguousarray(miller, dtype=np.int32)
    g2 = np.ascontiguousarray(g2, dtype=np.float64)
    vhat = np.ascontiguousarray(vhat, dtype=np.complex128).reshape(-1)
    gridc = np.ascontiguousarray(grid, dtype=np.int32)
    if rows is None:
        rows = np.arange(ng, dtype=np.int32)
    rows = np.ascontiguousarray(rows, dtype=np.int32)
    if beta is None or beta.shape[0] == 0:
        nproj, bptr, dptr = 0, None, None
    else:
        beta = np.ascontiguousarray(beta, dtype=np.complex128)
        d_dense = np.ascontiguousarray(d_dense, dtype=np.float64)
        nproj = beta.shape[0]
        assert beta.shape == (nproj, ng) and d_dense.shape == (nproj, nproj)
        bptr, dptr = beta.ctypes.data, d_dense.ctypes.data
    out = np.empty((nb, rows.shape[0]), dtype=np.complex128)
    rc = lib.oracle_hpsi_rows(ng, nb, miller.ctypes.data, g2.ctypes.data, psi.ctypes.data,
                              gridc.ctypes.data, vhat.ctypes.data, nproj, bptr, dptr,
                              rows.shape[0], rows.ctypes.data, out.ctypes.data)
    assert rc == 0
    return out
