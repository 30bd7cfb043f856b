"""ORACLE (test infrastructure, never on the product path): GW plane-wave matrix elements.

    M_{nn'}(k, q, G) = < n k+q | exp(i (q+G).r) | n' k >                       PAPER.md:1319-1321 (eq. 56)
for the G with |q+G|^2 < E_cut (strict, as printed).  With Bloch states psi_{nk}(r) = exp(i k.r) sum_G c_{nk}(G) exp(i G.r)
(eq. 9 sign, reading A5) the plane-wave factors exp(-i(k+q).r) exp(i(q+G).r) exp(i k.r) = exp(i G.r) leave
    M_{nn'}(G) = sum_{G''} conj(c_{n,k+q}(G'' + G)) c_{n'k}(G'')                (the "convolution in k-space" of the text)
summed over the sphere of k, with c_{n,k+q} zero outside the sphere of k+q.  No cell-volume factor (reading A10).
Reading A21: eq. 56 is the definition; eq. 57's "FFT^-1( phi* phi' ), phi = FFT(psi)" names the directions
the other way round from eq. 9 and is taken to mean "synthesise both states on the grid, multiply, analyse with
exp(+i G.r) / N".  On the FFT box the lookup G'' + G is taken modulo the grid (reading A8), which is what any grid-based
evaluation computes; on a grid with n_i >= 2 m_wfn + m_eps + 1 nothing wraps and the two coincide (pinned).

Explicit sums, long-double accumulation.  Pins: tests/test_oracle_mtxel.py.
"""
from __future__ import annotations

import numpy as np


def _flat(m, grid):
    n1, n2, n3 = (int(x) for x in grid)
    return ((m[:, 0] % n1) * n2 + (m[:, 1] % n2)) * n3 + (m[:, 2] % n3)


def matrix_elements(bra, miller_bra, ket, miller_ket, miller_eps, grid, wrap: bool = True) -> np.ndarray:
    """bra [nbra][ng(k+q)], ket [nket][ng(k)] -> M [nbra][nket][len(miller_eps)].

    wrap=True: G'' + G looked up modulo the box (reading A8); wrap=False: by Miller triple, zero if absent."""
    bra = np.asarray(bra, dtype=np.complex128)
    ket = np.asarray(ket, dtype=np.complex128)
    mb = np.asarray(miller_bra, dtype=np.int64)
    mk = np.asarray(miller_ket, dtype=np.int64)
    me = np.asarray(miller_eps, dtype=np.int64)
    nbox = int(np.prod(grid))
    out = np.empty((bra.shape[0], ket.shape[0], me.shape[0]), dtype=np.complex128)
    ketl = ket.astype(np.clongdouble)
    if wrap:
        where = np.full(nbox, -1, dtype=np.int64)
        where[_flat(mb, grid)] = np.arange(mb.shape[0])
    else:
        table = {tuple(t): i for i, t in enumerate(mb.tolist())}
    for ig, g in enumerate(me):
        tgt = mk + g[None, :]                                      # G'' + G for every G'' of the ket sphere
        if wrap:
            pos = where[_flat(tgt, grid)]
        else:
            pos = np.array([table.get(tuple(t), -1) for t in tgt.tolist()], dtype=np.int64)
        ok = pos >= 0
        a = np.conj(bra[:, pos[ok]]).astype(np.clongdouble)        # conj(c_{n,k+q}(G''+G))
        b = ketl[:, ok]
        out[:, :, ig] = (a[:, None, :] * b[None, :, :]).sum(axis=2).astype(np.complex128)
    return out


def matrix_elements_fft(bra, idx_bra, ket, idx_ket, idx_eps, grid) -> np.ndarray:
    """Second opinion with library FFTs (the route eq. 57 describes): synthesise, multiply, analyse with exp(+iG.r)/N."""
    nbox = int(np.prod(grid))

    def synth(c, idx):
        box = np.zeros((c.shape[0], nbox), dtype=np.complex128)
        box[:, idx] = c
        return np.fft.ifftn(box.reshape((-1,) + tuple(grid)), axes=(1, 2, 3)) * nbox      # sum_G c(G) exp(+iG.r)

    pb, pk = synth(np.asarray(bra), idx_bra), synth(np.asarray(ket), idx_ket)
    out = np.empty((pb.shape[0], pk.shape[0], len(idx_eps)), dtype=np.complex128)
    for i in range(pb.shape[0]):
        prod = np.conj(pb[i])[None] * pk
        out[i] = np.fft.ifftn(prod, axes=(1, 2, 3)).reshape(pk.shape[0], -1)[:, idx_eps]  # (1/N) sum_r f(r) exp(+iG.r)
    return out
