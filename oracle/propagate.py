"""ORACLE (test infrastructure, never on the product path): Taylor-series exponential of the KS Hamiltonian.

    exp(-i dt H) psi  ~=  sum_{r=0}^{k} (-i dt)^r / r!  H^r psi              PAPER.md:1131-1135 (eq. 52), prop_psi()

Followed literally: the powers H^r psi are built by repeated application of the H oracle, each multiplied by its own
coefficient (-i dt)^r / r! and added up in order r = 0..k.  No recurrence on the coefficients, no fusion.
`apply_h` is any callable psi [nb][ng] -> H psi [nb][ng] (the tests pass oracle.hpsi functions).

Split-operator exponential                                                  PAPER.md:1137-1139 (eq. 53)
    exp(-i dt H) ~= exp(-i dt T/2) exp(-i dt V) exp(-i dt T/2)
followed factor by factor, right to left.  T is diagonal in G (T(G) = 1/2 |k+G|^2, eq. 12 / eqs. 49-51), so its
exponential is the phase exp(-i dt |k+G|^2 / 4).  Reading A22: V is the LOCAL potential, a multiplication
by V(r_j) on the FFT grid, so exp(-i dt V) is the multiplication by E(r_j) = exp(-i dt V(r_j)) on that grid; back on the
sphere that is the convolution  sum_{G'} Ehat(G - G') psi(G')  with Ehat = (1/N) DFT of E (looked up modulo the box,
reading A8) -- written here as that plain O(N_G^2) sum, no FFT of a wavefunction.  The paper does not say what V
contains when projectors are present; they are not part of this propagator (use the Taylor form).
Pins: tests/test_oracle_propagate.py.
"""
from __future__ import annotations

import math

import numpy as np


def taylor_propagate(psi: np.ndarray, apply_h, dt: float, order: int) -> np.ndarray:
    psi = np.asarray(psi, dtype=np.complex128)
    out = np.zeros_like(psi)
    power = psi.copy()                                   # H^0 psi
    for r in range(order + 1):
        if r > 0:
            power = np.asarray(apply_h(power), dtype=np.complex128)      # H^r psi
        out = out + ((-1j * dt) ** r / math.factorial(r)) * power
    return out


def ehat_box(v_r: np.ndarray, grid, dt: float) -> np.ndarray:
    """Ehat on the whole box: (1/N) * forward DFT of E(r) = exp(-i dt V(r)) (library FFT as one step, the same step
    as hpsi.vhat_box, pinned against the naive DFT in tests/test_oracle_propagate.py)."""
    n = int(np.prod(grid))
    e = np.exp(-1j * dt * np.asarray(v_r, dtype=np.float64).reshape(grid))
    return np.fft.fftn(e) / n


def split_operator_propagate(psi: np.ndarray, miller: np.ndarray, g2: np.ndarray, v_r: np.ndarray, grid, dt: float,
                             rows=None) -> np.ndarray:
    """psi [nb][ng] -> exp(-i dt T/2) exp(-i dt V) exp(-i dt T/2) psi, eq. 53, on `rows` (default: all)."""
    from . import hpsi as oh
    psi = np.asarray(psi, dtype=np.complex128)
    g2 = np.asarray(g2, dtype=np.float64)
    half = np.exp(-1j * dt * (0.5 * g2) / 2.0)                      # exp(-i (dt/2) T(G)), T(G) = 1/2 |k+G|^2
    step1 = psi * half[None, :]                                     # rightmost factor first
    # middle factor: the convolution with Ehat by the explicit loops of hpsi_direct.c (its (L) term with a complex
    # "potential"; T switched off by g2 = 0, no projectors)
    step2 = oh.apply_h_rows(step1, miller, np.zeros_like(g2), ehat_box(v_r, grid, dt), grid, rows=rows)
    sel = slice(None) if rows is None else np.asarray(rows)
    return step2 * half[None, sel]
