"""ORACLE (test infrastructure, never on the product path): Taylor-series exponential of the KS Hamiltonian.

    exp(-i dt H) psi  ~=  sum_{r=0}^{k} (-i dt)^r / r!  H^r psi              PAPER.md:1131-1135 (eq. 52), prop_psi()

Followed literally: the powers H^r psi are built by repeated application of the H oracle, each multiplied by its own
coefficient (-i dt)^r / r! and added up in order r = 0..k.  No recurrence on the coefficients, no fusion.
`apply_h` is any callable psi [nb][ng] -> H psi [nb][ng] (the tests pass oracle.hpsi functions).
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
