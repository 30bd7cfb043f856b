"""Pins of the Taylor-propagator oracle (oracle/propagate.py, eq. 52)."""
import math

import numpy as np

from oracle import gsphere as og
from oracle import hpsi as oh
from oracle import propagate as op
from workloads import CONFIGS, cell_for, make_beta, make_dmatrix, make_psi, make_vloc


def _cfg1():
    cfg = CONFIGS["cfg1"]
    lat, pos = cell_for(cfg)
    miller, idx, g2 = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid, np.zeros(3))
    v = make_vloc(cfg, lat)
    beta = make_beta(cfg, lat, pos, np.zeros(3), miller)
    h = oh.h_matrix(miller, g2, oh.vhat_box(v, cfg.grid), cfg.grid, beta, oh.expand_d(make_dmatrix(cfg)))
    return cfg, idx, h


def test_orders_zero_and_one_are_what_eq52_says():
    cfg, idx, h = _cfg1()
    psi = make_psi(cfg, 0, idx.size)[:3]
    f = lambda x: (h @ x.T).T
    np.testing.assert_array_equal(op.taylor_propagate(psi, f, 0.3, 0), psi)
    np.testing.assert_allclose(op.taylor_propagate(psi, f, 0.3, 1), psi - 0.3j * f(psi), rtol=0, atol=1e-15)


def test_eigenvector_gets_the_truncated_exponential_of_its_eigenvalue():
    cfg, idx, h = _cfg1()
    w, u = np.linalg.eigh(h)
    vec = u[:, 5][None, :].astype(complex)            # H vec = w[5] vec
    dt, k = 0.07, 6
    got = op.taylor_propagate(vec, lambda x: (h @ x.T).T, dt, k)
    poly = sum((-1j * dt * w[5]) ** r / math.factorial(r) for r in range(k + 1))
    np.testing.assert_allclose(got, poly * vec, rtol=0, atol=1e-12)


def test_converges_to_the_exact_exponential_within_the_remainder_bound():
    cfg, idx, h = _cfg1()
    psi = make_psi(cfg, 0, idx.size)[:4]
    w, u = np.linalg.eigh(h)
    dt = 0.02
    exact = ((u * np.exp(-1j * dt * w)) @ (np.conj(u.T) @ psi.T)).T       # exp(-i dt H) psi by eigendecomposition
    x = dt * max(abs(w[0]), abs(w[-1]))                                   # dt * ||H||
    prev = None
    for k in (2, 4, 8):
        got = op.taylor_propagate(psi, lambda y: (h @ y.T).T, dt, k)
        err = np.max(np.linalg.norm(got - exact, axis=1))
        bound = x ** (k + 1) / math.factorial(k + 1) * math.exp(x)        # Lagrange remainder, unit-norm rows
        assert err <= bound + 1e-13, (k, err, bound)
        assert prev is None or err < prev
        prev = err
    # and the norm is conserved to the truncation order (exact propagator is unitary)
    assert np.max(np.abs(np.linalg.norm(got, axis=1) - 1.0)) <= bound + 1e-13
