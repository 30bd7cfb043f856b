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


# ---- split-operator exponential, PAPER.md:1137-1139 (eq. 53) ------------------------------------------------------
def _cfg1_local():
    cfg = CONFIGS["cfg1"]
    lat, pos = cell_for(cfg)
    miller, idx, g2 = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid, np.zeros(3))
    return cfg, lat, miller, idx, g2, make_vloc(cfg, lat)


def test_ehat_is_the_dft_of_the_phase_field_on_8cubed():
    from oracle import dft as od
    rng = np.random.default_rng(3)
    v = rng.standard_normal(512)
    want = od.naive_dftn(np.exp(-0.37j * v).reshape(8, 8, 8), -1) / 512
    np.testing.assert_allclose(op.ehat_box(v, (8, 8, 8), 0.37), want, atol=1e-13)


def test_split_operator_constant_potential_is_a_pure_phase():
    cfg, lat, miller, idx, g2, v = _cfg1_local()
    psi = make_psi(cfg, 0, idx.size)[:3]
    dt, v0 = 0.21, 0.7
    got = op.split_operator_propagate(psi, miller, g2, np.full_like(v, v0), cfg.grid, dt)
    want = np.exp(-1j * dt * (0.5 * g2 + v0))[None, :] * psi         # T and a constant V commute: exact exponential
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-13)
    np.testing.assert_allclose(op.split_operator_propagate(psi, miller, g2, v, cfg.grid, 0.0), psi, rtol=0, atol=1e-14)


def test_split_operator_single_cosine_gives_bessel_sidebands():
    """V = eps cos(G0.r): exp(-i dt V) = sum_n (-i)^n J_n(dt eps) exp(i n G0.r) (Jacobi-Anger), so a plane wave e_G
    goes to G + n G0 with weight (-i)^n J_n times the two kinetic half-phases: fixes the sign of i, the direction of
    the shift and the order of the three factors."""
    from scipy.special import jv
    cfg, lat, miller, idx, g2, _ = _cfg1_local()
    n1, n2, n3 = cfg.grid
    g0 = np.array([1, 0, -1])
    j = np.stack(np.meshgrid(np.arange(n1), np.arange(n2), np.arange(n3), indexing="ij"), axis=-1)
    eps, dt = 0.9, 0.6
    v = eps * np.cos(2 * np.pi * (j[..., 0] * g0[0] / n1 + j[..., 1] * g0[1] / n2 + j[..., 2] * g0[2] / n3))
    src = 17
    psi = np.zeros((1, idx.size), dtype=complex)
    psi[0, src] = 1.0
    got = op.split_operator_propagate(psi, miller, g2, v.reshape(-1), cfg.grid, dt)[0]
    where = {tuple(m): i for i, m in enumerate(miller.tolist())}
    want = np.zeros(idx.size, dtype=complex)
    for n in range(-12, 13):
        t = tuple((miller[src] + n * g0).tolist())
        if t in where:
            want[where[t]] = ((-1j) ** abs(n)) * jv(abs(n), dt * eps) * np.exp(-0.25j * dt * (g2[src] + g2[where[t]]))
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-13)


def test_split_operator_matches_library_fft_route_and_never_gains_norm():
    from oracle import hpsi_fft as of
    cfg, lat, miller, idx, g2, v = _cfg1_local()
    psi = make_psi(cfg, 0, idx.size)[:4]
    dt = 0.13
    got = op.split_operator_propagate(psi, miller, g2, v, cfg.grid, dt)
    half = np.exp(-0.25j * dt * g2)
    box = of.g2r(psi * half, idx, cfg.grid) * np.exp(-1j * dt * v).reshape((1,) + cfg.grid)
    want = of.r2g(box, idx, cfg.grid) * half
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-13)
    assert np.all(np.linalg.norm(got, axis=1) <= 1.0 + 1e-13)         # phases are unitary, the sphere projects


def test_split_operator_approaches_the_exact_exponential_at_second_order():
    cfg, lat, miller, idx, g2, v = _cfg1_local()
    h = oh.h_matrix(miller, g2, oh.vhat_box(v, cfg.grid), cfg.grid)    # T + V_loc, no projectors (reading A22)
    w, u = np.linalg.eigh(h)
    psi = make_psi(cfg, 0, idx.size)[:2]
    errs = []
    for dt in (0.04, 0.02, 0.01):
        exact = ((u * np.exp(-1j * dt * w)) @ (np.conj(u.T) @ psi.T)).T
        got = op.split_operator_propagate(psi, miller, g2, v, cfg.grid, dt)
        errs.append(np.max(np.linalg.norm(got - exact, axis=1)))
    assert errs[0] < 5e-3
    for a, b in zip(errs[:-1], errs[1:]):                              # local error O(dt^2) (sphere projection) .. O(dt^3)
        assert 3.0 <= a / b <= 9.0, errs
