"""Pins of the GW plane-wave matrix-element oracle (oracle/mtxel.py, eqs. 56-57)."""
import numpy as np

from oracle import dft as od
from oracle import gsphere as og
from oracle import mtxel as om
from workloads import CONFIGS, cell_for, make_kpoints, make_psi


def _spheres(name="cfg2", ik_bra=1, ik_ket=0, ecut_eps=8.0, grid=None):
    cfg = CONFIGS[name]
    lat, _ = cell_for(cfg)
    grid = cfg.grid if grid is None else grid
    kpts = make_kpoints(cfg)
    kb, kk = kpts[ik_bra], kpts[ik_ket]
    mb, ib, _ = og.gsphere(lat, cfg.ecutwfc_ry, grid, kb)
    mk, ikx, _ = og.gsphere(lat, cfg.ecutwfc_ry, grid, kk)
    me, ie, g2e = og.gsphere(lat, ecut_eps, grid, kb - kk, strict=True)      # |q+G|^2 < E_cut, q = (k+q) - k
    return cfg, lat, grid, (mb, ib), (mk, ikx), (me, ie, g2e)


def test_eps_sphere_uses_the_strict_inequality_of_eq56():
    lat = 2 * np.pi * np.eye(3)                       # b = identity: |G|^2 = m.m exactly
    m_le, _, _ = og.gsphere(lat, 4.0, (8, 8, 8))
    m_lt, _, g2 = og.gsphere(lat, 4.0, (8, 8, 8), strict=True)
    assert (2, 0, 0) in {tuple(t) for t in m_le.tolist()}
    assert (2, 0, 0) not in {tuple(t) for t in m_lt.tolist()}
    assert m_le.shape[0] - m_lt.shape[0] == 6 and np.all(g2 < 4.0)


def test_single_plane_waves_give_a_kronecker_delta_at_g1_minus_g2():
    """bra = i e_{G1}, ket = e_{G2}:  M(G) = conj(i) delta(G, G1 - G2): fixes which factor is conjugated and the sign
    of G in exp(+i(q+G).r)."""
    cfg, lat, grid, (mb, ib), (mk, ik), (me, ie, _) = _spheres()
    where_e = {tuple(t): i for i, t in enumerate(me.tolist())}
    hits = 0
    near = [(sb, int(np.argmin(np.sum((mk - mb[sb]) ** 2, axis=1)))) for sb in (5, 40, 300)]    # G1 - G2 small: inside
    for sb, sk in near + [(100, 120), (0, mk.shape[0] - 1)]:
        bra = np.zeros((1, mb.shape[0]), dtype=complex)
        ket = np.zeros((1, mk.shape[0]), dtype=complex)
        bra[0, sb], ket[0, sk] = 1j, 1.0
        m = om.matrix_elements(bra, mb, ket, mk, me, grid)[0, 0]
        want = np.zeros(me.shape[0], dtype=complex)
        d = tuple((mb[sb] - mk[sk]).tolist())
        if d in where_e:
            want[where_e[d]] = -1j
            hits += 1
        np.testing.assert_allclose(m, want, rtol=0, atol=1e-15)
    assert hits >= 2


def test_q_zero_symmetries_and_norms():
    cfg, lat, grid, (mb, ib), (mk, ik), (me, ie, _) = _spheres(ik_bra=0, ik_ket=0, ecut_eps=10.0)
    psi = make_psi(cfg, 0, mk.shape[0])[:5]
    m = om.matrix_elements(psi, mb, psi, mk, me, grid)
    where_e = {tuple(t): i for i, t in enumerate(me.tolist())}
    g0 = where_e[(0, 0, 0)]
    np.testing.assert_allclose(m[:, :, g0], np.eye(5), rtol=0, atol=1e-14)              # M_nn'(0) = <n|n'>
    minus = np.array([where_e[tuple((-t).tolist())] for t in me])
    np.testing.assert_allclose(np.conj(m), np.transpose(m, (1, 0, 2))[:, :, minus], rtol=0, atol=1e-14)
    # |M| <= ||bra|| ||ket|| (Cauchy-Schwarz on every G)
    assert np.max(np.abs(m)) <= 1.0 + 1e-13


def test_brute_force_naive_dft_on_8cubed():
    """Definition on the grid: M(G) = (1/N) sum_r conj(phi_bra(r)) phi_ket(r) exp(+iG.r), phi(r) = sum_G c(G) exp(+iG.r),
    every transform by the naive DFT."""
    lat = 6.0 * np.eye(3)
    grid = (8, 8, 8)
    kb, kk = np.array([0.25, 0.0, -0.125]), np.array([0.0, 0.125, 0.0])
    mb, ib, _ = og.gsphere(lat, 3.5, grid, kb)
    mk, ik, _ = og.gsphere(lat, 3.5, grid, kk)
    me, ie, _ = og.gsphere(lat, 3.0, grid, kb - kk, strict=True)
    rng = np.random.default_rng(8)
    bra = rng.standard_normal((2, ib.size)) + 1j * rng.standard_normal((2, ib.size))
    ket = rng.standard_normal((3, ik.size)) + 1j * rng.standard_normal((3, ik.size))
    got = om.matrix_elements(bra, mb, ket, mk, me, grid)

    def synth(c, idx):
        box = np.zeros(512, dtype=complex)
        box[idx] = c
        return od.naive_dftn(box.reshape(grid), +1)

    for i in range(2):
        for j in range(3):
            f = np.conj(synth(bra[i], ib)) * synth(ket[j], ik)
            want = (od.naive_dftn(f, +1) / 512).reshape(-1)[ie]
            np.testing.assert_allclose(got[i, j], want, rtol=0, atol=1e-12)


def test_wrap_and_no_wrap_agree_on_a_large_enough_grid_and_fft_route_agrees():
    cfg, lat, grid, (mb, ib), (mk, ik), (me, ie, _) = _spheres()
    assert all(n >= 2 * max(np.abs(mb).max(), np.abs(mk).max()) + np.abs(me).max() + 1 for n in grid)
    rng = np.random.default_rng(4)
    bra = rng.standard_normal((3, ib.size)) + 1j * rng.standard_normal((3, ib.size))
    ket = rng.standard_normal((2, ik.size)) + 1j * rng.standard_normal((2, ik.size))
    a = om.matrix_elements(bra, mb, ket, mk, me, grid, wrap=True)
    b = om.matrix_elements(bra, mb, ket, mk, me, grid, wrap=False)
    np.testing.assert_allclose(a, b, rtol=0, atol=1e-13)
    c = om.matrix_elements_fft(bra, ib, ket, ik, ie, grid)
    np.testing.assert_allclose(a, c, rtol=0, atol=1e-11)
    # on a grid that is too small the lookups wrap: the two readings differ, the grid route follows `wrap`
    lat, small = 10.26 * np.eye(3), (11, 11, 11)
    kb, kk = np.array([0.3, 0.0, -0.2]), np.zeros(3)
    mb, ib, _ = og.gsphere(lat, 12.0, small, kb)
    mk, ik, _ = og.gsphere(lat, 12.0, small, kk)
    me, ie, _ = og.gsphere(lat, 6.0, small, kb - kk, strict=True)
    assert small[0] < 2 * max(np.abs(mb).max(), np.abs(mk).max()) + np.abs(me).max() + 1
    bra = rng.standard_normal((2, ib.size)) + 1j * rng.standard_normal((2, ib.size))
    ket = rng.standard_normal((2, ik.size)) + 1j * rng.standard_normal((2, ik.size))
    a = om.matrix_elements(bra, mb, ket, mk, me, small, wrap=True)
    b = om.matrix_elements(bra, mb, ket, mk, me, small, wrap=False)
    assert np.max(np.abs(a - b)) > 1e-3
    np.testing.assert_allclose(a, om.matrix_elements_fft(bra, ib, ket, ik, ie, small), rtol=0, atol=1e-11)
