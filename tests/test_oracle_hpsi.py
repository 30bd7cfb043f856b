"""Pins for oracle O2 (direct-sum H apply).

Each test fixes one term against something that is not the oracle itself:
closed forms, a textbook rank-1 operator, BLAS zgemm, brute-force DFT on 8^3,
Hermiticity, and the paper's FFT route.
"""
import numpy as np
import pytest
import scipy.linalg.blas as blas

from oracle import dft as od
from oracle import gsphere as og
from oracle import hpsi as oh
from oracle import hpsi_fft as of
from workloads import CONFIGS, cell_for, make_beta, make_dmatrix, make_kpoints, make_psi, make_vloc

FCC = 0.5 * 10.26 * np.array([[-1.0, 0, 1], [0, 1, 1], [-1, 1, 0]])


def _small(ecut=6.0, grid=(8, 8, 8), k=(0.0, 0.0, 0.0)):
    miller, idx, g2 = og.gsphere(FCC, ecut, grid, k)
    return miller, idx, g2, grid


def _rand_psi(rng, nb, ng):
    return rng.standard_normal((nb, ng)) + 1j * rng.standard_normal((nb, ng))


def test_plane_wave_is_eigenvector_for_constant_v():
    # V = V0, D = 0  =>  H e_G = (1/2|k+G|^2 + V0) e_G exactly (eq. 12)
    k = (0.2, -0.1, 0.3)
    miller, idx, g2, grid = _small(k=k)
    v0 = -0.37
    vhat = oh.vhat_box(np.full(512, v0), grid)
    ng = idx.size
    psi = np.eye(ng, dtype=np.complex128)
    for out in (oh.apply_h_dense(psi, miller, g2, vhat, grid), oh.apply_h_rows(psi, miller, g2, vhat, grid)):
        np.testing.assert_allclose(out, np.diag(0.5 * g2 + v0), atol=1e-14)


def test_single_complex_fourier_component_shifts_by_plus_g0():
    # V(r) = exp(+i G0.r)  =>  Vhat = delta_{G,G0}  =>  (L psi)(G) = psi(G - G0): fixes sign and operand order
    miller, idx, g2, grid = _small()
    n = np.array(grid)
    g0 = np.array([1, 0, -1])
    j = np.stack(np.meshgrid(*[np.arange(x) for x in grid], indexing="ij"), axis=-1)
    v = np.exp(2j * np.pi * np.sum(j * g0 / n, axis=-1)).reshape(-1)
    vhat = np.fft.fftn(v.reshape(grid)) / 512          # complex V: bypass the real-V helper
    rng = np.random.default_rng(5)
    psi = _rand_psi(rng, 3, idx.size)
    look = {tuple(m): i for i, m in enumerate(miller)}
    want = np.zeros_like(psi)
    for i, m in enumerate(miller):
        src = look.get(tuple(m - g0))
        if src is not None:
            want[:, i] = psi[:, src]
    zero = np.zeros_like(g2)
    np.testing.assert_allclose(oh.apply_h_rows(psi, miller, zero, vhat, grid), want, atol=1e-13)
    np.testing.assert_allclose(oh.apply_h_dense(psi, miller, zero, vhat, grid), want, atol=1e-13)


def test_cosine_potential_couples_g_plus_minus_g0_with_weight_one():
    miller, idx, g2, grid = _small()
    n = np.array(grid)
    g0 = np.array([0, 1, 1])
    j = np.stack(np.meshgrid(*[np.arange(x) for x in grid], indexing="ij"), axis=-1)
    v = 2 * np.cos(2 * np.pi * np.sum(j * g0 / n, axis=-1)).reshape(-1)
    vhat = oh.vhat_box(v, grid)
    rng = np.random.default_rng(6)
    psi = _rand_psi(rng, 2, idx.size)
    look = {tuple(m): i for i, m in enumerate(miller)}
    want = np.zeros_like(psi)
    for i, m in enumerate(miller):
        for s in (+1, -1):
            src = look.get(tuple(m + s * g0))
            if src is not None:
                want[:, i] += psi[:, src]
    got = oh.apply_h_rows(psi, miller, np.zeros_like(g2), vhat, grid)
    np.testing.assert_allclose(got, want, atol=1e-13)


def test_rank_one_projector_is_beta_times_vdot():
    miller, idx, g2, grid = _small()
    rng = np.random.default_rng(7)
    ng = idx.size
    beta = _rand_psi(rng, 1, ng)
    psi = _rand_psi(rng, 4, ng)
    vhat = np.zeros(512, dtype=np.complex128)
    d = np.array([[1.0]])
    got = oh.apply_h_rows(psi, miller, np.zeros(ng), vhat, grid, beta, d)
    want = np.stack([beta[0] * np.vdot(beta[0], psi[n]) for n in range(4)])
    np.testing.assert_allclose(got, want, rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(oh.apply_h_dense(psi, miller, np.zeros(ng), vhat, grid, beta, d), want,
                               rtol=1e-13, atol=1e-13)


def test_nonlocal_term_reduces_to_zgemm():
    cfg = CONFIGS["cfg1"]
    lat, pos = cell_for(cfg)
    miller, idx, g2 = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid)
    beta = make_beta(cfg, lat, pos, np.zeros(3), miller)
    rng = np.random.default_rng(8)
    a = rng.standard_normal((8, 8))
    d = a + a.T                                        # full dense symmetric D
    psi = make_psi(cfg, 0, idx.size)
    vhat = np.zeros(int(np.prod(cfg.grid)), dtype=np.complex128)
    got = oh.apply_h_rows(psi, miller, np.zeros_like(g2), vhat, cfg.grid, beta, d)
    p = blas.zgemm(1.0, np.conj(beta), psi.T)          # [nproj][nb]
    want = blas.zgemm(1.0, (d @ p).T, beta)
    np.testing.assert_allclose(got, want, rtol=1e-12, atol=1e-14)


@pytest.mark.parametrize("kpt", [(0.0, 0.0, 0.0), (0.25, -0.4, 0.1)])
def test_hermiticity_full_h(kpt):
    cfg = CONFIGS["cfg1"]
    lat, pos = cell_for(cfg)
    miller, idx, g2 = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid, kpt)
    vhat = oh.vhat_box(make_vloc(cfg, lat), cfg.grid)
    beta = make_beta(cfg, lat, pos, np.array(kpt), miller)
    rng = np.random.default_rng(9)
    blocks = make_dmatrix(CONFIGS["cfg5"])[:2]
    d = oh.expand_d(blocks)
    psi = _rand_psi(rng, 3, idx.size)
    phi = _rand_psi(rng, 3, idx.size)
    hpsi = oh.apply_h_rows(psi, miller, g2, vhat, cfg.grid, beta, d)
    hphi = oh.apply_h_rows(phi, miller, g2, vhat, cfg.grid, beta, d)
    lhs = np.conj(phi) @ hpsi.T                        # <phi_a|H psi_b>
    rhs = np.conj(np.conj(psi) @ hphi.T).T             # conj <psi_b|H phi_a>
    np.testing.assert_allclose(lhs, rhs, rtol=0, atol=1e-11 * np.max(np.abs(lhs)))
    # linearity
    c = 0.3 - 1.1j
    both = oh.apply_h_rows(psi + c * phi, miller, g2, vhat, cfg.grid, beta, d)
    np.testing.assert_allclose(both, hpsi + c * hphi, atol=1e-12 * np.max(np.abs(both)))


def test_dense_and_loop_spellings_agree_and_rows_subset():
    cfg = CONFIGS["cfg1"]
    lat, pos = cell_for(cfg)
    k = make_kpoints(CONFIGS["cfg2"])[3]
    miller, idx, g2 = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid, k)
    vhat = oh.vhat_box(make_vloc(cfg, lat), cfg.grid)
    beta = make_beta(cfg, lat, pos, k, miller)
    d = oh.expand_d(make_dmatrix(cfg))
    psi = make_psi(cfg, 0, idx.size)
    a = oh.apply_h_dense(psi, miller, g2, vhat, cfg.grid, beta, d)
    b = oh.apply_h_rows(psi, miller, g2, vhat, cfg.grid, beta, d)
    np.testing.assert_allclose(a, b, rtol=0, atol=1e-13 * np.max(np.abs(a)))
    rows = np.array([0, 7, 100, idx.size - 1], dtype=np.int32)
    c = oh.apply_h_rows(psi, miller, g2, vhat, cfg.grid, beta, d, rows=rows)
    np.testing.assert_array_equal(c, b[:, rows])


def test_brute_force_naive_dft_apply_on_8cubed():
    # local term through naive DFTs written from the definition (no library FFT) == direct sum
    miller, idx, g2, grid = _small(ecut=5.0)
    assert all(2 * np.max(np.abs(miller[:, i])) + 1 <= 8 for i in range(3))
    rng = np.random.default_rng(10)
    v = rng.standard_normal(512)
    psi = _rand_psi(rng, 2, idx.size)
    vhat = od.naive_dftn(v.reshape(grid), -1).reshape(-1) / 512
    want = []
    for n in range(2):
        box = np.zeros(512, dtype=np.complex128)
        box[idx] = psi[n]
        pr = od.naive_dftn(box.reshape(grid), +1)                # psi(r) (scale cancels below)
        vp = od.naive_dftn(pr * v.reshape(grid), -1).reshape(-1) / 512
        want.append(vp[idx] + 0.5 * g2 * psi[n])
    got = oh.apply_h_rows(psi, miller, g2, vhat, grid)
    np.testing.assert_allclose(got, np.stack(want), atol=1e-12)


def test_vhat_synthesises_v_at_sampled_points():
    # V(r_j) = sum_G Vhat(G) exp(+i G.r_j), plain loop over the box at a few points
    cfg = CONFIGS["cfg1"]
    lat, _ = cell_for(cfg)
    v = make_vloc(cfg, lat)
    grid = cfg.grid
    vhat = oh.vhat_box(v, grid).reshape(grid)
    f = [np.fft.fftfreq(n, 1 / n) for n in grid]
    rng = np.random.default_rng(11)
    for _ in range(3):
        j = rng.integers(0, 24, size=3)
        ph = np.exp(2j * np.pi * (f[0][:, None, None] * j[0] / 24 + f[1][None, :, None] * j[1] / 24
                                  + f[2][None, None, :] * j[2] / 24))
        val = np.sum(vhat * ph)
        assert abs(val - v.reshape(grid)[tuple(j)]) < 1e-12


@pytest.mark.parametrize("name", ["cfg1", "cfg3"])
def test_fft_route_agrees_with_direct_sum(name):
    cfg = CONFIGS[name]
    lat, pos = cell_for(cfg)
    miller, idx, g2 = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid)
    v = make_vloc(cfg, lat)
    vhat = oh.vhat_box(v, cfg.grid)
    beta = make_beta(cfg, lat, pos, np.zeros(3), miller)
    d = oh.expand_d(make_dmatrix(cfg))
    psi = make_psi(cfg, 0, idx.size, nbands=4)
    a = oh.apply_h_rows(psi, miller, g2, vhat, cfg.grid, beta, d)
    b = of.apply_h_fft(psi, idx, g2, v, cfg.grid, beta, d)
    for n in range(4):
        assert np.max(np.abs(a[n] - b[n])) <= 1e-12 * np.max(np.abs(a[n]))


def test_expand_d_is_the_block_diagonal_embedding():
    """oracle.hpsi.expand_d against scipy.linalg.block_diag (a library routine the oracle does not call): the blocks sit on
    the diagonal in order, everything else is zero (D couples projectors of one atom only)."""
    import scipy.linalg
    from oracle import hpsi as oh
    rng = np.random.default_rng(3)
    for nblk, bs in ((1, 4), (3, 2), (5, 18), (7, 1)):
        b = rng.standard_normal((nblk, bs, bs))
        np.testing.assert_array_equal(oh.expand_d(b), scipy.linalg.block_diag(*b))
