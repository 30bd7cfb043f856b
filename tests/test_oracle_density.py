"""Pins of the density oracle (oracle/density.py): closed forms, Parseval, the library FFT as a second opinion."""
import numpy as np

from oracle import density as od
from oracle import gsphere as og
from workloads import CONFIGS, cell_for, make_psi

GRID = (8, 8, 8)
LAT = 6.0 * np.eye(3)


def _sphere():
    return og.gsphere(LAT, 6.0, GRID, np.zeros(3))


def test_single_plane_wave_gives_constant_density():
    miller, idx, g2 = _sphere()
    psi = np.zeros((1, idx.size), dtype=complex)
    psi[0, 7] = 0.6 - 0.8j * 2
    n = od.density(psi, miller, [1.5], GRID)
    np.testing.assert_allclose(n, 1.5 * abs(psi[0, 7]) ** 2, rtol=1e-14)


def test_two_plane_waves_closed_form_fixes_sign_and_axes():
    # n(r) = |c1|^2 + |c2|^2 + 2 Re(conj(c1) c2 exp(i (G2-G1).r)),  (G2-G1).r_j = 2 pi sum_a dm_a j_a / n_a
    miller, idx, g2 = _sphere()
    i1, i2 = 3, 20
    c1, c2 = 0.7 + 0.2j, -0.4 + 0.9j
    psi = np.zeros((1, idx.size), dtype=complex)
    psi[0, i1], psi[0, i2] = c1, c2
    dm = miller[i2] - miller[i1]
    assert np.count_nonzero(dm) >= 2            # a shift that distinguishes the axes
    n = od.density(psi, miller, [1.0], GRID).reshape(GRID)
    j = np.stack(np.meshgrid(*[np.arange(g) for g in GRID], indexing="ij"), axis=-1)
    phase = 2 * np.pi * (j * dm / np.array(GRID)).sum(axis=-1)
    want = abs(c1) ** 2 + abs(c2) ** 2 + 2 * np.real(np.conj(c1) * c2 * np.exp(1j * phase))
    np.testing.assert_allclose(n, want, atol=1e-13)


def test_parseval_sum_and_nonnegativity_and_linearity_in_occupations():
    miller, idx, g2 = _sphere()
    rng = np.random.default_rng(4)
    psi = rng.standard_normal((3, idx.size)) + 1j * rng.standard_normal((3, idx.size))
    occ = np.array([2.0, 1.0, 0.25])
    n = od.density(psi, miller, occ, GRID)
    assert np.all(n >= 0)
    # sum_r |psi(r)|^2 = N * sum_G |psi(G)|^2 for the unnormalised synthesis on a grid that holds the sphere
    want = np.prod(GRID) * np.sum(occ * np.sum(np.abs(psi) ** 2, axis=1))
    assert abs(n.sum() - want) <= 1e-12 * want
    n2 = od.density(psi, miller, 3 * occ, GRID, scale=0.5)
    np.testing.assert_allclose(n2, 1.5 * n, rtol=1e-14)


def test_agrees_with_library_inverse_fft_on_the_box():
    cfg = CONFIGS["cfg1"]
    lat, _ = cell_for(cfg)
    miller, idx, g2 = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid, np.zeros(3))
    psi = make_psi(cfg, 0, idx.size)[:2]
    rng = np.random.default_rng(5)
    pts = rng.integers(0, cfg.grid[0], size=(40, 3))
    got = od.psi_at_points(psi, miller, cfg.grid, pts)
    box = np.zeros((2, int(np.prod(cfg.grid))), dtype=complex)
    box[:, idx] = psi                                        # scatter by the index map
    ref = np.fft.ifftn(box.reshape(2, *cfg.grid), axes=(1, 2, 3)) * np.prod(cfg.grid)
    want = ref[:, pts[:, 0], pts[:, 1], pts[:, 2]]
    np.testing.assert_allclose(got, want, atol=1e-12 * np.max(np.abs(want)))
