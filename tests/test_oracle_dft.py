"""Pins for oracle O3 (naive DFT) and for the library-FFT steps the oracle side uses."""
import numpy as np

from oracle import dft as od
from oracle import gsphere as og
from oracle import hpsi as oh
from oracle import hpsi_fft as of


def test_naive_dft_matches_pointwise_triple_sum():
    rng = np.random.default_rng(1)
    f = rng.standard_normal((4, 3, 5)) + 1j * rng.standard_normal((4, 3, 5))
    full = od.naive_dftn(f, -1)
    for m in [(0, 0, 0), (1, 2, 3), (3, 1, 4), (2, 0, 1)]:
        assert abs(full[m] - od.naive_dftn_pointwise(f, m, -1)) < 1e-12
    back = od.naive_dftn(f, +1)
    for m in [(1, 1, 1), (3, 2, 0)]:
        assert abs(back[m] - od.naive_dftn_pointwise(f, m, +1)) < 1e-12


def test_library_fft_agrees_with_naive_dft_on_8cubed():
    rng = np.random.default_rng(2)
    f = rng.standard_normal((8, 8, 8)) + 1j * rng.standard_normal((8, 8, 8))
    np.testing.assert_allclose(np.fft.fftn(f), od.naive_dftn(f, -1), atol=1e-11)
    np.testing.assert_allclose(np.fft.ifftn(f) * 512, od.naive_dftn(f, +1), atol=1e-11)
    v = rng.standard_normal(512)
    np.testing.assert_allclose(oh.vhat_box(v, (8, 8, 8)), od.naive_dftn(v.reshape(8, 8, 8), -1) / 512,
                               atol=1e-13)


def test_round_trip_and_parseval_on_the_box():
    rng = np.random.default_rng(3)
    f = rng.standard_normal((8, 8, 8)) + 1j * rng.standard_normal((8, 8, 8))
    F = od.naive_dftn(f, -1)
    np.testing.assert_allclose(od.naive_dftn(F, +1) / 512, f, atol=1e-12)
    # A5: sum_r |f|^2 = (1/N) sum_G |F|^2
    assert abs(np.sum(np.abs(f) ** 2) - np.sum(np.abs(F) ** 2) / 512) < 1e-9


def test_r2g_is_fftn_take_idx_identity():
    # to_g() == fftn(data.reshape(grid_shape)).take(idxgrid)
    lat = 5.107 * np.array([[.5, .5, .5], [-.5, .5, .5], [-.5, -.5, .5]])
    grid = (18, 18, 18)
    miller, idx, g2 = og.gsphere(lat, 160.0, grid)
    rng = np.random.default_rng(4)
    r = rng.random(5832) + 1j * rng.random(5832)
    got = of.r2g(r[None, :], idx, grid)[0]
    np.testing.assert_allclose(got, np.fft.fftn(r.reshape(grid)).take(idx), atol=1e-11)
    # g2r then r2g on the sphere is the identity (sphere -> box -> sphere)
    psi = rng.standard_normal((2, idx.size)) + 1j * rng.standard_normal((2, idx.size))
    np.testing.assert_allclose(of.r2g(of.g2r(psi, idx, grid), idx, grid), psi, atol=1e-12)
