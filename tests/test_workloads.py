"""The seeded generators produce what DESIGN.md section 4 says (harness checks, no method arithmetic)."""
import numpy as np

from workloads import CONFIGS, cell_for, make_dmatrix, make_kpoints, make_psi, make_vloc


def test_cells():
    for name, nat in [("cfg1", 2), ("cfg3", 8), ("cfg4", 64), ("cfg5", 216)]:
        lat, pos = cell_for(CONFIGS[name])
        assert pos.shape == (nat, 3) and CONFIGS[name].nproj == 4 * nat
        # nearest-neighbour distance of the diamond structure: a*sqrt(3)/4
        d = np.linalg.norm(pos[1] - pos[0])
        assert abs(d - 10.26 * np.sqrt(3) / 4) < 1e-12


def test_vloc_is_real_bounded_and_band_limited():
    cfg = CONFIGS["cfg1"]
    lat, _ = cell_for(cfg)
    v = make_vloc(cfg, lat)
    assert v.dtype == np.float64 and v.shape == (24 ** 3,)
    assert abs(np.max(np.abs(v)) - 1.0) < 1e-15
    c = np.fft.fftn(v.reshape(cfg.grid))
    b = 2 * np.pi * np.linalg.inv(lat).T
    f = np.fft.fftfreq(24, 1 / 24)
    m = np.stack(np.meshgrid(f, f, f, indexing="ij"), axis=-1)
    g2 = np.sum((m @ b) ** 2, axis=-1)
    assert np.max(np.abs(c[g2 > 4 * cfg.ecutwfc_ry])) < 1e-9 * np.max(np.abs(c))
    np.testing.assert_array_equal(v, make_vloc(cfg, lat))       # seeded => reproducible


def test_psi_is_orthonormal_and_seeded():
    cfg = CONFIGS["cfg1"]
    psi = make_psi(cfg, 0, 537)
    np.testing.assert_allclose(np.conj(psi) @ psi.T, np.eye(8), atol=1e-13)
    np.testing.assert_array_equal(psi, make_psi(cfg, 0, 537))


def test_d_blocks_and_kpoints():
    d = make_dmatrix(CONFIGS["cfg5"])
    assert d.shape == (216, 4, 4)
    for blk in d[:10]:
        np.testing.assert_array_equal(blk, blk.T)
        w = np.linalg.eigvalsh(blk)
        assert w.min() >= 0.1 - 1e-12 and w.max() <= 1.0 + 1e-12
    np.testing.assert_array_equal(make_dmatrix(CONFIGS["cfg1"])[1], np.diag([1.0, .5, .5, .5]))
    k = make_kpoints(CONFIGS["cfg2"])
    assert k.shape == (10, 3) and np.all(k >= -0.5) and np.all(k < 0.5)
    assert np.all(make_kpoints(CONFIGS["cfg5"]) == 0)
