"""Pins for oracle O1 (G-sphere, index map) against what the paper prints and the maths fixes."""
import itertools
import math
import os

import numpy as np
import pytest

from oracle import gsphere as og
from tests.common import G2_TOL_U, UNIT_ROUNDOFF, exact_g2
from workloads import CONFIGS, cell_for, make_kpoints

GOLD = os.path.join(os.path.dirname(__file__), "golden", "bcc_fe_gspace.txt")


def _gold():
    d = {}
    with open(GOLD) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            d[k] = [float(x) for x in v]
    return d


def _bcc():
    g = _gold()
    lat = g["alat"][0] * np.array([g["a1"], g["a2"], g["a3"]])
    return g, lat


def test_reciprocal_axes_match_paper_print():
    g, lat = _bcc()
    b = og.reciprocal_lattice(lat)
    tpiba = 2 * math.pi / g["alat"][0]
    assert abs(tpiba - g["tpiba"][0]) < 5e-6                      # PAPER.md:625 prints 1.23031
    np.testing.assert_allclose(b / tpiba, np.array([g["b1"], g["b2"], g["b3"]]), atol=1e-12)
    np.testing.assert_allclose(lat @ b.T, 2 * math.pi * np.eye(3), atol=1e-12)


def test_bcc_example_counts_and_listing():
    g, lat = _bcc()
    grid = tuple(int(x) for x in g["grid_shape"])
    miller, idx, g2 = og.gsphere(lat, g["ecut_ry"][0], grid)
    assert miller.shape[0] == int(g["size_g"][0])                 # 2243
    assert int(np.prod(grid)) == int(g["size_r"][0])              # 5832
    mg = og.min_grid(miller)
    assert mg == (17, 17, 17) and all(m <= n for m, n in zip(mg, grid))
    # printed head / tail of the listing; C-order => fastest axis is the third
    assert list(miller[:5, 2]) == [int(x) for x in g["comp_head"]]
    assert list(miller[-5:, 2]) == [int(x) for x in g["comp_tail"]]
    assert [f"{x:5.1f}" for x in g2[:5]] == [f"{x:5.1f}" for x in g["g2_head"]]
    assert [f"{x:5.1f}" for x in g2[-5:]] == [f"{x:5.1f}" for x in g["g2_tail"]]


def test_index_map_is_take_index_of_c_order_box():
    g, lat = _bcc()
    grid = (18, 18, 18)
    miller, idx, g2 = og.gsphere(lat, 160.0, grid)
    assert np.all(np.diff(idx) > 0)
    # idx must address the numpy fftfreq position of each Miller triple
    f1 = np.fft.fftfreq(18, 1 / 18).astype(int)
    box = np.stack(np.meshgrid(f1, f1, f1, indexing="ij"), axis=-1).reshape(-1, 3)
    np.testing.assert_array_equal(box[idx], miller)


def test_inversion_symmetry_at_gamma_and_volume_estimate():
    for name in ("cfg1", "cfg3"):
        cfg = CONFIGS[name]
        lat, _ = cell_for(cfg)
        miller, idx, g2 = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid)
        s = {tuple(m) for m in miller}
        assert all((-a, -b, -c) in s for (a, b, c) in s)
        vol = abs(np.linalg.det(lat))
        est = vol * cfg.ecutwfc_ry ** 1.5 / (6 * math.pi ** 2)
        assert abs(miller.shape[0] - est) / est < 0.08


@pytest.mark.parametrize("name,ng", [("cfg1", 537), ("cfg2", 725), ("cfg3", 2945), ("cfg4", 23847)])
def test_sphere_sizes_of_configs(name, ng):
    # sizes enumerated independently in SURVEY.md section 8 table ([computed] there)
    cfg = CONFIGS[name]
    lat, _ = cell_for(cfg)
    miller, idx, g2 = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid)
    assert miller.shape[0] == ng


def test_brute_force_k_point_sphere():
    lat = 0.5 * 10.26 * np.array([[-1.0, 0, 1], [0, 1, 1], [-1, 1, 0]])
    b = og.reciprocal_lattice(lat)
    k = np.array([0.31, -0.17, 0.44])
    ecut = 9.0
    grid = (16, 16, 16)
    miller, idx, g2 = og.gsphere(lat, ecut, grid, k)
    ref = []
    for m in itertools.product(range(-7, 8), repeat=3):
        q = (np.array(m) + k) @ b
        if q @ q <= ecut:
            ref.append(((m[0] % 16) * 16 + (m[1] % 16)) * 16 + (m[2] % 16))
    assert sorted(ref) == list(idx)
    q = (miller + k) @ b
    np.testing.assert_allclose(g2, np.sum(q * q, axis=1), rtol=1e-14)


@pytest.mark.parametrize("name,ik", [("cfg1", 0), ("cfg2", 3), ("cfg3", 0), ("bcc", 0)])
def test_g2_against_exact_rational_evaluation(name, ik):
    """A14: the oracle's |k+G|^2 against an exact evaluation (rational arithmetic, one final rounding), within the
    rounding bound derived from the operation count (tests/common.py G2_TOL_U).  A wrong reciprocal axis, a
    transposed B or a dropped k fails this by many orders of magnitude."""
    if name == "bcc":
        _, lat = _bcc()
        k, ecut, grid = np.zeros(3), 160.0, (18, 18, 18)
    else:
        cfg = CONFIGS[name]
        lat, _ = cell_for(cfg)
        k, ecut, grid = make_kpoints(cfg)[ik], cfg.ecutwfc_ry, cfg.grid
    miller, idx, g2 = og.gsphere(lat, ecut, grid, k)
    ex, scale = exact_g2(lat, k, miller)
    assert np.all(np.abs(g2 - ex) <= G2_TOL_U * UNIT_ROUNDOFF * scale)
    assert np.all(ex <= ecut * (1 + 1e-12))


def test_grid_too_small_is_an_error():
    lat, _ = cell_for(CONFIGS["cfg1"])
    with pytest.raises(ValueError):
        og.gsphere(lat, 25.0, (8, 8, 8))
