"""GPU parity of the density accumulation against oracle/density.py (-m gpu).

Tolerance 1e-11 relative to max n(r) (north_star's tolerance on the natural scale; sums of non-negative terms).
"""
import numpy as np
import pytest

from tests.common import TOL, problem
from oracle import density as od

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def qm():
    import __graft_entry__ as ge
    ge.build()
    import paper_2308_07277_b200 as q
    return q


def _density(qm, p, psi, occ, batches, weight=1.0, scale=1.0, k_all=False):
    import torch
    dev = torch.device("cuda:0")
    gs = qm.GSpace(p["lat"], p["cfg"].ecutwfc_ry, p["cfg"].grid, p["k"][None, :])
    gs.density_reset()
    b0 = 0
    for nb in batches:
        gs.density_accumulate(torch.from_numpy(np.ascontiguousarray(psi[b0:b0 + nb])).to(dev),
                              torch.from_numpy(np.ascontiguousarray(occ[b0:b0 + nb])).to(dev), weight=weight)
        b0 += nb
    rho = gs.density_get(scale=scale)
    torch.cuda.synchronize()
    out = rho.cpu().numpy()
    gs.close()
    return out


def test_density_all_points_cfg1(qm):
    p = problem("cfg1")
    occ = np.array([2.0, 2.0, 2.0, 2.0, 1.0, 0.5, 0.0, 0.25])
    got = _density(qm, p, p["psi"], occ, [3, 5], weight=0.5, scale=0.1)     # two band batches accumulate
    ref = od.density(p["psi"], p["miller"], 0.5 * occ, p["cfg"].grid, scale=0.1)
    assert np.max(np.abs(got - ref)) <= TOL * np.max(ref)


def test_density_k_point_cfg2(qm):
    p = problem("cfg2", 3)                       # a seeded random k: |psi|^2 does not see the Bloch phase
    occ = np.linspace(2.0, 0.1, p["psi"].shape[0])
    rng = np.random.default_rng(3)
    pts = rng.integers(0, p["cfg"].grid[0], size=(300, 3))
    got = _density(qm, p, p["psi"], occ, [16]).reshape(p["cfg"].grid)
    ref = od.density(p["psi"], p["miller"], occ, p["cfg"].grid, points=pts)
    assert np.max(np.abs(got[pts[:, 0], pts[:, 1], pts[:, 2]] - ref)) <= TOL * np.max(ref)


@pytest.mark.parametrize("name,nb,batches", [("cfg3", 64, [64]), ("cfg4", 32, [32]), ("cfg5", 32, [16, 16])])
def test_density_sampled_points_and_parseval(qm, name, nb, batches):
    p = problem(name, 0, nbands=nb, orthonormalise=False)
    grid = p["cfg"].grid
    occ = np.random.default_rng(1).uniform(0.0, 2.0, size=nb)
    got = _density(qm, p, p["psi"], occ, batches).reshape(grid)
    rng = np.random.default_rng(2)
    pts = np.concatenate([[[0, 0, 0], [grid[0] - 1, grid[1] - 1, grid[2] - 1]], rng.integers(0, grid[0], size=(48, 3))])
    ref = od.density(p["psi"], p["miller"], occ, grid, points=pts)
    assert np.max(np.abs(got[pts[:, 0], pts[:, 1], pts[:, 2]] - ref)) <= TOL * np.max(ref)
    # properties at full size: non-negative, and sum_r n = N * sum_i f_i ||psi_i||^2 (Parseval; the grid holds the sphere)
    assert got.min() >= 0.0
    want = np.prod(grid) * np.sum(occ * np.sum(np.abs(p["psi"]) ** 2, axis=1))
    assert abs(got.sum() - want) <= 1e-11 * want


def test_density_is_bitwise_reproducible_and_needs_reset(qm):
    import torch
    dev = torch.device("cuda:0")
    p = problem("cfg3")
    occ = np.ones(p["psi"].shape[0])
    a = _density(qm, p, p["psi"], occ, [64])
    b = _density(qm, p, p["psi"], occ, [64])
    assert np.array_equal(a, b)
    gs = qm.GSpace(p["lat"], p["cfg"].ecutwfc_ry, p["cfg"].grid, p["k"][None, :])
    with pytest.raises(qm.QmError):
        gs.density_accumulate(torch.from_numpy(p["psi"]).to(dev), torch.from_numpy(occ).to(dev))
    gs.close()
