"""GPU parity of qm_subspace (S = <a_i|b_j>) against oracle/subspace.py (-m gpu).

Tolerance: |dS_ij| <= 1e-11 * ||a_i|| ||b_j|| (the north_star's 1e-11 relative to the natural scale of an inner
product; DESIGN.md section 3 A13 carried over).  Sizes span several 64 x 64 tiles, ragged tile edges, a ragged K tail,
and the full-size cfg5 sphere on sampled entries.
"""
import numpy as np
import pytest

from tests.common import TOL, problem
from oracle import subspace as osub

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def qm():
    import __graft_entry__ as ge
    ge.build()
    import paper_2308_07277_b200 as q
    return q


def _run(qm, p, a, b):
    import torch
    dev = torch.device("cuda:0")
    gs = qm.GSpace(p["lat"], p["cfg"].ecutwfc_ry, p["cfg"].grid, p["k"][None, :])
    s = gs.subspace(torch.from_numpy(a).to(dev), torch.from_numpy(b).to(dev))
    torch.cuda.synchronize()
    out = s.cpu().numpy()
    gs.close()
    return out


def _rand(rng, n, ng):
    return rng.standard_normal((n, ng)) + 1j * rng.standard_normal((n, ng))


@pytest.mark.parametrize("name,na,nb", [("cfg1", 8, 8), ("cfg1", 1, 3), ("cfg3", 64, 64), ("cfg3", 70, 130),
                                        ("cfg2", 16, 16)])
def test_subspace_all_elements(qm, name, na, nb):
    p = problem(name)
    ng = p["idx"].size                      # 537 / 725..752 / 2945: none a multiple of the 16-wide K slice
    rng = np.random.default_rng(na * 1000 + nb)
    a, b = _rand(rng, na, ng), _rand(rng, nb, ng)
    got = _run(qm, p, a, b)
    ref = osub.vdot_matrix(a, b)
    scale = np.linalg.norm(a, axis=1)[:, None] * np.linalg.norm(b, axis=1)[None, :]
    assert np.max(np.abs(got - ref) / scale) <= TOL


def test_subspace_overlap_of_orthonormal_block_and_hermitian_h(qm):
    import torch
    dev = torch.device("cuda:0")
    p = problem("cfg3")
    gs = qm.GSpace(p["lat"], p["cfg"].ecutwfc_ry, p["cfg"].grid, p["k"][None, :])
    psi = torch.from_numpy(p["psi"]).to(dev)
    s = gs.subspace(psi, psi).cpu().numpy()
    assert np.max(np.abs(s - np.eye(s.shape[0]))) <= 1e-12          # generator orthonormalises the rows
    gs.set_vloc(torch.from_numpy(p["v"]).to(dev))
    gs.set_nonlocal(0, torch.from_numpy(p["beta"]).to(dev), torch.from_numpy(p["dblk"]).to(dev))
    h = gs.subspace(psi, gs.apply_h(psi)).cpu().numpy()              # <psi_i|H psi_j>
    assert np.max(np.abs(h - np.conj(h.T))) <= 1e-11 * np.max(np.abs(h))
    s2 = gs.subspace(psi, psi).cpu().numpy()
    assert np.array_equal(s, s2)                                     # fixed-order split-K: bitwise reproducible
    gs.close()


def test_subspace_full_size_sampled_entries(qm):
    """cfg5 sphere (80 725 plane waves), 96 x 80 block: every entry against the library product (second opinion),
    sampled entries against the oracle."""
    p = problem("cfg5", 0, nbands=96, orthonormalise=False)
    ng = p["idx"].size
    rng = np.random.default_rng(9)
    a, b = p["psi"], _rand(rng, 80, ng)
    got = _run(qm, p, a, b)
    scale = np.linalg.norm(a, axis=1)[:, None] * np.linalg.norm(b, axis=1)[None, :]
    assert np.max(np.abs(got - np.conj(a) @ b.T) / scale) <= TOL
    ii, jj = rng.integers(0, 96, size=12), rng.integers(0, 80, size=12)
    for i, j in zip(ii, jj):
        ref = osub.vdot_matrix(a[i:i + 1], b[j:j + 1])[0, 0]
        assert abs(got[i, j] - ref) <= TOL * scale[i, j]


def test_subspace_bench_shape_512_by_512_sampled_entries(qm):
    """The shape bench.py times (512 x 512 states on the cfg5 sphere): 256 sampled entries, the four corners
    among them, against oracle/subspace.py; every entry against the library product as a second opinion."""
    p = problem("cfg5", 0, nbands=512, orthonormalise=False)
    ng = p["idx"].size
    rng = np.random.default_rng(21)
    a, b = p["psi"], _rand(rng, 512, ng)
    got = _run(qm, p, a, b)
    scale = np.linalg.norm(a, axis=1)[:, None] * np.linalg.norm(b, axis=1)[None, :]
    assert np.max(np.abs(got - np.conj(a) @ b.T) / scale) <= TOL
    ii = np.concatenate([[0, 0, 511, 511], rng.integers(0, 512, size=252)])
    jj = np.concatenate([[0, 511, 0, 511], rng.integers(0, 512, size=252)])
    for i, j in zip(ii, jj):
        ref = osub.vdot_matrix(a[i:i + 1], b[j:j + 1])[0, 0]
        assert abs(got[i, j] - ref) <= TOL * scale[i, j], (i, j)
