"""GPU parity at full size against the direct-sum oracle, on what bench.py runs, and on non-cubic boxes (-m gpu).

SURVEY.md 8(c): ">= 2 full batches (32 bands) through the oracle"; readings A17 (call batch and one call with all
bands) and A19 (full / D = 0 / V = 0).  What the direct-sum oracle (oracle/hpsi_direct.c) sees at full size:
  cfg5  every output row of two 16-band call batches (bands 0-31);  rows sampled, 3 bands at the first, a middle and
        the last batch position of the 512-band run (both launch configurations: 32 calls of 16, one call of 512)
  cfg4  every output row of one 32-band call batch; sampled rows of 3 x 3 bands of the 256-band run
Every other element of the 512 / 256-band runs is compared with the paper's FFT route (oracle/hpsi_fft.py, library
FFT + BLAS), which is itself tied to the direct sum in tests/test_oracle_hpsi.py and by the all-row batches above.
"""
import numpy as np
import pytest

from tests.common import TOL, band_errors, problem
from oracle import density as od
from oracle import gsphere as og
from oracle import hpsi as oh
from oracle import hpsi_fft as of
from workloads import CONFIGS, make_beta

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def qm():
    import __graft_entry__ as ge
    ge.build()
    import paper_2308_07277_b200 as q
    return q


def _torch():
    import torch
    return torch, torch.device("cuda:0")


def _setup(qm, p):
    torch, dev = _torch()
    gs = qm.GSpace(p["lat"], p["ecut"], p["grid"], np.asarray(p["k"])[None, :])
    np.testing.assert_array_equal(gs.index_map(0), p["idx"])
    gs.set_vloc(torch.from_numpy(p["v"]).to(dev))
    gs.set_nonlocal(0, torch.from_numpy(p["beta"]).to(dev), torch.from_numpy(p["dblk"]).to(dev))
    return gs


def _cfg_problem(name, nbands):
    p = dict(problem(name, 0, nbands=nbands, orthonormalise=False))
    p["ecut"], p["grid"] = p["cfg"].ecutwfc_ry, p["cfg"].grid
    return p


@pytest.mark.parametrize("name,cb,nbatch", [("cfg5", 16, 2), ("cfg4", 32, 1)])
def test_all_rows_of_full_call_batches_against_direct_sum(qm, name, cb, nbatch):
    """Every element of `nbatch` call batches, in bench.py's launch configuration, against the O(N_G^2) oracle."""
    torch, dev = _torch()
    p = _cfg_problem(name, cb * nbatch)
    gs = _setup(qm, p)
    psi = torch.from_numpy(p["psi"]).to(dev)
    out = torch.empty_like(psi)
    for b0 in range(0, cb * nbatch, cb):
        gs.apply_h(psi[b0:b0 + cb], out[b0:b0 + cb])
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    ref = oh.apply_h_rows(p["psi"], p["miller"], p["g2"], p["vhat"], p["grid"], p["beta"], oh.expand_d(p["dblk"]))
    e_inf, e_2 = band_errors(got, ref)
    assert e_inf <= TOL and e_2 <= TOL, (e_inf, e_2)
    gs.close()


@pytest.mark.parametrize("name", ["cfg5", "cfg4"])
def test_all_bands_one_call_and_batched_step(qm, name):
    """The two launch configurations bench.py times: all bands in ONE qm_apply_h call (A17) and the step of
    nbands / call_batch consecutive calls.  Every band against the FFT route; bands at the first, a middle and the
    last batch position against the direct sum on sampled rows."""
    torch, dev = _torch()
    cfg = CONFIGS[name]
    nb, cb = cfg.nbands, cfg.call_batch
    p = _cfg_problem(name, nb)
    gs = _setup(qm, p)
    psi = torch.from_numpy(p["psi"]).to(dev)
    one = gs.apply_h(psi).cpu().numpy()
    out = torch.empty_like(psi)
    for b0 in range(0, nb, cb):
        gs.apply_h(psi[b0:b0 + cb], out[b0:b0 + cb])
    torch.cuda.synchronize()
    step = out.cpu().numpy()
    d = oh.expand_d(p["dblk"])
    ng = p["idx"].size
    worst = 0.0
    for b0 in range(0, nb, 16):                      # FFT route, 16 bands at a time (host memory)
        alt = of.apply_h_fft(p["psi"][b0:b0 + 16], p["idx"], p["g2"], p["v"], p["grid"], p["beta"], d)
        for got in (one, step):
            e_inf, e_2 = band_errors(got[b0:b0 + 16], alt)
            worst = max(worst, e_inf, e_2)
    assert worst <= TOL, worst
    rng = np.random.default_rng(5)
    rows = np.unique(np.concatenate([[0, 1, ng - 2, ng - 1], rng.integers(0, ng, size=60)])).astype(np.int32)
    nbatch = nb // cb
    bands = np.concatenate([[b * cb, b * cb + cb // 2, b * cb + cb - 1] for b in (0, nbatch // 2, nbatch - 1)])
    ref = oh.apply_h_rows(np.ascontiguousarray(p["psi"][bands]), p["miller"], p["g2"], p["vhat"], p["grid"],
                          p["beta"], d, rows=rows)
    for got in (one, step):
        e_inf, _ = band_errors(got[np.ix_(bands, rows)], ref)
        assert e_inf <= TOL, e_inf
    gs.close()


# ---- boxes with n3 != n1 and non-cubic lattices ------------------------------------------------------------------
def _custom(lat, pos, ecut, grid, k, nb, seed, db=4):
    """Inputs for an arbitrary cell through the same generators (beta: reading A11) and plain seeded draws."""
    lat = np.asarray(lat, dtype=np.float64)
    k = np.asarray(k, dtype=np.float64)
    miller, idx, g2 = og.gsphere(lat, ecut, grid, k)
    rng = np.random.default_rng(seed)
    ng = idx.size
    psi = rng.standard_normal((nb, ng)) + 1j * rng.standard_normal((nb, ng))
    v = rng.standard_normal(int(np.prod(grid)))
    v /= np.max(np.abs(v))
    beta = make_beta(None, lat, np.asarray(pos, dtype=np.float64), k, miller)
    a = rng.standard_normal((beta.shape[0] // db, db, db))
    dblk = 0.5 * (a + np.transpose(a, (0, 2, 1)))
    return dict(lat=lat, ecut=ecut, grid=tuple(grid), k=k, miller=miller, idx=idx, g2=g2, psi=psi, v=v,
                vhat=oh.vhat_box(v, grid), beta=beta, dblk=dblk)


_A = 10.26
_TETRA = np.diag([_A, _A, 1.5 * _A])
_BCC = 0.5 * 12.0 * np.array([[1.0, 1, 1], [-1, 1, 1], [-1, -1, 1]])
_HEX = np.array([[9.0, 0, 0], [-4.5, 4.5 * np.sqrt(3.0), 0], [0, 0, 14.0]])
_POS2 = [[0.0, 0.0, 0.0], [2.1, 2.4, 3.3]]
_BOX_CASES = [
    # id, lattice, ecut, grid, k, alias free?
    ("tetragonal_48x48x72", _TETRA, 30.0, (48, 48, 72), (0.0, 0.0, 0.0), True),
    ("tetragonal_36x36x48_k_aliased_in_z", _TETRA, 25.0, (36, 36, 48), (0.2, -0.1, 0.3), False),
    ("tetragonal_aliased_24x24x32", _TETRA, 25.0, (24, 24, 32), (0.0, 0.0, 0.0), False),
    ("tetragonal_aliased_48x48x36", np.diag([1.4 * _A, 1.4 * _A, _A]), 30.0, (48, 48, 36), (0.0, 0.0, 0.0), False),
    ("bcc_36", _BCC, 27.0, (36, 36, 36), (0.1, 0.2, -0.3), True),
    ("hexagonal_40x40x60", _HEX, 28.0, (40, 40, 60), (0.0, 0.0, 0.25), True),
]


@pytest.mark.parametrize("cid,lat,ecut,grid,k,alias_free", _BOX_CASES, ids=[c[0] for c in _BOX_CASES])
def test_other_boxes_full_h_debug_hooks_and_density(qm, cid, lat, ecut, grid, k, alias_free):
    """n3 != n1 (per-axis z dispatch, z-label transposition in the V / density layouts, MODE 1/2 box strides),
    non-cubic and non-orthogonal lattices, aliased grids with larger radices: every element of the full H against the
    direct sum, g2r / r2g against the library FFT, density against the direct synthesis."""
    torch, dev = _torch()
    p = _custom(lat, _POS2, ecut, grid, k, nb=5, seed=len(cid))
    gs = _setup(qm, p)
    assert gs.alias_free(0) == alias_free
    psi = torch.from_numpy(p["psi"]).to(dev)
    got = gs.apply_h(psi).cpu().numpy()
    ref = oh.apply_h_rows(p["psi"], p["miller"], p["g2"], p["vhat"], grid, p["beta"], oh.expand_d(p["dblk"]))
    e_inf, e_2 = band_errors(got, ref)
    assert e_inf <= TOL and e_2 <= TOL, (e_inf, e_2)
    # debug hooks (A5) on the same box
    box = gs.g2r(psi).cpu().numpy()
    want = of.g2r(p["psi"], p["idx"], grid).reshape(5, -1)
    assert np.max(np.abs(box - want)) <= 1e-12 * np.max(np.abs(want))
    rng = np.random.default_rng(1)
    n = int(np.prod(grid))
    r = rng.standard_normal((2, n)) + 1j * rng.standard_normal((2, n))
    got_g = gs.r2g(torch.from_numpy(r).to(dev)).cpu().numpy()
    want_g = np.fft.fftn(r.reshape((2,) + tuple(grid)), axes=(1, 2, 3)).reshape(2, -1)[:, p["idx"]]
    assert np.max(np.abs(got_g - want_g)) <= 1e-12 * np.max(np.abs(want_g))
    # density on sampled points
    occ = np.linspace(2.0, 0.5, 5)
    gs.density_reset()
    gs.density_accumulate(psi, torch.from_numpy(occ).to(dev))
    rho = gs.density_get().cpu().numpy().reshape(grid)
    pts = np.stack([rng.integers(0, grid[i], size=200) for i in range(3)], axis=1)
    rref = od.density(p["psi"], p["miller"], occ, grid, points=pts)
    assert np.max(np.abs(rho[pts[:, 0], pts[:, 1], pts[:, 2]] - rref)) <= TOL * np.max(rref)
    gs.close()
