"""GPU parity on boxes the fused plane kernel does not take: the unfused y | x | y passes (gen_kernels.cuh) (-m gpu).

PAPER.md:689-712: `GSpace` takes any lattice and cut-off, so n1 != n2 (orthorhombic, hexagonal cells), axes longer than
144 and plane arrays beyond one SM's shared memory (the 432- and 1024-atom runs) are ordinary
inputs.  Every operation that goes through the xy passes is checked on such boxes against the same oracles as on the
fused path: qm_apply_h (full H, direct sum), the debug hooks, the density, the split-operator step and the GW matrix
elements; and the five-config path is re-run with the unfused passes forced (QM_FORCE_UNFUSED) against the direct sum.
Tolerance 1e-11 per band (A13) throughout.
"""
import os

import numpy as np
import pytest

from tests.common import TOL, band_errors, problem
from oracle import density as od
from oracle import gsphere as og
from oracle import hpsi as oh
from oracle import hpsi_fft as of
from oracle import mtxel as om
from oracle import propagate as op

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


class _forced_unfused:
    """The handle reads QM_FORCE_UNFUSED when it is created."""

    def __enter__(self):
        os.environ["QM_FORCE_UNFUSED"] = "1"

    def __exit__(self, *a):
        os.environ.pop("QM_FORCE_UNFUSED", None)


def _projectors(lat, miller, k, natoms, seed):
    """Four Gaussian projectors per atom (A11: s and three p) at seeded positions, dense symmetric 4x4 D blocks."""
    rng = np.random.default_rng(seed)
    pos = rng.random((natoms, 3)) @ lat
    b = 2.0 * np.pi * np.linalg.inv(lat).T
    q = (np.asarray(miller, dtype=np.float64) + np.asarray(k)[None, :]) @ b
    q2 = np.sum(q * q, axis=1)
    vol = abs(np.linalg.det(lat))
    rows = []
    for t in pos:
        sf = np.exp(-1j * (q @ t)) * np.exp(-q2 / 4.0) / np.sqrt(vol)
        rows.append(sf)
        for a in range(3):
            rows.append(-1j * q[:, a] * sf)
    a = rng.standard_normal((natoms, 4, 4))
    return np.ascontiguousarray(np.array(rows)), 0.5 * (a + np.transpose(a, (0, 2, 1)))


# (lattice rows, ecut [Ry], grid, k): n1 != n2 != n3; alias free / aliased; orthorhombic, hexagonal-type, triclinic
_ORTHO = np.diag([8.0, 10.5, 12.5])
_HEX = np.array([[9.0, 0.0, 0.0], [-4.5, 4.5 * np.sqrt(3.0), 0.0], [0.0, 0.0, 14.0]])
_TRI = np.array([[8.5, 0.3, -0.2], [1.1, 9.7, 0.4], [-0.6, 0.8, 11.9]])
_BOXES = [
    ("ortho", _ORTHO, 20.0, (24, 30, 36), (0.0, 0.0, 0.0)),
    ("ortho_k", _ORTHO, 20.0, (24, 32, 40), (0.21, -0.4, 0.13)),
    ("ortho_aliased", _ORTHO, 20.0, (12, 16, 18), (0.0, 0.0, 0.0)),
    ("hex", _HEX, 18.0, (24, 24, 36), (0.0, 0.0, 0.25)),          # n1 == n2: fused; same oracle, for contrast
    ("triclinic", _TRI, 16.0, (20, 24, 30), (0.1, 0.2, -0.3)),
    ("long_x", _ORTHO, 12.0, (48, 18, 20), (0.0, 0.0, 0.0)),
    ("long_y", _ORTHO, 12.0, (16, 60, 24), (0.0, 0.0, 0.0)),
]


@pytest.mark.parametrize("tag,lat,ecut,grid,k", _BOXES, ids=[b[0] for b in _BOXES])
def test_full_h_on_general_boxes(qm, tag, lat, ecut, grid, k):
    """Every element of qm_apply_h (T + L + NL) against the direct-sum oracle; index map bit exact."""
    torch, dev = _torch()
    kk = np.array(k, dtype=float)
    miller, idx, g2 = og.gsphere(lat, ecut, grid, kk)
    ng = idx.size
    rng = np.random.default_rng(len(tag) + ng)
    nb = 5
    psi = rng.standard_normal((nb, ng)) + 1j * rng.standard_normal((nb, ng))
    v = rng.standard_normal(int(np.prod(grid)))
    beta, dblk = _projectors(lat, miller, kk, 3, ng)
    gs = qm.GSpace(lat, ecut, grid, kk[None, :])
    assert np.array_equal(gs.index_map(0), idx)
    gs.set_vloc(torch.from_numpy(v).to(dev))
    gs.set_nonlocal(0, torch.from_numpy(beta).to(dev), torch.from_numpy(dblk).to(dev))
    got = gs.apply_h(torch.from_numpy(psi).to(dev)).cpu().numpy()
    ref = oh.apply_h_rows(psi, miller, g2, oh.vhat_box(v, grid), grid, beta, oh.expand_d(dblk))
    e_inf, e_2 = band_errors(got, ref)
    assert e_inf <= TOL and e_2 <= TOL, (e_inf, e_2)
    gs.close()


def test_hooks_density_splitop_on_a_general_box(qm):
    """g2r / r2g, density, split-operator and matrix elements on an n1 != n2 != n3 box."""
    torch, dev = _torch()
    lat, ecut, grid = _ORTHO, 20.0, (24, 30, 36)
    kpts = np.array([[0.0, 0.0, 0.0], [0.25, -0.1, 0.3]])
    gs = qm.GSpace(lat, ecut, grid, kpts)
    rng = np.random.default_rng(5)
    n = int(np.prod(grid))
    v = rng.standard_normal(n)
    for ik in (0, 1):
        miller, idx, g2 = og.gsphere(lat, ecut, grid, kpts[ik])
        ng = idx.size
        psi = rng.standard_normal((3, ng)) + 1j * rng.standard_normal((3, ng))
        pg = torch.from_numpy(psi).to(dev)
        # debug hooks
        box = gs.g2r(pg, k=ik)
        ref_box = of.g2r(psi, idx, grid).reshape(3, -1)
        assert np.max(np.abs(box.cpu().numpy() - ref_box)) <= 1e-12 * np.max(np.abs(ref_box))
        back = gs.r2g(box, k=ik).cpu().numpy()
        ref_back = of.r2g(ref_box.reshape((3,) + grid), idx, grid)
        assert np.max(np.abs(back - ref_back)) <= 1e-12 * np.max(np.abs(ref_back))
        # split-operator step (eq. 53) against the direct-sum oracle
        dt = 0.04
        gs.split_operator_set(torch.from_numpy(v).to(dev), dt)
        got = gs.split_operator_propagate(pg, k=ik).cpu().numpy()
        ref = op.split_operator_propagate(psi, miller, g2, v, grid, dt)
        e_inf, e_2 = band_errors(got, ref)
        assert e_inf <= TOL and e_2 <= TOL, (ik, e_inf, e_2)
    # density at sampled points (eq. 2), two batches, against the direct synthesis
    miller, idx, g2 = og.gsphere(lat, ecut, grid, kpts[1])
    psi = rng.standard_normal((6, idx.size)) + 1j * rng.standard_normal((6, idx.size))
    occ = rng.random(6)
    gs.density_reset()
    for b0 in (0, 4):
        gs.density_accumulate(torch.from_numpy(np.ascontiguousarray(psi[b0:b0 + 4])).to(dev),
                              torch.from_numpy(np.ascontiguousarray(occ[b0:b0 + 4])).to(dev), weight=0.5, k=1)
    rho = gs.density_get(scale=2.0).cpu().numpy().reshape(-1)
    pts = np.stack([rng.integers(0, g, 400) for g in grid], axis=1)
    ref = od.density(psi, miller, occ, grid, points=pts, scale=1.0)
    flat = (pts[:, 0] * grid[1] + pts[:, 1]) * grid[2] + pts[:, 2]
    assert np.max(np.abs(rho[flat] - ref)) <= TOL * np.max(ref)
    assert rho.min() >= 0.0
    # GW matrix elements (eqs. 56-57) between the two k-points
    mb, ib, _ = og.gsphere(lat, ecut, grid, kpts[1])
    mk, ikk, _ = og.gsphere(lat, ecut, grid, kpts[0])
    bra = rng.standard_normal((2, ib.size)) + 1j * rng.standard_normal((2, ib.size))
    ket = rng.standard_normal((3, ikk.size)) + 1j * rng.standard_normal((3, ikk.size))
    me = gs.mtxel(1, 0, 6.0)
    # the epsilon sphere is the oracle's (strict cut-off at q = k_bra - k_ket, reading A21), not the library's own list
    m_eps, i_eps, _ = og.gsphere(lat, 6.0, grid, kpts[1] - kpts[0], strict=True)
    np.testing.assert_array_equal(me.miller(), m_eps)
    np.testing.assert_array_equal(me.index_map(), i_eps)
    got = me.apply(torch.from_numpy(bra).to(dev), torch.from_numpy(ket).to(dev)).cpu().numpy()
    ref = om.matrix_elements(bra, mb, ket, mk, m_eps, grid)
    scale = np.linalg.norm(bra, axis=1)[:, None, None] * np.linalg.norm(ket, axis=1)[None, :, None]
    assert np.max(np.abs(got - ref) / scale) <= TOL
    me.close()
    gs.close()


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3"])
def test_forced_unfused_matches_direct_sum(qm, name):
    """The BASELINE.json cells through the unfused passes: every element of the full H against the direct sum."""
    torch, dev = _torch()
    p = problem(name)
    cfg = p["cfg"]
    with _forced_unfused():
        gs = qm.GSpace(p["lat"], cfg.ecutwfc_ry, cfg.grid, p["k"][None, :])
    gs.set_vloc(torch.from_numpy(p["v"]).to(dev))
    gs.set_nonlocal(0, torch.from_numpy(p["beta"]).to(dev), torch.from_numpy(p["dblk"]).to(dev))
    got = gs.apply_h(torch.from_numpy(p["psi"]).to(dev)).cpu().numpy()
    ref = oh.apply_h_rows(p["psi"], p["miller"], p["g2"], p["vhat"], cfg.grid, p["beta"], oh.expand_d(p["dblk"]))
    e_inf, e_2 = band_errors(got, ref)
    assert e_inf <= TOL and e_2 <= TOL, (e_inf, e_2)
    gs.close()


def test_forced_unfused_cfg5_sampled_rows(qm):
    """cfg5 (one 16-band batch) through the unfused passes: sampled rows against the direct sum, all rows bitwise stable."""
    torch, dev = _torch()
    p = problem("cfg5", 0, nbands=16, orthonormalise=False)
    cfg = p["cfg"]
    with _forced_unfused():
        gs = qm.GSpace(p["lat"], cfg.ecutwfc_ry, cfg.grid)
    gs.set_vloc(torch.from_numpy(p["v"]).to(dev))
    gs.set_nonlocal(0, torch.from_numpy(p["beta"]).to(dev), torch.from_numpy(p["dblk"]).to(dev))
    psi = torch.from_numpy(p["psi"]).to(dev)
    first = gs.apply_h(psi).clone()
    assert torch.equal(first, gs.apply_h(psi))
    got = first.cpu().numpy()
    rows = np.sort(np.random.default_rng(3).choice(p["idx"].size, 48, replace=False)).astype(np.int32)
    ref = oh.apply_h_rows(p["psi"], p["miller"], p["g2"], p["vhat"], cfg.grid, p["beta"], oh.expand_d(p["dblk"]), rows=rows)
    d = np.abs(got[:, rows] - ref)
    assert np.max(d.max(axis=1) / np.abs(got).max(axis=1)) <= TOL
    gs.close()


# every FFT length above 144 on every axis (the z kernels take axis 3, the unfused y / x passes axes 2 / 1)
_LONG = [(160, 180, 192), (180, 192, 160), (192, 160, 180), (225, 240, 256), (240, 256, 225), (256, 225, 240)]


@pytest.mark.parametrize("grid", _LONG, ids=["x".join(map(str, g)) for g in _LONG])
def test_long_axes_local_and_kinetic_terms(qm, grid):
    """T + L on boxes with axes of 160 ... 256 points, sampled rows against the direct sum and every element against the
    library-FFT route (oracle/hpsi_fft.py)."""
    torch, dev = _torch()
    lat, ecut = np.diag([9.0, 10.0, 11.0]), 14.0
    kk = np.array([0.1, -0.2, 0.05])
    miller, idx, g2 = og.gsphere(lat, ecut, grid, kk)
    rng = np.random.default_rng(grid[0])
    nb = 2
    psi = rng.standard_normal((nb, idx.size)) + 1j * rng.standard_normal((nb, idx.size))
    v = rng.standard_normal(int(np.prod(grid)))
    gs = qm.GSpace(lat, ecut, grid, kk[None, :])
    assert np.array_equal(gs.index_map(0), idx)
    gs.set_vloc(torch.from_numpy(v).to(dev))
    gs.set_nonlocal(0, None, None)
    got = gs.apply_h(torch.from_numpy(psi).to(dev)).cpu().numpy()
    ref = of.apply_h_fft(psi, idx, g2, v, grid)
    e_inf, e_2 = band_errors(got, ref)
    assert e_inf <= TOL and e_2 <= TOL, (e_inf, e_2)
    rows = np.sort(rng.choice(idx.size, 24, replace=False)).astype(np.int32)
    ref2 = oh.apply_h_rows(psi, miller, g2, oh.vhat_box(v, grid), grid, rows=rows)
    assert np.max(np.abs(got[:, rows] - ref2)) <= TOL * np.max(np.abs(got))
    gs.close()


def test_512_atom_cell_local_and_kinetic(qm):
    """4 x 4 x 4 cubic diamond-structure supercell (512 atoms, a = 41.04 bohr, 30 Ry, 192^3): the plane array no longer fits
    one SM's shared memory.  Two bands, T + L: every element against the library-FFT route, sampled rows against the
    direct sum."""
    torch, dev = _torch()
    lat, ecut, grid = np.eye(3) * 41.04, 30.0, (192, 192, 192)
    miller, idx, g2 = og.gsphere(lat, ecut, grid)
    rng = np.random.default_rng(512)
    nb = 2
    psi = rng.standard_normal((nb, idx.size)) + 1j * rng.standard_normal((nb, idx.size))
    v = rng.standard_normal(int(np.prod(grid)))
    gs = qm.GSpace(lat, ecut, grid)
    assert np.array_equal(gs.index_map(0), idx)
    gs.set_vloc(torch.from_numpy(v).to(dev))
    gs.set_nonlocal(0, None, None)
    got = gs.apply_h(torch.from_numpy(psi).to(dev)).cpu().numpy()
    ref = of.apply_h_fft(psi, idx, g2, v, grid)
    e_inf, e_2 = band_errors(got, ref)
    assert e_inf <= TOL and e_2 <= TOL, (e_inf, e_2)
    rows = np.sort(rng.choice(idx.size, 16, replace=False)).astype(np.int32)
    ref2 = oh.apply_h_rows(psi, miller, g2, oh.vhat_box(v, grid), grid, rows=rows)
    assert np.max(np.abs(got[:, rows] - ref2)) <= TOL * np.max(np.abs(got))
    gs.close()
