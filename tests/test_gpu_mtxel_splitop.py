"""GPU parity of the split-operator propagator (eq. 53) and the GW plane-wave matrix elements (eqs. 56-57)
against oracle/propagate.py and oracle/mtxel.py (-m gpu).  SURVEY.md 8(f) ranks 3 (second half) and 4.

Tolerances: split-operator 1e-11 per band like qm_apply_h (A13); matrix elements 1e-11 ||bra_n|| ||ket_n'|| (the natural
scale of an inner product, as for qm_subspace).
"""
import numpy as np
import pytest

from tests.common import TOL, band_errors, problem
from oracle import gsphere as og
from oracle import mtxel as om
from oracle import propagate as op
from workloads import CONFIGS, cell_for, make_kpoints, make_psi

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


# ---- split-operator ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,ik,dt", [("cfg1", 0, 0.05), ("cfg2", 4, 0.2), ("cfg3", 0, 0.02)])
def test_split_operator_all_elements(qm, name, ik, dt):
    torch, dev = _torch()
    p = problem(name, ik)
    cfg = p["cfg"]
    gs = qm.GSpace(p["lat"], cfg.ecutwfc_ry, cfg.grid, p["k"][None, :])
    gs.split_operator_set(torch.from_numpy(p["v"]).to(dev), dt)
    psi = torch.from_numpy(p["psi"]).to(dev)
    got = gs.split_operator_propagate(psi).cpu().numpy()
    ref = op.split_operator_propagate(p["psi"], p["miller"], p["g2"], p["v"], cfg.grid, dt)
    e_inf, e_2 = band_errors(got, ref)
    assert e_inf <= TOL and e_2 <= TOL, (e_inf, e_2)
    # it never needs V_loc / projectors to be set, and a second dt replaces the tables
    gs.split_operator_set(torch.from_numpy(p["v"]).to(dev), 2 * dt)
    got2 = gs.split_operator_propagate(psi).cpu().numpy()
    ref2 = op.split_operator_propagate(p["psi"], p["miller"], p["g2"], p["v"], cfg.grid, 2 * dt)
    e_inf, e_2 = band_errors(got2, ref2)
    assert e_inf <= TOL and e_2 <= TOL, (e_inf, e_2)
    gs.close()


@pytest.mark.parametrize("name,nb", [("cfg4", 32), ("cfg5", 16)])
def test_split_operator_sampled_rows_full_size(qm, name, nb):
    torch, dev = _torch()
    p = problem(name, 0, nbands=nb, orthonormalise=False)
    cfg = p["cfg"]
    dt = 0.03
    gs = qm.GSpace(p["lat"], cfg.ecutwfc_ry, cfg.grid)
    gs.split_operator_set(torch.from_numpy(p["v"]).to(dev), dt)
    got = gs.split_operator_propagate(torch.from_numpy(p["psi"]).to(dev)).cpu().numpy()
    ng = p["idx"].size
    rows = np.unique(np.concatenate([[0, 1, ng - 2, ng - 1], np.random.default_rng(9).integers(0, ng, 60)])).astype(np.int32)
    ref = op.split_operator_propagate(p["psi"], p["miller"], p["g2"], p["v"], cfg.grid, dt, rows=rows)
    e_inf, _ = band_errors(got[:, rows], ref)
    assert e_inf <= TOL, e_inf
    # every element against the library-FFT spelling of the same three factors, and the norm never grows
    from oracle import hpsi_fft as of
    half = np.exp(-0.25j * dt * p["g2"])
    alt = of.r2g(of.g2r(p["psi"] * half, p["idx"], cfg.grid) * np.exp(-1j * dt * p["v"]).reshape((1,) + cfg.grid),
                 p["idx"], cfg.grid) * half
    e_inf, e_2 = band_errors(got, alt)
    assert e_inf <= TOL and e_2 <= TOL, (e_inf, e_2)
    assert np.all(np.linalg.norm(got, axis=1) <= np.linalg.norm(p["psi"], axis=1) * (1 + 1e-12))
    gs.close()


def test_split_operator_errors(qm):
    torch, dev = _torch()
    p = problem("cfg1")
    gs = qm.GSpace(p["lat"], p["cfg"].ecutwfc_ry, p["cfg"].grid)
    psi = torch.from_numpy(p["psi"]).to(dev)
    with pytest.raises(qm.QmError) as e:
        gs.split_operator_propagate(psi)
    assert e.value.code == -2                          # QM_ENOTSET
    gs.split_operator_set(torch.from_numpy(p["v"]).to(dev), 0.1)
    with pytest.raises(qm.QmError) as e:
        qm.qm_split_operator_propagate(gs.handle, psi, psi)
    assert e.value.code == -1                          # overlap
    gs.close()


# ---- GW matrix elements ------------------------------------------------------------------------------------------
def _mtxel_inputs(name, ik_bra, ik_ket, nbra, nket, seed):
    cfg = CONFIGS[name]
    lat, _ = cell_for(cfg)
    kpts = make_kpoints(cfg)
    mb, ib, _ = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid, kpts[ik_bra])
    mk, ik, _ = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid, kpts[ik_ket])
    rng = np.random.default_rng(seed)
    bra = rng.standard_normal((nbra, ib.size)) + 1j * rng.standard_normal((nbra, ib.size))
    ket = rng.standard_normal((nket, ik.size)) + 1j * rng.standard_normal((nket, ik.size))
    return cfg, lat, kpts, (mb, ib, bra), (mk, ik, ket)


def _mtxel_err(got, ref, bra, ket):
    scale = np.linalg.norm(bra, axis=1)[:, None, None] * np.linalg.norm(ket, axis=1)[None, :, None]
    return float(np.max(np.abs(got - ref) / scale))


@pytest.mark.parametrize("name,ik_bra,ik_ket,ecut_eps,nbra,nket", [
    ("cfg1", 0, 0, 9.0, 3, 5), ("cfg2", 7, 2, 8.0, 4, 3), ("cfg2", 3, 3, 12.0, 2, 2), ("cfg3", 0, 0, 10.0, 5, 4)])
def test_matrix_elements_all_elements(qm, name, ik_bra, ik_ket, ecut_eps, nbra, nket):
    torch, dev = _torch()
    cfg, lat, kpts, (mb, ib, bra), (mk, ik, ket) = _mtxel_inputs(name, ik_bra, ik_ket, nbra, nket, 11)
    gs = qm.GSpace(lat, cfg.ecutwfc_ry, cfg.grid, kpts)
    me = gs.mtxel(ik_bra, ik_ket, ecut_eps)
    m_eps, i_eps, _ = og.gsphere(lat, ecut_eps, cfg.grid, kpts[ik_bra] - kpts[ik_ket], strict=True)
    assert me.num_g() == i_eps.size
    np.testing.assert_array_equal(me.index_map(), i_eps)           # index work: bit exact
    np.testing.assert_array_equal(me.miller(), m_eps)
    got = me.apply(torch.from_numpy(bra).to(dev), torch.from_numpy(ket).to(dev)).cpu().numpy()
    ref = om.matrix_elements(bra, mb, ket, mk, m_eps, cfg.grid)
    assert _mtxel_err(got, ref, bra, ket) <= TOL
    # repeated calls are bitwise reproducible and do not depend on what the work spaces held before
    again = me.apply(torch.from_numpy(bra).to(dev), torch.from_numpy(ket).to(dev)).cpu().numpy()
    np.testing.assert_array_equal(got, again)
    me.close()
    gs.close()


def test_matrix_elements_wrapping_grid(qm):
    """A box that holds the spheres but not 2 m_wfn + m_eps + 1: the lookups wrap (reading A8 / A21) on both sides."""
    torch, dev = _torch()
    lat = 10.26 * np.eye(3)
    grid = (12, 12, 12)
    kpts = np.array([[0.3, 0.0, -0.2], [0.0, 0.0, 0.0]])
    mb, ib, _ = og.gsphere(lat, 12.0, grid, kpts[0])
    mk, ik, _ = og.gsphere(lat, 12.0, grid, kpts[1])
    m_eps, i_eps, _ = og.gsphere(lat, 6.0, grid, kpts[0] - kpts[1], strict=True)
    rng = np.random.default_rng(2)
    bra = rng.standard_normal((2, ib.size)) + 1j * rng.standard_normal((2, ib.size))
    ket = rng.standard_normal((3, ik.size)) + 1j * rng.standard_normal((3, ik.size))
    gs = qm.GSpace(lat, 12.0, grid, kpts)
    me = gs.mtxel(0, 1, 6.0)
    got = me.apply(torch.from_numpy(bra).to(dev), torch.from_numpy(ket).to(dev)).cpu().numpy()
    ref = om.matrix_elements(bra, mb, ket, mk, m_eps, grid, wrap=True)
    assert _mtxel_err(got, ref, bra, ket) <= TOL
    assert np.max(np.abs(ref - om.matrix_elements(bra, mb, ket, mk, m_eps, grid, wrap=False))) > 1e-3
    me.close()
    gs.close()


@pytest.mark.parametrize("name,nbra,nket,ecut_eps", [("cfg4", 4, 6, 8.0), ("cfg5", 3, 4, 6.0), ("cfg5", 16, 16, 6.0)])
def test_matrix_elements_sampled_full_size(qm, name, nbra, nket, ecut_eps):
    """Sampled G against the plane-wave sum of eq. 56 (oracle/mtxel.py), every element against the FFT route of eq. 57;
    the last case is the 16 x 16 block bench.py times."""
    torch, dev = _torch()
    cfg, lat, kpts, (mb, ib, bra), (mk, ik, ket) = _mtxel_inputs(name, 0, 0, nbra, nket, 5)
    gs = qm.GSpace(lat, cfg.ecutwfc_ry, cfg.grid, kpts)
    me = gs.mtxel(0, 0, ecut_eps)
    m_eps, i_eps, _ = og.gsphere(lat, ecut_eps, cfg.grid, np.zeros(3), strict=True)
    np.testing.assert_array_equal(me.index_map(), i_eps)
    got = me.apply(torch.from_numpy(bra).to(dev), torch.from_numpy(ket).to(dev)).cpu().numpy()
    nsel = 40 if nbra * nket <= 24 else 16              # the direct sum costs nbra * nket * ng per sampled G
    sel = np.unique(np.concatenate([[0, 1, i_eps.size - 1], np.random.default_rng(6).integers(0, i_eps.size, nsel)]))
    ref = om.matrix_elements(bra, mb, ket, mk, m_eps[sel], cfg.grid)
    assert _mtxel_err(got[:, :, sel], ref, bra, ket) <= TOL
    # every element against the library-FFT route of eq. 57 (second opinion)
    alt = om.matrix_elements_fft(bra, ib, ket, ik, i_eps, cfg.grid)
    assert _mtxel_err(got, alt, bra, ket) <= TOL
    me.close()
    gs.close()
