"""GPU parity of qm_taylor_propagate (eq. 52) against oracle/propagate.py (-m gpu)."""
import numpy as np
import pytest

from tests.common import TOL, band_errors, problem
from oracle import hpsi as oh
from oracle import propagate as op

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def qm():
    import __graft_entry__ as ge
    ge.build()
    import paper_2308_07277_b200 as q
    return q


@pytest.mark.parametrize("name,nb,order,dt", [("cfg1", 8, 4, 0.05), ("cfg1", 3, 0, 0.1), ("cfg1", 5, 1, 0.1),
                                               ("cfg3", 17, 4, 0.02)])
def test_taylor_propagator_matches_oracle(qm, name, nb, order, dt):
    import torch
    dev = torch.device("cuda:0")
    p = problem(name)
    psi = np.ascontiguousarray(p["psi"][:nb])
    gs = qm.GSpace(p["lat"], p["cfg"].ecutwfc_ry, p["cfg"].grid, p["k"][None, :])
    gs.set_vloc(torch.from_numpy(p["v"]).to(dev))
    gs.set_nonlocal(0, torch.from_numpy(p["beta"]).to(dev), torch.from_numpy(p["dblk"]).to(dev))
    got = gs.taylor_propagate(torch.from_numpy(psi).to(dev), dt, order).cpu().numpy()
    d = oh.expand_d(p["dblk"])
    apply_h = lambda x: oh.apply_h_rows(x, p["miller"], p["g2"], p["vhat"], p["cfg"].grid, p["beta"], d)
    ref = op.taylor_propagate(psi, apply_h, dt, order)
    e_inf, e_2 = band_errors(got, ref)
    assert e_inf <= TOL and e_2 <= TOL, (e_inf, e_2)
    if order >= 4:      # the exact propagator is unitary: norms are conserved to the truncation order
        x = dt * 0.5 * np.max(p["g2"]) * 1.5
        assert np.max(np.abs(np.linalg.norm(got, axis=1) - 1.0)) <= 10 * x ** (order + 1)
    gs.close()


@pytest.mark.parametrize("name,nb", [("cfg4", 32), ("cfg5", 16)])
def test_taylor_propagator_full_size(qm, name, nb):
    """eq. 52 at the sizes bench.py times (one call batch of cfg4 / cfg5, order 4): every element against
    oracle.propagate.taylor_propagate fed with the paper's FFT route for H (oracle/hpsi_fft.py, tied to the direct sum in
    tests/test_oracle_hpsi.py), and sampled rows with the LAST power H^4 psi = H (H^3 psi) taken by the direct sum
    (oracle/hpsi.py apply_h_rows(rows=...)), so that the scale-and-accumulate kernel runs at full size under test."""
    import math
    import torch
    from oracle import hpsi_fft as of
    dev = torch.device("cuda:0")
    p = problem(name, 0, nbands=nb)
    cfg, dt, order = p["cfg"], 0.02, 4
    psi = np.ascontiguousarray(p["psi"])
    gs = qm.GSpace(p["lat"], cfg.ecutwfc_ry, cfg.grid, p["k"][None, :])
    gs.set_vloc(torch.from_numpy(p["v"]).to(dev))
    gs.set_nonlocal(0, torch.from_numpy(p["beta"]).to(dev), torch.from_numpy(p["dblk"]).to(dev))
    got = gs.taylor_propagate(torch.from_numpy(psi).to(dev), dt, order).cpu().numpy()
    gs.close()
    d = oh.expand_d(p["dblk"])
    powers = []

    def h_fft(x):
        powers.append(x)                                  # the operand of the r-th application is H^(r-1) psi
        return of.apply_h_fft(x, p["idx"], p["g2"], p["v"], cfg.grid, p["beta"], d)

    ref = op.taylor_propagate(psi, h_fft, dt, order)
    e_inf, e_2 = band_errors(got, ref)
    assert e_inf <= TOL and e_2 <= TOL, (e_inf, e_2)
    ng = p["idx"].size
    rows = np.unique(np.concatenate([[0, 1, ng - 2, ng - 1], np.random.default_rng(4).integers(0, ng, 20)])).astype(np.int32)
    ref3 = op.taylor_propagate(psi, lambda x: of.apply_h_fft(x, p["idx"], p["g2"], p["v"], cfg.grid, p["beta"], d), dt, order - 1)
    last = oh.apply_h_rows(powers[order - 1], p["miller"], p["g2"], p["vhat"], cfg.grid, p["beta"], d, rows=rows)
    ref_rows = ref3[:, rows] + ((-1j * dt) ** order / math.factorial(order)) * last
    scale = np.max(np.abs(ref), axis=1)[:, None]
    assert np.max(np.abs(got[:, rows] - ref_rows) / scale) <= TOL
