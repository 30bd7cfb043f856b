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
