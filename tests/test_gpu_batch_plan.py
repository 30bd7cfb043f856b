"""qm_batch_plan_* beyond the happy path (-m gpu): a plan whose captured work-space addresses or projector shapes are no
longer those of the handle must refuse to launch (include/qm_hpsi.h, "STALE"), and a plan on a box that goes through the
unfused passes gives what the individual calls give."""
import os

import numpy as np
import pytest

from tests.common import TOL, band_errors, problem
from oracle import hpsi as oh

pytestmark = pytest.mark.gpu
QM_EINVAL = -1


@pytest.fixture(scope="module")
def qm():
    import __graft_entry__ as ge
    ge.build()
    import paper_2308_07277_b200 as q
    return q


def _setup(qm, name="cfg3", nproj_keep=None):
    import torch
    dev = torch.device("cuda:0")
    p = problem(name)
    cfg = p["cfg"]
    gs = qm.GSpace(p["lat"], cfg.ecutwfc_ry, cfg.grid, p["k"][None, :])
    gs.set_vloc(torch.from_numpy(p["v"]).to(dev))
    gs.set_nonlocal(0, torch.from_numpy(p["beta"]).to(dev), torch.from_numpy(p["dblk"]).to(dev))
    return torch, dev, p, gs


def test_plan_goes_stale_when_a_larger_call_moves_the_work_space(qm):
    """plan(8 bands) -> launch fine -> qm_apply_h(64 bands) re-allocates the stick planes -> the old graph would read and
    write freed memory: launch must return QM_EINVAL and launch nothing; a plan created afterwards works."""
    torch, dev, p, gs = _setup(qm)
    psi = torch.from_numpy(p["psi"]).to(dev)
    assert psi.shape[0] >= 64
    out8 = torch.zeros_like(psi[:8])
    plan = gs.batch_plan([(0, psi[:8], out8)])
    plan.launch()
    torch.cuda.synchronize()
    want8 = out8.clone()
    big = gs.apply_h(psi[:64])                          # needs 64 bands of work space: the 8-band block is freed
    torch.cuda.synchronize()
    assert torch.equal(big[:8], want8)                  # band results do not depend on the batch they are in
    out8.zero_()
    l0 = gs.launch_count()
    with pytest.raises(qm.QmError) as e:
        plan.launch()
    assert e.value.code == QM_EINVAL and "stale" in str(e.value)
    torch.cuda.synchronize()
    assert gs.launch_count() == l0 and not out8.any()   # nothing ran
    plan.close()
    plan2 = gs.batch_plan([(0, psi[:8], out8)])         # the work space is large enough now: no further move
    plan2.launch()
    gs.apply_h(psi[:32])                                # a smaller call moves nothing: the plan stays valid
    plan2.launch()
    torch.cuda.synchronize()
    assert torch.equal(out8, want8)
    plan2.close()
    gs.close()


def test_plan_goes_stale_when_the_projector_shape_changes(qm):
    """qm_set_nonlocal with another nproj after the plan was made: the graph holds the old tile counts -> QM_EINVAL.  The
    same nproj and d_block again (new values, same shape) keeps the plan valid and the launch uses the new values."""
    torch, dev, p, gs = _setup(qm)
    cfg = p["cfg"]
    psi = torch.from_numpy(np.ascontiguousarray(p["psi"][:16])).to(dev)
    out = torch.zeros_like(psi)
    plan = gs.batch_plan([(0, psi, out)])
    b = p["dblk"].shape[1]
    beta2 = np.ascontiguousarray(p["beta"] * 0.5)
    gs.set_nonlocal(0, torch.from_numpy(beta2).to(dev), torch.from_numpy(p["dblk"]).to(dev))       # same shape
    plan.launch()
    torch.cuda.synchronize()
    ref = oh.apply_h_rows(p["psi"][:16], p["miller"], p["g2"], p["vhat"], cfg.grid, beta2, oh.expand_d(p["dblk"]))
    e_inf, e_2 = band_errors(out.cpu().numpy(), ref)
    assert e_inf <= TOL and e_2 <= TOL
    nkeep = p["beta"].shape[0] - b                                                                 # one atom fewer
    gs.set_nonlocal(0, torch.from_numpy(np.ascontiguousarray(p["beta"][:nkeep])).to(dev),
                    torch.from_numpy(np.ascontiguousarray(p["dblk"][:-1])).to(dev))
    with pytest.raises(qm.QmError) as e:
        plan.launch()
    assert e.value.code == QM_EINVAL
    plan.close()
    gs.set_nonlocal(0, None, None)                                                                 # and local-only
    plan = gs.batch_plan([(0, psi, out)])
    gs.set_nonlocal(0, torch.from_numpy(p["beta"]).to(dev), torch.from_numpy(p["dblk"]).to(dev))
    with pytest.raises(qm.QmError) as e:
        plan.launch()
    assert e.value.code == QM_EINVAL
    plan.close()
    gs.close()


def test_plan_on_the_unfused_path(qm):
    """A batch plan on a handle that goes through the unfused y / x passes (QM_FORCE_UNFUSED): the capture makes no
    occupancy query or allocation, and the graph gives exactly what the individual calls give, against the oracle too."""
    import torch
    dev = torch.device("cuda:0")
    p0 = problem("cfg2", 0)
    cfg = p0["cfg"]
    os.environ["QM_FORCE_UNFUSED"] = "1"
    try:
        gs = qm.GSpace(p0["lat"], cfg.ecutwfc_ry, cfg.grid, p0["kpts"][:3])
    finally:
        os.environ.pop("QM_FORCE_UNFUSED", None)
    gs.set_vloc(torch.from_numpy(p0["v"]).to(dev))
    psi, out, want = [], [], []
    for ik in range(3):
        p = problem("cfg2", ik)
        gs.set_nonlocal(ik, torch.from_numpy(p["beta"]).to(dev), torch.from_numpy(p["dblk"]).to(dev))
        psi.append(torch.from_numpy(p["psi"]).to(dev))
        out.append(torch.zeros_like(psi[-1]))
    plan = gs.batch_plan([(ik, psi[ik], out[ik]) for ik in range(3)])      # before any plain call: capture is the first use
    for ik in range(3):
        want.append(gs.apply_h(psi[ik], k=ik).clone())
    for rep in range(2):
        for o in out:
            o.zero_()
        plan.launch()
        torch.cuda.synchronize()
        for ik in range(3):
            assert torch.equal(out[ik], want[ik]), (rep, ik)
    p = problem("cfg2", 2)
    ref = oh.apply_h_rows(p["psi"], p["miller"], p["g2"], p["vhat"], cfg.grid, p["beta"], oh.expand_d(p["dblk"]))
    e_inf, e_2 = band_errors(out[2].cpu().numpy(), ref)
    assert e_inf <= TOL and e_2 <= TOL
    plan.close()
    gs.close()
