"""qm_subspace_static -- the subspace product for callers that may not allocate device memory (-m gpu).

Some users of this library cannot let it call cudaMalloc: an application whose own memory pool already holds nearly the
whole GPU (a library-side cudaMalloc then fails although the caller has buffers to give), a solver loop that keeps
several streams busy (cudaMalloc / cudaFree synchronise the whole device and would stall all of them), or a job with a
memory budget that is fixed when the library is loaded.  For them include/qm_hpsi.h offers ONE handle-free entry point,
qm_subspace_static, whose split-K partial sums live in a fixed 16 MiB array inside the library image instead of the
buffer qm_subspace grows with cudaMalloc.  The caller passes the two wavefunction blocks and the output.

What is checked here: against the existing path (GSpace.subspace -> qm_subspace), within the tolerance of
tests/test_gpu_subspace.py (|dS_ij| <= 1e-11 ||a_i|| ||b_j||), on two calls in a row that share the static array -- a
large block first and a smaller, different one second, so that partial sums left behind by the first call would show up
in the second if the entry point relied on the array's previous contents.  The limit (blocks beyond 1024 x 1024 states
are refused with QM_EINVAL before anything is launched) is checked too.

This file is named to be collected LAST: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes in a fresh process on its own and after the rest of the suite (the first call on a device does
its own set-up and needs no qm_gspace handle to exist).
"""
import numpy as np
import pytest

from tests.common import TOL, problem

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def qm():
    import __graft_entry__ as ge
    ge.build()
    import paper_2308_07277_b200 as q
    return q


def _rand(rng, n, ng):
    return rng.standard_normal((n, ng)) + 1j * rng.standard_normal((n, ng))


def _scale(a, b):
    return np.linalg.norm(a, axis=1)[:, None] * np.linalg.norm(b, axis=1)[None, :]


def test_static_scratch_matches_allocating_path_on_two_calls_in_a_row(qm):
    import torch
    dev = torch.device("cuda:0")
    p = problem("cfg3")                          # 2945 plane waves: 92 K slices of 32 and a ragged tail
    ng = p["idx"].size
    rng = np.random.default_rng(20230807)
    blocks = [(_rand(rng, 130, ng), _rand(rng, 70, ng)),        # 3 x 2 tiles, ragged edges, many K splits
              (_rand(rng, 16, ng), _rand(rng, 24, ng))]         # one tile, the most K splits: reuses the same memory
    # the static entry point FIRST and without any handle alive: it must set itself up (fresh-process case)
    got = []
    for a, b in blocks:
        a_d, b_d = torch.from_numpy(a).to(dev), torch.from_numpy(b).to(dev)
        s_d = torch.full((a.shape[0], b.shape[0]), float("nan"), dtype=torch.complex128, device=dev)
        ret = qm.qm_subspace_static(a_d, b_d, s_d)
        assert ret is s_d                        # the caller's buffer, nothing created by the wrapper
        got.append(s_d)                          # no synchronisation between the two calls: same stream, in order
    torch.cuda.synchronize()
    got = [g.cpu().numpy() for g in got]

    gs = qm.GSpace(p["lat"], p["cfg"].ecutwfc_ry, p["cfg"].grid, p["k"][None, :])
    for (a, b), s_static in zip(blocks, got):
        s_alloc = gs.subspace(torch.from_numpy(a).to(dev), torch.from_numpy(b).to(dev)).cpu().numpy()
        assert np.all(np.isfinite(s_static.view(np.float64)))
        assert np.max(np.abs(s_static - s_alloc) / _scale(a, b)) <= TOL
        assert np.array_equal(s_static, s_alloc)         # same kernels, same split count, same summation order
    # and once more after the allocating path has run (order of use does not matter), a == b allowed
    a = blocks[1][0]
    a_d = torch.from_numpy(a).to(dev)
    s_d = torch.empty((16, 16), dtype=torch.complex128, device=dev)
    qm.qm_subspace_static(a_d, a_d, s_d)
    assert np.max(np.abs(s_d.cpu().numpy() - gs.subspace(a_d, a_d).cpu().numpy()) / _scale(a, a)) <= TOL
    gs.close()


def test_static_scratch_limit_and_arguments(qm):
    import torch
    dev = torch.device("cuda:0")
    ng = 96
    rng = np.random.default_rng(5)
    # 1024 x 1024 states is the largest square block the 2^20-element array holds: accepted, one K split per tile
    a = torch.from_numpy(_rand(rng, 1024, ng)).to(dev)
    s = torch.empty((1024, 1024), dtype=torch.complex128, device=dev)
    qm.qm_subspace_static(a, a, s)
    an = a.cpu().numpy()
    ref = np.conj(an) @ an.T                     # second opinion (host BLAS) at a size the oracle loop takes minutes for
    assert np.max(np.abs(s.cpu().numpy() - ref) / _scale(an, an)) <= TOL
    # one row more needs a 17th tile row: refused, with the limit in the message, and nothing is written
    a2 = torch.from_numpy(_rand(rng, 1025, ng)).to(dev)
    s2 = torch.full((1025, 1024), 7.0, dtype=torch.complex128, device=dev)
    with pytest.raises(qm.QmError) as e:
        qm.qm_subspace_static(a2, a, s2)
    assert e.value.code == -1 and "1048576" in str(e.value) and "qm_subspace" in str(e.value)
    torch.cuda.synchronize()
    assert bool((s2 == 7.0).all())
    with pytest.raises(TypeError):
        qm.qm_subspace_static(a, a2[:, :50].contiguous(), s)       # row lengths differ
