"""CPU thread-emulation of the FFT-path kernels vs numpy (host logic, no GPU).

tests/host_emu/emu_main.cu runs the same __host__ __device__ phase functions and the same
host-built stick tables as the CUDA kernels, with loops standing in for threads.  This checks the
index logic (sphere order, stick tables, padded/transposed line layouts, pruned x/y passes, every
radix codelet) against numpy's FFT.  It is a test of host logic, not a product code path.
"""
import os
import subprocess
import tempfile

import numpy as np
import pytest

from oracle import gsphere as og
from tests.common import G2_TOL_U, UNIT_ROUNDOFF, exact_g2

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "host_emu", "emu_main.cu")
FCC = 0.5 * np.array([[-1.0, 0, 1], [0, 1, 1], [-1, 1, 0]])


@pytest.fixture(scope="module")
def emu_bin():
    out = os.path.join(tempfile.gettempdir(), f"qm_emu_main_{os.getuid()}")
    deps = [SRC] + [os.path.join(ROOT, "paper_2308_07277_b200", "csrc", f)
                    for f in ("fft_phases.cuh", "fft_reg.cuh", "gspace_host.h", "qm_plan.h", "roots_gen.cuh")]
    if not os.path.exists(out) or os.path.getmtime(out) < max(os.path.getmtime(d) for d in deps):
        subprocess.run(["nvcc", "-std=c++17", "-O1", "-Wno-deprecated-gpu-targets", "-o", out, SRC], check=True)
    return out


# (n, lattice, ecut, k): chosen so that every supported radix pair is exercised at least once
CASES = [
    (8, 10.26 * FCC, 5.0, (0.0, 0.0, 0.0)),
    (12, 10.26 * FCC, 8.0, (0.1, -0.2, 0.3)),
    (16, 10.26 * FCC, 14.0, (0.0, 0.0, 0.0)),
    (18, 5.107 * np.array([[.5, .5, .5], [-.5, .5, .5], [-.5, -.5, .5]]), 160.0, (0.0, 0.0, 0.0)),
    (20, 10.26 * FCC, 20.0, (0.0, 0.0, 0.0)),
    (24, 10.26 * FCC, 25.0, (0.0, 0.0, 0.0)),
    (30, 10.26 * FCC, 30.0, (0.3, 0.3, -0.4)),
    (32, 10.26 * FCC, 30.0, (-0.45, 0.2, 0.1)),
    (36, 10.26 * np.eye(3), 20.0, (0.0, 0.0, 0.0)),
    (40, 10.26 * np.eye(3), 25.0, (0.0, 0.0, 0.0)),
    (48, 10.26 * np.eye(3), 30.0, (0.0, 0.0, 0.0)),
    (60, 14.0 * np.eye(3), 30.0, (0.0, 0.0, 0.0)),
    (64, 14.0 * np.eye(3), 30.0, (0.0, 0.0, 0.0)),
    (72, 16.0 * np.eye(3), 30.0, (0.0, 0.0, 0.0)),
    (80, 18.0 * np.eye(3), 30.0, (0.0, 0.0, 0.0)),
    (96, 20.52 * np.eye(3), 30.0, (0.0, 0.0, 0.0)),
    (100, 20.52 * np.eye(3), 30.0, (0.2, 0.1, -0.3)),
    (108, 22.0 * np.eye(3), 30.0, (0.0, 0.0, 0.0)),
    (120, 24.0 * np.eye(3), 30.0, (0.0, 0.0, 0.0)),
    (128, 26.0 * np.eye(3), 30.0, (0.0, 0.0, 0.0)),
    (144, 30.78 * np.eye(3), 30.0, (0.0, 0.0, 0.0)),
    # lengths above 144 (z kernels and the unfused passes on the GPU; the same line factorisations here)
    (160, 12.0 * np.eye(3), 16.0, (0.0, 0.0, 0.0)),
    (180, 12.0 * np.eye(3), 16.0, (0.1, 0.0, -0.2)),
    (192, 12.0 * np.eye(3), 16.0, (0.0, 0.0, 0.0)),
    (225, 12.0 * np.eye(3), 16.0, (0.0, 0.0, 0.0)),
    (240, 12.0 * np.eye(3), 16.0, (0.0, 0.0, 0.0)),
    (256, 12.0 * np.eye(3), 16.0, (0.0, 0.0, 0.0)),
]


@pytest.mark.parametrize("n,lat,ecut,k", CASES, ids=[f"n{c[0]}" for c in CASES])
def test_emulated_fft_path_matches_numpy(emu_bin, n, lat, ecut, k):
    grid = (n, n, n)
    miller, idx, g2 = og.gsphere(lat, ecut, grid, k)
    ng = idx.size
    rng = np.random.default_rng(n)
    nb = 2 if n < 96 else 1
    psi = rng.standard_normal((nb, ng)) + 1j * rng.standard_normal((nb, ng))
    v = rng.standard_normal(n ** 3)
    with tempfile.TemporaryDirectory() as d:
        np.ascontiguousarray(lat, dtype=np.float64).tofile(os.path.join(d, "lat.bin"))
        psi.tofile(os.path.join(d, "psi.bin"))
        v.tofile(os.path.join(d, "v.bin"))
        pre = os.path.join(d, "out")
        subprocess.run([emu_bin, str(n), os.path.join(d, "lat.bin"), repr(ecut), repr(k[0]), repr(k[1]), repr(k[2]),
                        str(nb), os.path.join(d, "psi.bin"), os.path.join(d, "v.bin"), pre], check=True,
                       capture_output=True)
        got_idx = np.fromfile(pre + ".idx", dtype=np.int32)
        got_g2 = np.fromfile(pre + ".g2", dtype=np.float64)
        hloc = np.fromfile(pre + ".hloc", dtype=np.complex128).reshape(nb, ng)
        g2r = np.fromfile(pre + ".g2r", dtype=np.complex128).reshape(nb, n, n, n)
        r2g = np.fromfile(pre + ".r2g", dtype=np.complex128).reshape(nb, ng)
    np.testing.assert_array_equal(got_idx, idx)                 # host tables vs oracle: bit exact
    # A14: the library's host |k+G|^2 table against the exact rational evaluation (not against the oracle's spelling)
    sel = np.arange(ng) if ng <= 2000 else np.random.default_rng(1).integers(0, ng, 2000)
    ex, sc = exact_g2(lat, k, miller[sel])
    assert np.all(np.abs(got_g2[sel] - ex) <= G2_TOL_U * UNIT_ROUNDOFF * sc)
    box = np.zeros((nb, n ** 3), dtype=np.complex128)
    box[:, idx] = psi
    psi_r = np.fft.ifftn(box.reshape(nb, n, n, n), axes=(1, 2, 3))
    scale = np.max(np.abs(psi_r))
    assert np.max(np.abs(g2r - psi_r)) < 1e-13 * scale * n
    back = np.fft.fftn(psi_r, axes=(1, 2, 3)).reshape(nb, -1)[:, idx]
    assert np.max(np.abs(r2g - back)) < 1e-12 * np.max(np.abs(back))
    want = np.fft.fftn(psi_r * v.reshape(1, n, n, n), axes=(1, 2, 3)).reshape(nb, -1)[:, idx] + 0.5 * g2 * psi
    assert np.max(np.abs(hloc - want)) < 1e-12 * np.max(np.abs(want))
