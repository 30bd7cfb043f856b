"""The C-ABI library loads and exports every symbol include/qm_hpsi.h declares (no compute without a GPU)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import __graft_entry__ as ge
    ge.build()
    import paper_2308_07277_b200 as qm
    return qm


def _declared():
    text = open(os.path.join(ROOT, "include", "qm_hpsi.h")).read()
    return sorted(set(re.findall(r"QM_API\s+(?:const\s+char\s*\*|int)\s*(qm_\w+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert len(names) >= 20
    cdll = ctypes.CDLL(lib.LIB_PATH)
    for n in names:
        assert hasattr(cdll, n), n
    assert sorted(lib.EXPORTS) == names          # the binding covers the whole header
    assert "sm_100a" in lib.qm_version()


def test_no_cpu_fallback_and_argument_errors(lib):
    import torch
    assert lib.qm_fft_size_supported(144) and lib.qm_fft_size_supported(24) and not lib.qm_fft_size_supported(7)
    lat = np.eye(3) * 10.26
    with pytest.raises(lib.QmError) as e:
        lib.qm_gspace_create(lat, 30.0, (7, 7, 7))
    assert e.value.code == -3                    # QM_EGRID: unsupported length
    with pytest.raises(lib.QmError) as e:
        lib.qm_gspace_create(lat, -1.0, (48, 48, 48))
    assert e.value.code == -1                    # QM_EINVAL
    if not torch.cuda.is_available():
        with pytest.raises(lib.QmError) as e:
            lib.qm_gspace_create(lat, 30.0, (48, 48, 48))
        assert e.value.code == -4                # QM_ECUDA: fails loudly, no CPU path
        with pytest.raises(lib.QmError):
            lib.qm_probe_fp64_tensor_peak()


def test_product_does_not_import_oracle():
    # the product path must not route through oracle/ (or workloads/)
    pkg = os.path.join(ROOT, "paper_2308_07277_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, re.M), f
                assert "oracle/" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2308_07277_b200", text, re.M), f
            assert "libqm_hpsi" not in text and "csrc" not in text, f
