"""CPU-only checks of the boundary: libepr.so builds (nvcc cross-compiles sm_100a without a GPU), loads, and
exports every symbol include/epr.h declares; the binding fails loudly without a device (no CPU fallback)."""
import ctypes
import os
import re
import shutil

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "epr.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(epr_[a-z_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_2601_22793_b200 import build, lib_path
    if not os.path.exists(lib_path()):
        if shutil.which("nvcc") is None:
            pytest.skip("nvcc not available and libepr.so not built")
        build.build()
    return ctypes.CDLL(lib_path())


def test_header_symbols_are_exported(lib):
    names = _declared()
    assert {"epr_plan", "epr_forward", "epr_adjoint", "epr_precondition", "epr_retrieve"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/epr.h but not exported"


def test_binding_lists_the_same_entry_points():
    from paper_2601_22793_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()


def test_no_cpu_fallback_without_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    import paper_2601_22793_b200 as E
    with pytest.raises(E.EprError) as ei:
        E.epr_plan(256, 256, 6.5e-6, 1.0, [100.0], [1.0], [1000.0])
    assert ei.value.status == 3            # EPR_ECUDA: fails loudly


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2601_22793_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.replace("no oracle", ""), f"{f} mentions the oracle"


def test_host_binding_rejects_non_float32_buffers():
    """epr_retrieve_host takes float32 host buffers only: a float64 or 2-byte tensor of the right shape would make the
    library read / write the wrong number of bytes.  The check sits in the binding, ahead of the library call."""
    import numpy as np
    import torch
    from paper_2601_22793_b200 import binding

    class FakePlan:
        ny, nx, _h = 4, 8, None

    for bad in (torch.zeros((1, 4, 8), dtype=torch.float64), torch.zeros((1, 4, 8), dtype=torch.float16),
                torch.zeros((1, 4, 8), dtype=torch.bfloat16), np.zeros((1, 4, 8), dtype=np.float64)):
        with pytest.raises(TypeError):
            binding.epr_retrieve_host(FakePlan(), bad, bad, 1, 1.0)
