"""CPU checks of the boundary: the library builds, loads without a GPU, exports every symbol that
include/vmat.h declares, and refuses to compute without a device (no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1005_4396_b200 import build

    return ctypes.CDLL(build.build())


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "vmat.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(vmat_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lib):
    import paper_1005_4396_b200 as vm

    names = declared_symbols()
    assert len(names) >= 12
    assert set(names) == set(vm.SYMBOLS)
    for n in names:
        assert hasattr(lib, n), n


def test_default_options(lib):
    import paper_1005_4396_b200 as vm

    o = vm.default_options()
    assert o.validate == 1 and o.master_eps > 0 and o.master_max_inner > 0


def test_create_argument_checks_run_before_any_cuda_call():
    import paper_1005_4396_b200 as vm

    L = vm.load_library()
    assert L.vmat_create(None, None, None, None) == vm.VMAT_EINVAL
    assert b"NULL" in L.vmat_last_error(None)
    assert L.vmat_destroy(None) == vm.VMAT_OK


def test_no_cpu_fallback_without_a_device():
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_1005_4396_b200 as vm

    rp = np.zeros(2 * 1 * 2 + 1, np.int64)
    z = np.zeros(4, np.float32)
    with pytest.raises(vm.VmatError) as e:
        vm.Plan.create(rp, np.zeros(0, np.int32), np.zeros(0, np.float32), z, z, z, np.array([0.0, 2.0]), 1, 2, 1, 0.1,
                       stream=0)
    assert e.value.code == vm.VMAT_ECUDA


def test_product_does_not_touch_the_oracle():
    # the product path shares no code with oracle/ and never imports it
    pkg = os.path.join(ROOT, "paper_1005_4396_b200")
    for d, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(d, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "vmat_oracle" not in src, f
