"""C-ABI checks that need no GPU: the library loads, exports every symbol include/fdas.h
declares, and rejects bad arguments before touching CUDA."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def F():
    from paper_2206_12205_b200 import _build, fdas
    _build.build()
    fdas.lib()
    return fdas


def declared_functions():
    src = open(os.path.join(ROOT, "include", "fdas.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fdas_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(F):
    names = declared_functions()
    assert len(names) >= 15
    L = ctypes.CDLL(F.LIB_PATH)
    for n in names:
        assert hasattr(L, n), n
    assert sorted(F.EXPORTS) == names


def test_status_strings(F):
    assert F.fdas_status_string(0) == "FDAS_OK"
    assert F.fdas_status_string(F.FDAS_ERR_NOT_BUILT) == "FDAS_ERR_NOT_BUILT"
    assert F.fdas_status_string(99) == "FDAS_ERR_UNKNOWN"


@pytest.mark.parametrize("args", [
    (1 << 16, -1.0, 2.0, 1024, 1),      # zmax < 0
    (1 << 16, 20.0, 0.0, 1024, 1),      # dz <= 0
    (1 << 16, 20.0, 2.0, 1000, 1),      # seglen not a supported power of two
    (1 << 16, 20.0, 2.0, 1024, 7),      # unknown precision
    ((1 << 16) + 1, 20.0, 2.0, 1024, 1),  # N odd
    (1024, 20.0, 2.0, 1024, 1),         # N < 2*seglen
    (1 << 16, 480.0, 2.0, 512, 1),      # seglen <= 2*m_max (m_max = 256)
    (1 << 16, 20.0, 0.001, 1024, 1),    # K too large
])
def test_plan_create_rejects_bad_arguments(F, args):
    rc, h = F.fdas_plan_create(*args)
    assert rc == F.FDAS_ERR_INVALID_ARG and not h.value


def test_unsupported_and_null_handling(F):
    rc, h = F.fdas_plan_create(1 << 16, 20.0, 2.0, 8192, 1)
    assert rc == F.FDAS_ERR_UNSUPPORTED and not h.value
    assert F.lib().fdas_plan_create(None, 1 << 16, 20.0, 2.0, 1024, 1) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_plan_destroy(None) == F.FDAS_OK
    assert F.fdas_last_cuda_error(None) == -1
    assert F.fdas_build_templates(None) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_convolve(None, 0, 0) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_plan_info(None)[0] == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_set_algorithm(None, F.FDAS_ALGO_MMA) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_get_algorithm(None)[0] == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_tapmatrix_host(None, 0, 0) == F.FDAS_ERR_INVALID_ARG


def test_no_cpu_fallback_without_a_device(F):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    rc, h = F.fdas_plan_create(1 << 16, 20.0, 2.0, 1024, 1)
    assert rc == F.FDAS_ERR_CUDA and not h.value


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2206_12205_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "fdas_oracle" not in txt, f
