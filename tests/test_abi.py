"""CPU-side checks of the boundary: the C-ABI library loads without a GPU and exports every symbol that
include/fmm.h declares; argument errors are status codes, never aborts."""
import ctypes as C
import os
import re

import pytest

from paper_2511_15269_b200 import build as fbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    fbuild.build()
    from paper_2511_15269_b200 import fmm
    return fmm.lib()


def test_every_declared_symbol_is_exported(L):
    hdr = open(os.path.join(ROOT, "include", "fmm.h")).read()
    names = set(re.findall(r"\b(fmm_[a-z0-9_]+)\s*\(", hdr))
    assert {"fmm_plan_create", "fmm_evaluate", "fmm_plan_destroy"} <= names
    from paper_2511_15269_b200 import fmm
    assert names == set(fmm.EXPORTS)
    for n in names:
        assert hasattr(L, n), n


def test_argument_errors_are_status_codes(L):
    from paper_2511_15269_b200 import fmm
    h = C.c_void_p()
    adm = fmm.fmm_admissibility(0.77, 0)
    # NULL positions
    st = L.fmm_plan_create(None, 10, 4, 8, 2, C.byref(adm), fmm.FMM_F32, None, C.byref(h))
    assert st == fmm.FMM_ERR_INVALID_ARG and h.value is None and "NULL" in fmm.fmm_last_error()
    dummy = C.c_void_p(16)
    for (N, p, nmax, s, theta) in [(0, 4, 8, 2, 0.77), (10, -1, 8, 2, 0.77), (10, 99, 8, 2, 0.77), (10, 4, 0, 2, 0.77), (10, 4, 8, 0, 0.77),
                                   (10, 4, 8, 2, 0.0), (10, 4, 8, 2, 1.0), (10, 4, 8, 2, float("nan"))]:
        adm = fmm.fmm_admissibility(theta, 0)
        st = L.fmm_plan_create(dummy, N, p, nmax, s, C.byref(adm), fmm.FMM_F32, None, C.byref(h))
        assert st == fmm.FMM_ERR_INVALID_ARG and h.value is None
    adm = fmm.fmm_admissibility(0.77, 2)  # cross_level is 0 (same-level lists) or 1 (level marching)
    assert L.fmm_plan_create(dummy, 10, 4, 8, 2, C.byref(adm), fmm.FMM_F32, None, C.byref(h)) == fmm.FMM_ERR_INVALID_ARG
    assert L.fmm_evaluate(None, None, None, None, None) == fmm.FMM_ERR_INVALID_ARG
    assert L.fmm_plan_destroy(None) == fmm.FMM_OK
    assert fmm.fmm_version().startswith("paper_2511_15269_b200")


def test_no_cpu_fallback_without_device(L):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2511_15269_b200 import fmm
    h = C.c_void_p()
    adm = fmm.fmm_admissibility(0.77, 0)
    st = L.fmm_plan_create(C.c_void_p(16), 10, 4, 8, 2, C.byref(adm), fmm.FMM_F32, None, C.byref(h))
    assert st == fmm.FMM_ERR_CUDA and "no CPU fallback" in fmm.fmm_last_error()


def test_product_does_not_import_oracle():
    pk = os.path.join(ROOT, "paper_2511_15269_b200")
    for dp, _, fs in os.walk(pk):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "oracle/" not in src.replace("oracle/ ", "").replace("of oracle/", "").replace("with oracle/", ""), f
