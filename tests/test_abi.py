"""The C-ABI library loads and exports every symbol include/lra.h declares; argument validation that needs
no GPU.  (No compute calls here: those are the -m gpu parity tests.)"""
import ctypes as C
import os
import re

import pytest

from paper_2508_17187_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "lra.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lra_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_are_exported():
    names = declared_functions()
    assert {"lra_plan_create", "lra_plan_destroy", "lra_bin", "lra_bin_export", "lra_grid", "lra_degrid",
            "lra_strerror"} <= set(names)
    lib = B.lib()
    for n in names:
        assert hasattr(lib, n), f"{n} declared in lra.h but not exported by liblra.so"
    assert set(B.EXPORTED) == set(names)


def test_binding_mirrors_the_c_names():
    for n in declared_functions():
        if n in ("lra_last_cuda_error",):
            continue
        assert callable(getattr(B, n)), n


def test_strerror_and_validation_without_gpu():
    lib = B.lib()
    assert B.lra_strerror(0) == "ok" and "invalid" in B.lra_strerror(1) and "order" in B.lra_strerror(4)
    h = C.c_void_p()
    assert lib.lra_plan_create(C.byref(h), None) == B.LRA_EINVAL and not h.value
    assert lib.lra_plan_create(None, None) == B.LRA_EINVAL
    import numpy as np
    sup = np.array([4], np.int32)   # even support: rejected before any CUDA call
    off = np.array([0], np.int64)
    dat = np.zeros(16, np.complex64)
    d = B.lra_plan_desc(64, 64, 1, 1, 1, 32, 0, 1.0, 1.0, 1, sup.ctypes.data, off.ctypes.data, dat.ctypes.data, 0, 0)
    assert lib.lra_plan_create(C.byref(h), C.byref(d)) == B.LRA_EINVAL
    d.ncorr = 5
    assert lib.lra_plan_create(C.byref(h), C.byref(d)) == B.LRA_EINVAL
    assert lib.lra_plan_destroy(None) == B.LRA_EINVAL
    assert lib.lra_grid(None, None, None, None, None, None) == B.LRA_EINVAL
    with pytest.raises(B.LraError):
        B.lra_plan_create(64, 64, 1, 1, 1, 1.0, 1.0, sup, off, dat)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2508_17187_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "lra_ref" not in txt and "from oracle" not in txt and "import oracle" not in txt, f
