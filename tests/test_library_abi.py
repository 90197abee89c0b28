"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol that
include/cpm.h declares, validates parameters before touching the device, and fails loudly
(CPM_ERR_CUDA) instead of falling back when no device is present."""
import ctypes as C

import numpy as np
import pytest


@pytest.fixture(scope="module")
def pk():
    import paper_2312_09317_b200 as m
    m.load_library()
    return m


def test_library_exports_every_declared_symbol(pk):
    L = pk.load_library()
    names = pk.exported_symbols()
    assert {"cpm_create", "cpm_destroy", "cpm_set_lattice", "cpm_step", "cpm_get_lattice", "cpm_get_cell_stats",
            "cpm_get_act", "cpm_set_act", "cpm_get_counters", "cpm_get_schedule", "cpm_last_error"} <= set(names)
    for n in names:
        assert hasattr(L, n), n


def _params(pk, **over):
    from paper_2312_09317_b200.binding import _Params
    p = _Params()
    J = np.array([[0, 1], [1, 1]], np.int32)
    p.ndim = 2; p.dims[0] = 32; p.dims[1] = 32; p.dims[2] = 1
    p.n_types = 2; p.J = J.ctypes.data_as(C.POINTER(C.c_int32)); p.T = 20.0; p.max_cells = 1
    for k, v in over.items():
        setattr(p, k, v)
    return p, J


def test_validation_happens_before_the_device_is_touched(pk):
    L = pk.load_library()
    h = C.c_void_p()
    p, keep = _params(pk, ndim=4)
    assert L.cpm_create(C.byref(p), C.byref(h)) == -2
    p, keep = _params(pk, T=-1.0)
    assert L.cpm_create(C.byref(p), C.byref(h)) == -1
    p, keep = _params(pk, subsection=5)
    assert L.cpm_create(C.byref(p), C.byref(h)) == -2
    p, keep = _params(pk, max_cells=1 << 24)
    assert L.cpm_create(C.byref(p), C.byref(h)) == -3
    p, keep = _params(pk, neighbourhood=1)
    assert L.cpm_create(C.byref(p), C.byref(h)) == -3
    assert L.cpm_create(None, C.byref(h)) == -1
    assert L.cpm_step(None, 1) == -1


def test_no_cpu_fallback(pk):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    L = pk.load_library()
    h = C.c_void_p()
    p, keep = _params(pk)
    assert L.cpm_create(C.byref(p), C.byref(h)) == -4      # CPM_ERR_CUDA
    with pytest.raises(pk.CPMError) as e:
        pk.CPM((32, 32), J=[[0, 1], [1, 1]], max_cells=1)
    assert e.value.code == -4


def test_product_does_not_import_the_oracle():
    import os
    import re
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    pkg = os.path.join(root, "paper_2312_09317_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, re.M), f
                assert "cpm_oracle" not in text and "liboracle" not in text, f
