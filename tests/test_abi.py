"""Host-side checks of the C-ABI boundary (no GPU needed): the library loads, exports every symbol
include/qnep.h declares, and fails loudly -- never silently falls back -- when there is no CUDA device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2601_19034_b200 as Q
import qnep_inputs as I

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2601_19034_b200 import build
    build.build()
    return Q.load_library()


def test_header_symbols_are_exported(lib):
    header = open(os.path.join(ROOT, "include", "qnep.h")).read()
    declared = set(re.findall(r"\b(qnep_[a-z_]+)\s*\(", header))
    assert declared == set(Q.ABI_SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name


def test_abi_version_matches_header(lib):
    header = open(os.path.join(ROOT, "include", "qnep.h")).read()
    (v,) = re.findall(r"#define QNEP_ABI_VERSION (\d+)", header)
    assert int(v) == Q.ABI_VERSION == lib.qnep_abi_version()


def test_struct_layout_matches_header():
    # the ctypes mirrors must have the C layout (8-byte aligned doubles)
    assert C.sizeof(Q.qnep_model_desc) == 80          # 72 bytes of round 1 + l_max_4b, l_max_5b
    assert C.sizeof(Q.qnep_es_desc) == 40
    assert Q.qnep_model_desc.rc_r.offset == 32 and Q.qnep_model_desc.sqrt_eps_inf.offset == 56
    assert Q.qnep_model_desc.l_max_4b.offset == 72 and Q.qnep_model_desc.l_max_5b.offset == 76
    assert Q.qnep_es_desc.alpha.offset == 8 and Q.qnep_es_desc.grid.offset == 20


def test_product_does_not_import_oracle():
    """The oracle is test infrastructure: nothing under the product package or the input generators names it."""
    for base in ("paper_2601_19034_b200", "qnep_inputs"):
        for dirpath, _, files in os.walk(os.path.join(ROOT, base)):
            for f in files:
                if f.endswith((".py", ".cu", ".cuh", ".h")):
                    text = open(os.path.join(dirpath, f)).read()
                    for line in text.splitlines():
                        s = line.strip()
                        if s.startswith(("import ", "from ", "#include")):
                            assert "oracle" not in s, (f, s)


def test_invalid_arguments_are_rejected(lib):
    w = I.config0()
    m, e = Q._model_struct(w.model), Q._es_struct(w.es)
    h = C.c_void_p()
    p = np.ascontiguousarray(w.params, dtype=np.float32)
    assert lib.qnep_create(None, p.ctypes.data_as(C.c_void_p), p.shape[0], C.byref(e), C.byref(h)) == Q.QNEP_ERR_INVALID_ARG
    assert lib.qnep_create(C.byref(m), p.ctypes.data_as(C.c_void_p), p.shape[0] - 1, C.byref(e), C.byref(h)) == Q.QNEP_ERR_INVALID_ARG
    assert b"n_params" in lib.qnep_last_error(None)
    m.l_max = 6
    assert lib.qnep_create(C.byref(m), p.ctypes.data_as(C.c_void_p), p.shape[0], C.byref(e), C.byref(h)) in (
        Q.QNEP_ERR_UNSUPPORTED, Q.QNEP_ERR_INVALID_ARG)
    m = Q._model_struct(w.model)
    e.method = 2
    e.grid[0] = 48
    assert lib.qnep_create(C.byref(m), p.ctypes.data_as(C.c_void_p), p.shape[0], C.byref(e), C.byref(h)) == Q.QNEP_ERR_UNSUPPORTED


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(Q.QnepError) as ei:
        Q.from_workload(I.config0())
    assert ei.value.code == Q.QNEP_ERR_CUDA
