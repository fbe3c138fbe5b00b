"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/ppm.h declares; argument validation that needs no device; no-fallback behaviour."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2510_07764_b200 as ppm
from paper_2510_07764_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _header_symbols():
    txt = open(os.path.join(ROOT, "include", "ppm.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(ppm_[a-z0-9_]+)\s*\(", txt)))


def test_library_builds_and_exports_every_declared_symbol():
    lib = ppm.load_library()
    names = _header_symbols()
    assert "ppm_create" in names and "ppm_evaluate" in names and "ppm_fold_response" in names
    assert "ppm_loglike" in names and "ppm_load_atmosphere" in names
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTS) == names       # the binding covers exactly the header


def test_config_struct_matches_header():
    txt = open(os.path.join(ROOT, "include", "ppm.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} ppm_config;", txt, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = re.findall(r"int32_t\s+([a-z_, ]+);", body)
    flat = [f.strip() for grp in fields for f in grp.split(",")]
    assert flat == [n for n, _ in binding._Config._fields_]


def test_argument_validation_without_device():
    lib = ppm.load_library()
    h = C.c_void_p()
    e = np.array([1.0, 2.0])
    cfg = binding._Config(0, 4, 4, 4, 0, 2, 0, 0, 1, 1, 0)        # n_spots = 0
    assert lib.ppm_create(C.byref(cfg), e.ctypes.data_as(binding._dp), None, C.byref(h)) == -1
    assert b"n_spots" in lib.ppm_last_error()
    cfg = binding._Config(1, 4, 4, 4, 0, 2, 0, 0, 1, 1, 0)
    bad = np.array([2.0, 1.0])
    assert lib.ppm_create(C.byref(cfg), bad.ctypes.data_as(binding._dp), None, C.byref(h)) == -1
    cfg = binding._Config(1, 4, 4, 4, 0, 2, 0, 1, 1, 1, 0)        # precision = 1 not implemented
    assert lib.ppm_create(C.byref(cfg), e.ctypes.data_as(binding._dp), None, C.byref(h)) == -1


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("device present")
    with pytest.raises(ppm.PPMError):
        ppm.PPM(dict(n_spots=1, n_theta=4, n_phi=4, n_phase=4, emission=0, oblate=0), [1.0, 2.0])
    lib = ppm.load_library()
    h = C.c_void_p()
    e = np.array([1.0, 2.0])
    cfg = binding._Config(1, 4, 4, 4, 0, 2, 0, 0, 1, 1, 0)
    assert lib.ppm_create(C.byref(cfg), e.ctypes.data_as(binding._dp), None, C.byref(h)) == -3   # PPM_ERR_CUDA


def test_product_does_not_import_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2510_07764_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "ppm_oracle" not in src, f
