"""CPU checks of the boundary: libao.so builds, loads, exports every symbol include/ao.h declares,
and fails loudly (no CPU fallback) when there is no CUDA device.  No compute call is made."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1608_00386_b200 import binding, build as ao_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    ao_build.build()
    return binding.load_library()


def test_every_declared_symbol_is_exported(lib):
    header = open(os.path.join(ROOT, "include", "ao.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(ao_[a-z_0-9]+)\s*\(", header))
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None


def test_no_torch_types_in_signatures():
    header = open(os.path.join(ROOT, "include", "ao.h")).read()
    assert "torch" not in header.replace("torch tensors", "") and "at::" not in header


def test_null_and_bad_arguments_are_reported(lib):
    assert lib.ao_last_error() is not None
    h = C.c_void_p()
    rc = lib.ao_geometry_create(None, None, 0, None, 0, None, 0, 5e-7, 0, C.byref(h))
    assert rc == 1 and h.value is None and b"NULL" in lib.ao_last_error()
    a = np.ones((8, 8), np.float32)
    p = binding.ao_pupil(8, 0.1, a.ctypes.data_as(C.POINTER(C.c_float)))
    bad = binding.ao_wfs(2, 4, 6, 4, 2, 0.5, a.ctypes.data_as(C.POINTER(C.c_float)))     # bin*n_pix > fft
    rc = lib.ao_geometry_create(C.byref(p), C.byref(bad), 1, None, 0, None, 0, 5e-7, 0, C.byref(h))
    assert rc == 2
    big = binding.ao_wfs(1, 8, 96, 8, 12, 0.5, a.ctypes.data_as(C.POINTER(C.c_float)))   # fft > 64 not pow2
    rc = lib.ao_geometry_create(C.byref(p), C.byref(big), 1, None, 0, None, 0, 5e-7, 0, C.byref(h))
    assert rc == 3
    rc = lib.ao_geometry_create(C.byref(p), None, 0, None, 0, None, 0, 5e-7, 100, C.byref(h))   # psf_fft not pow2
    assert rc == 3
    assert lib.ao_geometry_destroy(None) == 0
    assert lib.ao_workspace_bytes(None, 4) == 0
    assert lib.ao_phase_offset(None, 0, 0) == C.c_size_t(-1).value
    assert lib.ao_trace_layers(None, 0, 1, 2e-3, None, None) == 1


def test_fails_loudly_without_a_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    a = np.ones((8, 8), np.float32)
    p = binding.ao_pupil(8, 0.1, a.ctypes.data_as(C.POINTER(C.c_float)))
    h = C.c_void_p()
    rc = lib.ao_geometry_create(C.byref(p), None, 0, None, 0, None, 0, 5e-7, 0, C.byref(h))
    assert rc == 4 and h.value is None            # AO_ERR_CUDA, never a silent CPU path
    from paper_1608_00386_b200 import inputs
    with pytest.raises(RuntimeError):
        binding.Geometry(inputs.make_config(0))


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1608_00386_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "ao_oracle" not in src, f
    orc = open(os.path.join(ROOT, "oracle", "ao_oracle.c")).read()
    assert '#include "ao' not in orc and "csrc" not in orc.split("*/")[1]
