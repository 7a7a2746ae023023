"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/blipgpu.h declares; the binding declares the same set; without a GPU the product path
fails loudly (no CPU fallback); the product package never touches oracle/."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_1204_1121_b200 as blip

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols(header=None):
    """Function names declared in include/*.h (comments stripped)."""
    names = set()
    for h in sorted(os.listdir(os.path.join(ROOT, "include"))):
        if not h.endswith(".h") or (header and h != header):
            continue
        text = open(os.path.join(ROOT, "include", h)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names |= set(re.findall(r"\b(blipgpu_[a-z0-9_]+)\s*\(", text))
    return sorted(names)


def test_header_symbols_are_exported_and_bound():
    names = declared_symbols()
    assert {"blipgpu_create", "blipgpu_eval", "blipgpu_eval_host", "blipgpu_destroy",
            "blipgpu_reserve", "blipgpu_strerror"} <= set(names)
    L = blip.lib()
    for n in names:
        assert hasattr(L, n), f"{n} declared in blipgpu.h but not exported"
    assert sorted(blip.SIGNATURES) == names
    # the boundary proper carries no test / benchmark instrumentation
    boundary = set(declared_symbols("blipgpu.h"))
    assert not boundary & {"blipgpu_set_tuning", "blipgpu_probe_fp32", "blipgpu_set_profiling",
                           "blipgpu_last_kernel_ms", "blipgpu_launch_count", "blipgpu_last_path"}


def test_library_reads_no_environment_knobs():
    for f in os.listdir(os.path.join(ROOT, "paper_1204_1121_b200", "csrc")):
        assert "getenv" not in open(os.path.join(ROOT, "paper_1204_1121_b200", "csrc", f)).read(), f


def test_strerror_is_total():
    L = blip.lib()
    for code in (0, -1, -2, -3, -4, 17):
        assert len(L.blipgpu_strerror(code)) > 0


def test_destroy_null_is_ok_and_null_handles_are_rejected():
    L = blip.lib()
    assert L.blipgpu_destroy(None) == blip.OK
    assert L.blipgpu_reserve(None, 10) == blip.EINVAL
    assert L.blipgpu_eval(None, None, 1, 1, None, None, None, 4, None, None) == blip.EINVAL
    assert L.blipgpu_launch_count(None) == 0


def test_create_argument_validation_needs_no_gpu():
    L = blip.lib()
    A = np.eye(3).reshape(9) * 10.0
    c = np.zeros((4, 4, 4, 2), dtype=np.float32)
    out = ctypes.c_void_p(0)

    def create(lat, grid, norb):
        lat = np.ascontiguousarray(lat, dtype=np.float64)
        g = np.ascontiguousarray(grid, dtype=np.int32)
        return L.blipgpu_create(lat.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                g.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), norb,
                                ctypes.c_void_p(c.ctypes.data), 0, None, ctypes.byref(out))

    assert create(A, (3, 4, 4), 2) == blip.EINVAL           # n_a < 4
    assert create(A, (4, 4, 4), 0) == blip.EINVAL           # L < 1
    bad = A.copy(); bad[0] = np.nan
    assert create(bad, (4, 4, 4), 2) == blip.EINVAL
    assert create(A, (2048, 2048, 2048), 2) == blip.EINVAL  # >= 2^31 grid points
    assert out.value is None


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    c = np.zeros((4, 4, 4, 2), dtype=np.float32)
    with pytest.raises(Exception):
        blip.blipgpu_create(np.eye(3) * 10.0, (4, 4, 4), 2, c)


def test_product_path_does_not_reference_the_oracle():
    pkg = os.path.join(ROOT, "paper_1204_1121_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "blip_oracle" not in text, f
