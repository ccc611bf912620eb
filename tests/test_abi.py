"""-m "not gpu": the C-ABI library loads and exports every symbol include/pivot_iv.h declares; argument validation
(which needs no GPU) returns the documented error codes; the Python binding refuses to run without a CUDA device."""
import ctypes
import os
import re

import pytest
import torch

import paper_2606_17065_b200 as pv
from paper_2606_17065_b200 import build as pbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    pbuild.build()
    return pv.load_library()


def _declared():
    text = open(os.path.join(ROOT, "include", "pivot_iv.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pivot_iv_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert len(names) >= 12
    assert sorted(pv.EXPORTS) == names
    for n in names:
        assert getattr(lib, n) is not None


def test_version_and_strerror(lib):
    assert pv.pivot_iv_version() == 100
    for code in range(0, -9, -1):
        assert "unknown" not in pv.pivot_iv_strerror(code)
    assert "unknown" in pv.pivot_iv_strerror(-99)


def test_argument_validation_without_gpu(lib):
    i64 = ctypes.c_int64
    assert lib.pivot_iv_forward(None, i64(4), None, None, None, None) == -1          # NULL inputs struct
    from paper_2606_17065_b200.binding import _Inputs
    inp = _Inputs(8, 8, 8, 8, None, 8, 8)
    assert lib.pivot_iv_forward(ctypes.byref(inp), i64(4), 8, 8, 8, None) == -5      # mixed r/q
    inp = _Inputs(8, 8, 8, None, None, 8, 8)
    assert lib.pivot_iv_forward(ctypes.byref(inp), i64(-1), 8, 8, 8, None) == -2     # n < 0
    assert lib.pivot_iv_forward(ctypes.byref(inp), i64(0), None, None, None, None) == 0   # n == 0 no-op
    assert lib.pivot_iv_forward(ctypes.byref(inp), i64(4), None, 8, 8, None) == -1
    assert lib.pivot_iv_backward(8, 8, 8, ctypes.c_double(1e-8), 3, i64(4), 8, None) == -3    # modes are 0, 1, 2
    assert lib.pivot_iv_backward(8, 8, 8, ctypes.c_double(1e-8), -1, i64(4), 8, None) == -3
    assert lib.pivot_iv_backward_inputs(ctypes.byref(inp), 8, 8, 8, 8, ctypes.c_double(1e-8), 7, i64(4), 8, 8, 8, 8, None, None, None) == -3
    assert lib.pivot_iv_backward_inputs(ctypes.byref(inp), 8, 8, 8, 8, ctypes.c_double(1e-8), 0, i64(4), 8, None, 8, 8, None, None, None) == -1
    assert lib.pivot_iv_black_price(ctypes.byref(inp), None, i64(4), 8, None, None) == -1
    assert lib.pivot_iv_black_price(ctypes.byref(inp), 8, i64(0), 8, None, None) == 0
    assert lib.pivot_iv_backward(8, 8, 8, ctypes.c_double(-1.0), 0, i64(4), 8, None) == -4
    assert lib.pivot_iv_backward(8, 8, 8, ctypes.c_double(float("nan")), 0, i64(4), 8, None) == -4
    assert lib.pivot_iv_backward(None, 8, 8, ctypes.c_double(0.0), 0, i64(4), 8, None) == -1
    assert lib.pivot_iv_backward(None, None, None, ctypes.c_double(0.0), 1, i64(0), None, None) == 0
    assert lib.pivot_iv_pipeline_create(None, 0, i64(16), 2) == -1
    h = ctypes.c_void_p()
    assert lib.pivot_iv_pipeline_create(ctypes.byref(h), 0, i64(0), 2) == -7
    assert lib.pivot_iv_pipeline_create(ctypes.byref(h), 0, i64(16), 9) == -7
    assert lib.pivot_iv_pipeline_destroy(None) == 0
    assert lib.pivot_iv_pipeline_set_host_access(None, 0) == -1
    assert lib.pivot_iv_status_histogram(8, i64(-1), 8, None) == -2
    assert lib.pivot_iv_status_histogram(8, i64(4), None, None) == -1
    assert lib.pivot_iv_status_histogram(None, i64(4), 8, None) == -1
    assert lib.pivot_iv_status_histogram(None, i64(0), 8, None) == 0
    assert lib.pivot_iv_pipeline_last_host_path(None) == -1
    assert lib.pivot_iv_pipeline_set_forward_kernel(None, 0) == -1


def test_binding_constants_are_the_header_defines():
    """Every numeric #define of include/pivot_iv.h that the binding mirrors carries the same value there."""
    text = open(os.path.join(ROOT, "include", "pivot_iv.h")).read()
    defs = {m.group(1): int(m.group(2)) for m in re.finditer(r"#define\s+PIVOT_([A-Z0-9_]+)\s+\(?(-?\d+)\)?", text)}
    mirrored = {"GATE_MASK": pv.GATE_MASK, "GATE_ATTENUATE": pv.GATE_ATTENUATE, "GATE_STRICT": pv.GATE_STRICT,
                "RT_GATED": pv.RT_GATED, "RT_NAIVE": pv.RT_NAIVE, "FWD_AUTO": pv.FWD_AUTO, "FWD_COMPACT": pv.FWD_COMPACT,
                "FWD_ROWWISE": pv.FWD_ROWWISE, "FWD_FP64_ONLY": pv.FWD_FP64_ONLY, "HOST_AUTO": pv.HOST_AUTO,
                "HOST_STAGED": pv.HOST_STAGED, "HOST_DIRECT": pv.HOST_DIRECT, "STATIC_MAX_ROWS": pv.STATIC_MAX_ROWS}
    for name, value in mirrored.items():
        assert defs[name] == value, name


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_binding_fails_loudly_without_cuda():
    x = torch.ones(4, dtype=torch.float64)
    with pytest.raises(pv.PivotError):
        pv.pivot_iv_forward(x, x, x, x, x)
    with pytest.raises(pv.PivotError):
        pv.pivot_iv_backward(x, x, torch.zeros(4, dtype=torch.uint8), 1e-8, 0)
    with pytest.raises(pv.PivotError):
        pv.Pipeline()


def test_product_never_imports_oracle():
    """The product path may not route through the CPU oracle: no file of the package mentions it."""
    pkg = os.path.join(ROOT, "paper_2606_17065_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "pyoracle" not in src and "lbr_oracle" not in src and "import oracle" not in src, f
