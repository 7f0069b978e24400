"""CPU checks of the boundary: libqsl.so loads and exports every function include/qsl.h declares; the binding refuses
to compute without a CUDA device (no CPU fallback); the oracle is not imported by the product."""
import ctypes
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions(header="qsl.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(qsl_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    import paper_1609_00724_b200 as qsl
    names = _declared_functions()
    assert {"qsl_field_create", "qsl_field_destroy", "qsl_trace", "qsl_fledge_dense", "qsl_fledge_sparse", "qsl_select",
            "qsl_refine", "qsl_strerror"} <= set(names)
    lib = ctypes.CDLL(qsl.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), n
    assert qsl.lib().qsl_compiled_arch() == 100
    assert qsl.lib().qsl_strerror(-1).decode() == "invalid argument"
    # every header under include/ belongs to one of the two libraries
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == ["qsl.h", "qsl_peaks.h"]


def test_peaks_library_is_separate_from_the_product_library():
    """The roofline-denominator micro-kernels of bench.py live in libqsl_peaks.so (include/qsl_peaks.h): every symbol that
    header declares is exported there, and libqsl.so exports none of them."""
    import paper_1609_00724_b200 as qsl
    names = _declared_functions("qsl_peaks.h")
    assert names == ["qsl_peak_fma", "qsl_peak_gather"]
    peaks, prod = ctypes.CDLL(qsl.PEAKS_LIB_PATH), ctypes.CDLL(qsl.LIB_PATH)
    for n in names:
        assert hasattr(peaks, n), n
        assert not hasattr(prod, n), n
    assert not any("peak" in n for n in _declared_functions())


def test_struct_layouts_match_header_sizes():
    """ctypes mirrors of the ABI structs: sizes as a C compiler lays them out (x86-64 SysV)."""
    from paper_1609_00724_b200 import binding as B
    assert ctypes.sizeof(B._GridDesc) == 4 * 4 + 6 * 8 + 3 * 8 + 5 * 4 + 4           # 5 trailing ints + tail padding
    assert ctypes.sizeof(B._TraceParams) == 48 + 8 + 8 + 8 + 8 + 8 + 8 + 8 + 8   # ... flags (+pad), tol
    assert ctypes.sizeof(B._TraceOut) == 12 * 8
    assert ctypes.sizeof(B._Lattice) == 8 + 24 + 4 * 24
    assert ctypes.sizeof(B._Levels) == 7 * 8


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback():
    import paper_1609_00724_b200 as qsl
    z = torch.zeros(8, dtype=torch.float64)
    with pytest.raises(qsl.QslError):
        qsl.qsl_field_create(2, 2, 2, z, z, z, lo=(0, 0, 0), hi=(1, 1, 1))
    with pytest.raises(qsl.QslError):
        qsl.qsl_fledge_dense(torch.zeros((4, 4), dtype=torch.float64), 2)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1609_00724_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower(), os.path.join(dirpath, f)      # no file of the product may mention it
