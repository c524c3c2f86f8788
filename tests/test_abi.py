"""The C-ABI library loads and exports every symbol include/nf.h declares (no compute calls:
this runs without a GPU)."""
import ctypes
import os
import re

from paper_1810_02916_b200 import build, nf

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "nf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nf_[a-z_0-9]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    path = build.build()
    lib = ctypes.CDLL(path)
    declared = _declared_symbols()
    assert len(declared) >= 10
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/nf.h but not exported by libnf.so"
    assert sorted(nf.EXPORTS) == declared


def test_host_only_calls():
    lib = nf.load_library(build.build())
    assert lib.nf_version() >= 100
    assert abs(lib.nf_spline_equivalent_eps(1.0) - 2.16) < 1e-6
    assert lib.nf_last_error(None) == b"nf: null context"
    assert lib.nf_destroy(None) == nf.NF_OK


def test_no_cpu_fallback_without_gpu():
    import pytest
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError):
        nf.Context()
