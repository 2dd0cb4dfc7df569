"""CPU-only checks of the boundary: the shared library builds, loads, and exports every symbol the header
declares; without a GPU every entry point that needs one fails loudly (no CPU fallback)."""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "frb200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fr_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_loads_and_exports_header_symbols():
    from paper_1409_0405_b200 import binding, build
    build.build()
    lib = binding.load()
    decl = _declared()
    assert len(decl) >= 15
    for name in decl:
        assert hasattr(lib, name), "libfrb200.so does not export %s" % name
    assert sorted(binding.SYMBOLS) == decl


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from fr_inputs import cases
    from paper_1409_0405_b200 import Context, FrError, binding
    with pytest.raises(FrError) as ei:
        Context(cases.config1())
    assert ei.value.status == binding.FR_ECUDA
    with pytest.raises(FrError):
        binding.gemm(np.eye(3), 0, 16, 0, 16, 16)
    with pytest.raises(FrError):
        binding.probe_peaks()


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1409_0405_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("no CPU fallback", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_1409_0405_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "`paper_1409_0405_b200/`", "")
