"""CPU-only: the C-ABI library builds, loads, and exports every symbol include/lqcd.h declares
(no compute calls without a GPU; there is no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "lqcd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lqcd_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_north_star_entry_points():
    syms = declared_symbols()
    for name in ("lqcd_geom_create", "lqcd_clover_build", "lqcd_dw_apply", "lqcd_dwdag_apply", "lqcd_cg_solve"):
        assert name in syms


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2503_16994_b200 import binding, build

    build.build()
    lib = ctypes.CDLL(binding.LIB_PATH)
    syms = declared_symbols()
    assert len(syms) >= 20
    for name in syms:
        assert hasattr(lib, name), name
    assert sorted(binding.EXPORTS) == syms


def test_no_cpu_fallback_without_device():
    """Without a CUDA device geometry creation must fail loudly with LQCD_ECUDA."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2503_16994_b200 import binding as B

    with pytest.raises(B.LqcdError) as e:
        B.geom_create((4, 4, 4, 4))
    assert e.value.status == B.ECUDA
    assert B.field_bytes(None, B.FIELD_SPINOR) == 0


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2503_16994_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "oracle/" not in text and "liblqcd_oracle" not in text, f
