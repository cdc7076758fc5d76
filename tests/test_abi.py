"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/stroke_expand.h declares, and the record / style layouts are the documented sizes.  No compute calls."""
import ctypes as C
import os
import re
import shutil

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "stroke_expand.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sx_[a-z_]+|stroke_expand[a-z_]*)\s*\(", src)) - {"sx_alloc_fn"})


@pytest.fixture(scope="module")
def so_path():
    from paper_2405_00127_b200 import build
    if shutil.which("nvcc") is None and not os.path.exists("/usr/local/cuda/bin/nvcc"):
        if not os.path.exists(build.SO):
            pytest.skip("no nvcc and no prebuilt library")
        return build.SO
    return build.build()


def test_header_declares_the_north_star_calls():
    names = _declared()
    for need in ("sx_create", "sx_destroy", "sx_count", "sx_write", "stroke_expand", "stroke_expand_host"):
        assert need in names


def test_library_exports_every_declared_symbol(so_path):
    L = C.CDLL(so_path)
    for name in _declared():
        assert hasattr(L, name), name


def test_binding_lists_the_same_names(so_path):
    from paper_2405_00127_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()
    L = binding.lib()
    assert binding.sx_strerror(0) == "ok" and "capacity" in binding.sx_strerror(binding.SX_E_CAPACITY)
    for name in binding.EXPORTS:
        assert callable(getattr(binding, name)) and hasattr(L, name)


def test_record_and_style_layouts():
    from paper_2405_00127_b200 import binding, scenes
    assert scenes.STYLE_DTYPE.itemsize == 16
    assert binding.ARC_DTYPE.itemsize == 32 and binding.RECORD_BYTES == {0: 16, 1: 32, 2: 16}
    src = open(HEADER).read()
    assert "sx_line; /* SX_MODE_LINE: 16 bytes" in src and "sx_arc; /* SX_MODE_ARC: 32 bytes" in src


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2405_00127_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "stroke_oracle" not in txt, f
