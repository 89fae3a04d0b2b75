"""CPU: the C-ABI library builds for sm_100a, loads, and exports every symbol include/lbm.h declares
(no compute calls -- there is no GPU here); host-side logic that needs no device."""
import os
import re

import pytest

import paper_2112_08926_b200 as lbm
from paper_2112_08926_b200 import build as lbm_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def library():
    lbm_build.build()
    return lbm.lib()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "lbm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lbm_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported_and_bound(library):
    names = _declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(library, n), n
        assert n in lbm.SYMBOLS, f"{n} is declared in lbm.h but not bound in the Python module"
    assert sorted(lbm.SYMBOLS) == names


def test_size_helpers_need_no_device(library):
    assert lbm.bytes_per_cell(19, "FP32") == 2 * 19 * 4 + 1
    assert lbm.bytes_per_cell(19, "FP16C") == 2 * 19 * 2 + 1
    assert lbm.bytes_per_cell(27, "P16_1S") == 109
    assert lbm.bytes_per_cell(5, "FP32") == -1
    assert lbm.bytes_per_cell(19, "FP64") == 305 and lbm.bytes_per_cell(19, "FP64_FP32") == 153
    assert lbm.ddf_buffer_bytes(8, 8, 4, 27, "FP64") == 8 * 8 * 4 * 27 * 8
    assert lbm.ddf_buffer_bytes(3, 3, 3, 19, "FP32") % 256 == 0
    assert lbm.launch_count() == 0


def test_product_does_not_touch_the_oracle():
    """The oracle is test infrastructure: nothing under the package may import or link it."""
    pkg = os.path.join(ROOT, "paper_2112_08926_b200")
    for dirpath, _, files in os.walk(pkg):
        if os.path.basename(dirpath) == "build":
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "liblbm_oracle" not in src, f
                assert "oracle.h" not in src, f


def test_sass_is_sm100a(library):
    """the shipped library carries sm_100a code (and only that)"""
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", lbm.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert not re.search(r"sm_(?!100a)\d+", out)
