"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol include/snk.h declares
(no compute calls: there is no GPU here)."""
import ctypes
import os
import re

import pytest

from paper_2303_14280_b200 import build as snk_build
from paper_2303_14280_b200 import snk


@pytest.fixture(scope="module")
def lib_path():
    return snk_build.build()


def _declared_symbols():
    txt = open(snk.HEADER_PATH).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(snk_[a-z0-9_A-Z]+)\s*\(", txt)))


def test_header_symbols_are_exported(lib_path):
    lib = ctypes.CDLL(lib_path)
    names = _declared_symbols()
    assert "snk_create" in names and "snk_set_grid" in names and "snk_build_K" in names
    for n in names:
        assert hasattr(lib, n), "libsnk.so does not export %s" % n
    assert set(names) == set(snk.EXPORTS)


def test_binding_loads_and_reports_version(lib_path):
    lib = snk.load()
    assert snk.version().startswith("snk ")
    assert ctypes.sizeof(snk.SnkStats) == 9 * 8 + 13 * 8 + 30 * 8 + 8 + 8      # sizeof(snk_stats) of include/snk.h


def test_product_never_imports_oracle():
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    pk = os.path.join(root, "paper_2303_14280_b200")
    for dp, _, fs in os.walk(pk):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                t = open(os.path.join(dp, f)).read()
                assert "import oracle" not in t and "from oracle" not in t and "snk_oracle" not in t, f
    # and the oracle does not touch the CUDA path
    for f in os.listdir(os.path.join(root, "oracle")):
        if f.endswith((".py", ".cpp")):
            t = open(os.path.join(root, "oracle", f)).read()
            assert "libsnk" not in t and "csrc" not in t.replace("paper_2303_14280_b200/csrc", "") or f == "oracle.py"
            assert "import snk" not in t and "from paper_2303_14280_b200 import snk" not in t
