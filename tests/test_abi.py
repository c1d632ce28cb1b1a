"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol
that include/sd_b200.h declares, and the Python binding declares the same set.  No compute
call is made (there is no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built():
    import __graft_entry__ as g
    g.build()
    from paper_1205_6333_b200 import sd
    return sd


def _declared_symbols():
    with open(os.path.join(ROOT, "include", "sd_b200.h")) as f:
        text = f.read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sd_[a-z_0-9]+)\s*\(", text)) - {"sd_force_fn"})


def test_header_declares_the_north_star_entry_points():
    names = _declared_symbols()
    for required in ("sd_create", "sd_mobility_apply", "sd_step", "sd_destroy"):
        assert required in names


def test_library_exports_every_declared_symbol(built):
    lib = ctypes.CDLL(built.LIB_PATH)
    for name in _declared_symbols():
        assert hasattr(lib, name), f"{name} declared in sd_b200.h but not exported"


def test_binding_covers_the_header(built):
    assert sorted(built.SYMBOLS) == _declared_symbols()
    built.load_library()


def test_no_cpu_fallback_without_a_device(built):
    """On a box without a GPU sd_create must fail loudly with SD_ERR_UNSUPPORTED."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(built.SdError) as ei:
        built.Context(16, 1.0, 1.0)
    assert ei.value.status == built.ERR_UNSUPPORTED
    assert "no CPU fallback" in str(ei.value)


def test_product_path_does_not_touch_the_oracle():
    """Nothing under paper_1205_6333_b200/ may import or link oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_1205_6333_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                with open(os.path.join(dirpath, fn)) as f:
                    src = f.read()
                for pat in (r"^\s*(from|import)\s+oracle", r"sd_oracle", r"libsd_oracle",
                            r"#include\s*[\"<][^\">]*oracle", r"sdo_"):
                    assert not re.search(pat, src, flags=re.M), (fn, pat)
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            with open(os.path.join(ROOT, "oracle", fn)) as f:
                src = f.read()
            assert "import paper_1205_6333_b200" not in src
            assert "from paper_1205_6333_b200" not in src
            assert "csrc" not in src.replace("paper_1205_6333_b200/csrc/", "")
