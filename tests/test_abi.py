"""The C-ABI library builds for sm_100a, loads without a GPU, and exports every symbol include/spray.h declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2604_20124_b200 import build
    path = build.build()
    return ctypes.CDLL(str(path))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "spray.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(spray_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    names = declared_symbols()
    assert len(names) >= 14
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/spray.h but not exported"


def test_binding_lists_the_same_symbols():
    import paper_2604_20124_b200 as P
    assert sorted(P.EXPORTS) == declared_symbols()
    P.load()


def test_version_string(lib):
    lib.spray_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.spray_version()


def test_no_cpu_fallback_without_gpu():
    import torch
    import paper_2604_20124_b200 as P
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(P.SprayError):
        P.Spray(16, 8)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2604_20124_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "spray_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2604_20124_b200" not in txt and "libspray_b200" not in txt
