"""-m "not gpu": the C-ABI library builds, loads and exports every symbol include/vor.h declares;
argument validation that needs no device; the product never routes through the oracle."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1607_00908_b200 import build
    build.build()
    from paper_1607_00908_b200 import binding
    return binding.load_library()


def header_functions():
    src = open(os.path.join(ROOT, "include", "vor.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(?:int|int64_t|const char\*)\s+((?:vor|field|match)_\w+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    from paper_1607_00908_b200 import binding
    names = header_functions()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/vor.h but not exported"
        assert n in binding.SIGNATURES, f"{n} has no ctypes prototype in binding.py"
    assert sorted(binding.SIGNATURES) == names


def test_null_and_range_validation_without_device(lib):
    assert lib.vor_create(None, 64, 32, 0) == -1
    h = C.c_void_p()
    assert lib.vor_create(C.byref(h), 1, 32, 0) == -1          # L < 2
    assert lib.vor_create(C.byref(h), 64, 0, 0) == -1          # max_sites < 1
    assert lib.vor_destroy(None) == -1
    assert lib.vor_label(None, None, None) == -1
    assert lib.vor_last_error(None) == b"null context"


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1607_00908_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "vor_oracle" not in text and "liboracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_1607", text, flags=re.M), f
            assert not re.search(r"#\s*include\s*[<\"].*(csrc|vor\.h|\.cuh)", text), f


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    from paper_1607_00908_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.load_library()
