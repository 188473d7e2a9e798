"""CPU checks of the boundary: liblt.so builds for sm_100a, loads without a GPU, exports
every symbol include/lt.h declares, and fails loudly (no CPU fallback) without a device."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2306_06744_b200 import build as B
    from paper_2306_06744_b200 import lt
    B.build()
    return lt.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "lt.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lt_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_exported(lib):
    from paper_2306_06744_b200 import lt
    names = declared_symbols()
    assert len(names) >= 25
    for n in names:
        assert hasattr(lib, n), "liblt.so does not export %s" % n
    # the binding declares a signature for every exported entry point and nothing else
    assert sorted(lt.SIGNATURES) == names


def test_strerror_and_version(lib):
    assert lib.lt_version() >= 100
    assert lib.lt_strerror(0) == b"ok"
    for code in range(-7, 0):
        assert lib.lt_strerror(code) not in (b"ok", b"unknown status")
    assert lib.lt_strerror(-99) == b"unknown status"


def test_no_cpu_fallback(lib):
    """Without a CUDA device the product path must fail loudly, not compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    h = C.c_void_p()
    rc = lib.lt_build(2, 1, 3, None, None, None, C.byref(h))
    assert rc in (-2, -3) and not h.value
    # argument errors are reported before any device work
    assert lib.lt_build(5, 1, 3, None, None, None, C.byref(h)) == -1


def test_product_does_not_import_oracle():
    """The product shares no code with the oracle (tier rule 3)."""
    pkg = os.path.join(ROOT, "paper_2306_06744_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", txt, flags=re.M), f
                assert "lto.cpp" not in txt and "liblto" not in txt, f
    orc = open(os.path.join(ROOT, "oracle", "lto.cpp")).read()
    assert "lt.h" not in orc.replace("include/lt.h)", "") or "#include \"lt.h\"" not in orc
    assert "#include \"../include" not in orc and "csrc" not in orc.replace("paper_2306_06744_b200/csrc", "")
