"""The checked build (liblt_debug.so, -DLT_DEBUG): device-side assertions on every located index, table
write position, ticket and look-back word stand in for compute-sanitizer, which is closed on the GPU
pool this library is developed on.  The cases run in a subprocess so that a trap
cannot poison this process's CUDA context."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_checked_build_exports_the_same_symbols():
    import ctypes as C
    from paper_2306_06744_b200 import build as B
    from paper_2306_06744_b200 import lt
    L = C.CDLL(B.build(debug=True))
    for name in lt.SIGNATURES:
        assert hasattr(L, name), name
    L.lt_debug_build.restype = C.c_int
    assert L.lt_debug_build() == 1 and lt.lib().lt_debug_build() == int(os.environ.get("LT_DEBUG_LIB") == "1")
    # the assertion texts are in the binary (the checks were not compiled out)
    blob = open(B.LIB_DEBUG, "rb").read()
    for text in (b"keys[lo] <= bound", b"(v >> 62) <= 2", b"p_conf >= 0"):
        assert text in blob, text


@pytest.mark.gpu
def test_small_cases_through_the_checked_build():
    from paper_2306_06744_b200 import build as B
    B.build(debug=True)
    env = dict(os.environ, LT_DEBUG_LIB="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "debug_build_cases.py")], env=env,
                       capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, "checked build failed:\n" + r.stdout[-2000:] + "\n" + r.stderr[-4000:]
    assert "debug build cases ok" in r.stdout and "Assertion" not in r.stderr
