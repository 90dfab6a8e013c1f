"""CPU-only checks of the C-ABI boundary: the library builds, loads, and exports every symbol tm.h declares."""
import ctypes
import os
import re

import paper_1311_4462_b200 as tm
from paper_1311_4462_b200 import build as tm_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "tm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tm_[a-z_0-9]+)\s*\(", text)))


def test_library_builds_and_exports_every_declared_symbol():
    path = tm_build.build()
    assert os.path.exists(path)
    L = ctypes.CDLL(path)
    syms = declared_symbols()
    assert len(syms) >= 20
    for s in syms:
        assert hasattr(L, s), "libtm_b200.so does not export %s" % s
    assert sorted(tm.EXPORTS) == syms


def test_binding_uses_the_same_names_and_enum_values():
    text = open(os.path.join(ROOT, "include", "tm.h")).read()
    for name, val in re.findall(r"\b(TM_[A-Z_0-9]+)\s*=\s*(-?\d+)", text):
        assert getattr(tm, name) == int(val), name
    for s in tm.EXPORTS:
        if s != "tm_last_error" and s != "tm_field_device_ptr":
            assert callable(getattr(tm, s)), s


def test_argument_errors_need_no_gpu():
    """Validation that happens before any CUDA call."""
    L = tm.lib()
    h = ctypes.c_void_p()
    bad = (ctypes.c_int * 4)(4, 4, 5, 8)
    assert L.tm_init(bad, 0, ctypes.byref(h)) == tm.TM_ERR_DIMS
    assert b"even" in L.tm_last_error()
    small = (ctypes.c_int * 4)(2, 4, 4, 8)
    assert L.tm_init(small, 0, ctypes.byref(h)) == tm.TM_ERR_DIMS
    assert L.tm_init(None, 0, ctypes.byref(h)) == tm.TM_ERR_ARG
    assert L.tm_field_bytes(None, tm.TM_DOUBLE, 1) == 0
    assert L.tm_sync(None) == tm.TM_ERR_ARG


def test_product_path_does_not_import_the_oracle():
    """The CUDA path and its binding never touch oracle/ (or _work/)."""
    pkg = os.path.join(ROOT, "paper_1311_4462_b200")
    for dirpath, _, files in os.walk(pkg):
        if "build" in os.path.relpath(dirpath, pkg).split(os.sep)[-1:] and dirpath.endswith("csrc/build"):
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU fallback", ""), f
                assert "_work/" not in src, f


def test_header_is_plain_c(tmp_path):
    """include/tm.h is a C boundary: it compiles as C99 with no C++ or CUDA types in the signatures."""
    import subprocess
    src = tmp_path / "hdr.c"
    src.write_text('#include "tm.h"\nint main(void) { return TM_OK + TM_RECON_8 + TM_BASIS_CHIRAL; }\n')
    r = subprocess.run(["gcc", "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-I", os.path.join(ROOT, "include"),
                        "-c", str(src), "-o", str(tmp_path / "hdr.o")], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
