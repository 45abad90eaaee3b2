"""CPU-side checks of the boundary: libhb.so builds for sm_100a, loads, and exports
exactly the symbols include/hb.h declares.  No compute call is made (no GPU here)."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1308_5587_b200 import build
    return build.build()


def _declared():
    text = open(os.path.join(ROOT, "include", "hb.h")).read()
    return sorted(set(re.findall(r"^HB_API[^;(]*?\b(hb_\w+)\s*\(", text, flags=re.M)))


def test_header_declares_the_calls_the_north_star_lists():
    names = _declared()
    for required in ("hb_create", "hb_build_cells", "hb_build_nlist", "hb_compute_lj", "hb_step_nve", "hb_sort"):
        assert required in names
    assert len(names) == 35


def test_library_exports_every_declared_symbol(libpath):
    lib = ctypes.CDLL(libpath)
    for name in _declared():
        assert hasattr(lib, name), f"{name} declared in hb.h but not exported"
    out = subprocess.check_output(["nm", "-D", "--defined-only", libpath], text=True)
    exported = sorted(ln.split()[-1] for ln in out.splitlines() if " T " in ln)
    assert exported == _declared(), "exports and header differ"
    lib.hb_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.hb_version()


def test_binding_names_match_header(libpath):
    from paper_1308_5587_b200 import hb
    assert sorted(hb.EXPORTS) == _declared()
    for name in _declared():
        short = name[3:]
        if short in ("create", "destroy", "last_error", "version"):
            continue
        assert hasattr(hb.System, short), f"binding lacks System.{short}"


def test_library_is_sm100a_sass_only(libpath):
    out = subprocess.check_output(["cuobjdump", "-lelf", libpath], text=True)
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_null_handle_is_rejected_without_a_gpu(libpath):
    lib = ctypes.CDLL(libpath)
    lib.hb_build_cells.argtypes = [ctypes.c_void_p]
    assert lib.hb_build_cells(None) == -1          # HB_EINVAL
    lib.hb_last_error.restype = ctypes.c_char_p
    lib.hb_last_error.argtypes = [ctypes.c_void_p]
    assert lib.hb_last_error(None) == b"null handle"


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1308_5587_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.replace("the oracle", "").replace("The oracle", "") or f == "workloads.py", f
                assert "orc_" not in text and "liborc" not in text, f
