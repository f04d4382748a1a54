"""The C-ABI library loads on a box without a GPU and exports every symbol include/gcamb_los.h
declares; the binding names them all; no compute call is made here."""
import ctypes
import os
import re

from paper_2509_25110_b200 import build, los

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "gcamb_los.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gcamb_los_\w+)\s*\(", text)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    lib_path = build.build_extension()
    lib = ctypes.CDLL(lib_path)
    names = declared_symbols()
    assert len(names) >= 11
    for name in names:
        assert hasattr(lib, name), f"{name} declared in gcamb_los.h but not exported"
    assert sorted(los.EXPORTS) == names


def test_errors_without_touching_the_gpu():
    lib = los.load_library()
    assert lib.gcamb_los_plan_info(None, None, None, None, None, None, None) == 1      # GCAMB_EINVAL
    assert b"null" in lib.gcamb_los_last_error()
    assert lib.gcamb_los_plan_destroy(None) == 0
