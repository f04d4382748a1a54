"""The C-ABI library loads on a box without a GPU and exports every symbol include/gcamb_los.h
declares; the binding names them all; no compute call is made here."""
import ctypes
import os
import re

from paper_2509_25110_b200 import build, los

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols(header, prefix):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(%s\w+)\s*\(" % prefix, text)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    lib_path = build.build_extension()
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == ["gcamb_los.h", "gcamb_probe.h"]
    # the product library: every symbol of gcamb_los.h, and nothing of the bench-only probe header
    lib = ctypes.CDLL(lib_path)
    names = declared_symbols("gcamb_los.h", "gcamb_los_")
    assert len(names) >= 10
    for name in names:
        assert hasattr(lib, name), f"{name} declared in gcamb_los.h but not exported"
    assert sorted(los.EXPORTS) == names
    # the probe library (bench.py's roofline denominators)
    probe = ctypes.CDLL(build.PROBE_LIB)
    probe_names = declared_symbols("gcamb_probe.h", "gcamb_probe_")
    assert sorted(los.PROBE_EXPORTS) == probe_names and len(probe_names) == 2
    for name in probe_names:
        assert hasattr(probe, name) and not hasattr(lib, name)


def test_errors_without_touching_the_gpu():
    lib = los.load_library()
    assert lib.gcamb_los_plan_info(None, None, None, None, None, None, None) == 1      # GCAMB_EINVAL
    assert b"null" in lib.gcamb_los_last_error()
    assert lib.gcamb_los_plan_destroy(None) == 0
