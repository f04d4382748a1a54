"""Builds libgcamb_los.so (the product) and libgcamb_probe.so (bench.py's roofline probes, not part
of the method) in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2509_25110_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgcamb_los.so")
PROBE_LIB = os.path.join(HERE, "libgcamb_probe.so")
# (source, extra flags, object tag): transfer.cu is compiled once per (sparse, n_src) entry, in parallel
UNITS = [("api.cu", [], "api"), ("plan.cu", [], "plan"), ("cls.cu", [], "cls"), ("fused.cu", [], "fused"), ("interp.cu", [], "interp"), ("tensor.cu", [], "tensor"),
         ("srcinterp.cu", [], "srcinterp")] + [
    ("transfer.cu", [f"-DGCAMB_TU_SPARSE={sp}", f"-DGCAMB_TU_NSRC={ns}"], f"transfer_s{sp}n{ns}")
    for sp in (0, 1) for ns in (2, 3, 4)] + [
    ("transfer.cu", ["-DGCAMB_TU_SPARSE=0", f"-DGCAMB_TU_NSRC={ns}", "-DGCAMB_TU_CURVED=1"], f"transfer_curved_n{ns}")
    for ns in (2, 3)]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "--fmad=true", "-Xcompiler", "-fPIC", "-cudart", "shared",
    "-I", os.path.join(ROOT, "include"), "-I", CSRC,
]


def _stale() -> bool:
    if not (os.path.exists(LIB) and os.path.exists(PROBE_LIB)):
        return True
    t = min(os.path.getmtime(LIB), os.path.getmtime(PROBE_LIB))
    inc = os.path.join(ROOT, "include")
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(inc, f) for f in os.listdir(inc)] + [__file__]
    return any(os.path.getmtime(d) > t for d in deps)


def build_extension(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    debug = ["-DGCAMB_DEBUG"] if os.environ.get("GCAMB_DEBUG") == "1" else []   # device asserts on every index
    objdir = tempfile.mkdtemp(prefix="gcamb_build_")
    try:
        def compile_unit(unit):
            src, flags, tag = unit
            obj = os.path.join(objdir, tag + ".o")
            cmd = [nvcc, *NVCC_FLAGS, *debug, *flags, *(["-Xptxas", "-v"] if verbose else []),
                   "-c", os.path.join(CSRC, src), "-o", obj]
            subprocess.run(cmd, check=True)
            return obj
        with ThreadPoolExecutor(max_workers=min(len(UNITS) + 1, os.cpu_count() or 1)) as pool:
            probe = pool.submit(compile_unit, ("probe.cu", [], "probe"))
            objs = list(pool.map(compile_unit, UNITS))
            probe_obj = probe.result()
        link = [nvcc, "-shared", "-cudart", "shared", "-gencode", "arch=compute_100a,code=sm_100a"]
        tmp, tmp_probe = f"{LIB}.{os.getpid()}.tmp", f"{PROBE_LIB}.{os.getpid()}.tmp"
        subprocess.run([*link, *objs, "-o", tmp], check=True)
        subprocess.run([*link, probe_obj, "-o", tmp_probe], check=True)
    finally:
        shutil.rmtree(objdir, ignore_errors=True)
    os.replace(tmp_probe, PROBE_LIB)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build_extension(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
