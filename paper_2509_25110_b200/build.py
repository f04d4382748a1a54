"""Builds libgcamb_los.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2509_25110_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgcamb_los.so")
SOURCES = ["api.cu", "plan.cu", "transfer.cu", "cls.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "--fmad=true", "-Xcompiler", "-fPIC", "-shared", "-cudart", "shared",
    "-I", os.path.join(ROOT, "include"), "-I", CSRC,
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(ROOT, "include", "gcamb_los.h"), __file__]
    return any(os.path.getmtime(d) > t for d in deps)


def build_extension(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = f"{LIB}.{os.getpid()}.tmp"
    debug = ["-DGCAMB_DEBUG"] if os.environ.get("GCAMB_DEBUG") == "1" else []   # device asserts on every index
    cmd = [nvcc, *NVCC_FLAGS, *debug, *(["-Xptxas", "-v"] if verbose else []),
           *[os.path.join(CSRC, s) for s in SOURCES], "-o", tmp]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build_extension(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
