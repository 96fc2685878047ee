"""Compile csrc/ into paper_1409_5826_b200/libkinnet.so for sm_100a (in-tree)."""
from __future__ import annotations

import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libkinnet.so")
SOURCES = [os.path.join(CSRC, "kinnet.cu"), os.path.join(CSRC, "schedule.cpp")]
HEADERS = [os.path.join(CSRC, "schedule.h"), os.path.join(HERE, "..", "include", "kinnet.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC,-O2,-Wall",
    "-shared", "-cudart", "static",
]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA extension cannot be built")
    return exe


PEAKS_SRC = os.path.join(CSRC, "peaks.cu")
PEAKS_BIN = os.path.join(HERE, "kinnet_peaks")


def build_peaks(force: bool = False) -> str:
    """Micro-benchmark binary for the FP64 / shared-memory roofline denominators."""
    if force or not os.path.exists(PEAKS_BIN) or os.path.getmtime(PEAKS_BIN) < os.path.getmtime(PEAKS_SRC):
        tmp = PEAKS_BIN + f".tmp{os.getpid()}"
        subprocess.check_call([nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo",
                               "-std=c++17", "-cudart", "static", PEAKS_SRC, "-o", tmp])
        os.replace(tmp, PEAKS_BIN)
    return PEAKS_BIN


def build(force: bool = False, verbose: bool = False) -> str:
    deps = SOURCES + HEADERS + [__file__]
    newest = max(os.path.getmtime(p) for p in deps)
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < newest:
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), *SOURCES, "-o", tmp]
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    import sys

    print(build(force=True, verbose="-v" in sys.argv))
    print(build_peaks(force=True))
