"""Compile csrc/ into paper_1409_5826_b200/libkinnet.so for sm_100a (in-tree).

Objects are built in parallel (the pull kernel is instantiated once per state
type and mode, csrc/pull_inst.cu; the two-species kernel once per state type,
mode and side-a slot capacity, csrc/pull2_inst.cu) and cached under csrc/build/
by mtime.
"""
from __future__ import annotations

import os
import shutil
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libkinnet.so")
HEADERS = [os.path.join(CSRC, h) for h in ("schedule.h", "zone_pull.cuh", "zone_pull2.cuh", "device_util.cuh")] + [
    os.path.join(HERE, "..", "include", "kinnet.h")]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = [*ARCH, "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC,-O2,-Wall"]

# (object name, source, extra defines)
UNITS = [
    ("kinnet.o", "kinnet.cu", []),
    ("schedule.o", "schedule.cpp", []),
] + [
    (f"pull_f{bits}_{mode}.o", "pull_inst.cu",
     [f"-DPULL_REAL={real}", f"-DPULL_ADAPT={int(mode == 'adaptive')}",
      f"-DPULL_FN=pull_kernel_f{bits}_{mode}"])
    for bits, real in ((64, "double"), (32, "float")) for mode in ("adaptive", "fixed")
] + [
    (f"pull2_f{bits}_{mode}_cap{cap}.o", "pull2_inst.cu",
     [f"-DPULL_REAL={real}", f"-DPULL_ADAPT={int(mode == 'adaptive')}",
      f"-DPULL_FN=pull2_kernel_f{bits}_{mode}", f"-DPULL_CAP={cap}",
      *(["-DPULL2_DEFINE_SUPPORTED"] if (bits, mode) == (64, "adaptive") else [])])
    for bits, real in ((64, "double"), (32, "float")) for mode in ("adaptive", "fixed") for cap in (20, 24)
]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA extension cannot be built")
    return exe


def _compile(unit, force: bool, verbose: bool) -> tuple[str, bool]:
    name, src, defs = unit
    src = os.path.join(CSRC, src)
    obj = os.path.join(OBJ, name)
    newest = max(os.path.getmtime(p) for p in [src, *HEADERS, __file__])
    if not force and os.path.exists(obj) and os.path.getmtime(obj) >= newest:
        return obj, False
    tmp = obj + f".tmp{os.getpid()}"
    cmd = [nvcc(), *NVCC_FLAGS, *defs, *(["-Xptxas", "-v"] if verbose else []), "-c", src, "-o", tmp]
    subprocess.check_call(cmd)
    os.replace(tmp, obj)
    return obj, True


def build(force: bool = False, verbose: bool = False) -> str:
    sources = {os.path.join(CSRC, src) for _, src, _ in UNITS}
    newest = max(os.path.getmtime(p) for p in [*sources, *HEADERS, __file__])
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB  # up to date (the object cache does not travel to the GPU box)
    os.makedirs(OBJ, exist_ok=True)
    with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 1)) as pool:
        done = list(pool.map(lambda u: _compile(u, force, verbose), UNITS))
    if force or not os.path.exists(LIB) or any(changed for _, changed in done):
        tmp = LIB + f".tmp{os.getpid()}"
        subprocess.check_call([nvcc(), *ARCH, "-shared", "-cudart", "static",
                               *[obj for obj, _ in done], "-o", tmp])
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    import sys

    print(build(force=True, verbose="-v" in sys.argv))
