"""Micro-benchmarks behind bench.py's roofline denominators (bench_peaks.cu): plain FP64 issue
rate and conflict-free LDS bandwidth of the GPU it runs on.  `python bench_peaks.py` builds the
binary beside this file, runs it on cuda:0 and prints its one-line JSON; the committed copy of
that line is profiles/peaks.json.  A measurement tool of the bench, not part of the library."""
from __future__ import annotations

import json
import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "bench_peaks.cu")
BIN = os.path.join(HERE, "bench_peaks.bin")


def build(force: bool = False) -> str:
    if force or not os.path.exists(BIN) or os.path.getmtime(BIN) < os.path.getmtime(SRC):
        nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
        tmp = BIN + f".tmp{os.getpid()}"
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo",
                               "-std=c++17", "-cudart", "static", SRC, "-o", tmp])
        os.replace(tmp, BIN)
    return BIN


def measure() -> dict:
    out = subprocess.run([build()], check=True, capture_output=True, text=True).stdout
    return json.loads(out.strip().splitlines()[-1])


if __name__ == "__main__":
    print(json.dumps(measure()))
