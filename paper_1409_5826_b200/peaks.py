"""Run the FP64 / shared-memory micro-benchmarks (csrc/peaks.cu) on cuda:0 and
print their one-line JSON: `python -m paper_1409_5826_b200.peaks`."""
from __future__ import annotations

import json
import subprocess

from .build import build_peaks


def measure() -> dict:
    out = subprocess.run([build_peaks()], check=True, capture_output=True, text=True).stdout
    return json.loads(out.strip().splitlines()[-1])


if __name__ == "__main__":
    print(json.dumps(measure()))
