"""Writes the stored expected values under tests/golden/ from the CPU oracle.

    python tests/golden/make_golden.py

Calls only `oracle/` and the seeded input generators `gen/` (never the CUDA
path).  The files are regression pins of the oracle's own arithmetic: a later
change to the oracle that moves one of them must name, in its commit message,
the PAPER.md passage or DESIGN.md reading that justifies it.

  config1_oracle.txt   BASELINE.json configs[0] (g16, T9 = 3, rho = 1e8, X0 = X1 = 0.5):
                       final Y after the three fixed-dt runs of DESIGN.md section 3
                       (dt = 1e-10 x 10000: all Euler; dt = 1e-5 and 1e-4 x 1000:
                       mixed with Eq. (3)), with the count of asymptotic
                       species-steps.
"""
from __future__ import annotations

import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

RUNS = ((1e-10, 10_000), (1e-5, 1_000), (1e-4, 1_000))


def config1_lines():
    from gen import build_config
    from oracle import Oracle

    c = build_config(1)
    o = Oracle(c["network"])
    lines = ["# written by tests/golden/make_golden.py from oracle/ (fp64, hex floats)",
             "# run <dt> <n_steps> <n_asymptotic_species_steps>, then one line per species: index Y"]
    for dt, n in RUNS:
        out = o.integrate_fixed(c["T9"], c["rho"], c["Y0"], dt, n)
        lines.append(f"run {dt!r} {n} {int(out['n_asym'][0])}")
        lines += [f"{i} {float(v).hex()}" for i, v in enumerate(out["Y"][0])]
    return lines


def main():
    with open(os.path.join(HERE, "config1_oracle.txt"), "w") as fh:
        fh.write("\n".join(config1_lines()) + "\n")


if __name__ == "__main__":
    main()
