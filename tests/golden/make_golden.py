"""Writes tests/golden/oracle_regression.txt.  Calls ONLY oracle/ and workloads/ (never the CUDA path).

The paper prints no worked numeric example (PAPER.md has four equations and one table of ratios), so this
fixture is not a paper value: it freezes the oracle's own output on a small seeded input so that a later,
unintended change to oracle/hs_oracle.c or to workloads/ is caught.  The independent pins are in
tests/test_oracle_pins.py.  Regenerate with:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle      # noqa: E402
import workloads   # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.txt")
BINS = [0, 1, 2, 31, 32, 33, 127, 128, 129, 500, 1023, 1024, 2047, 2048, 3000, 4095]


def main():
    x, _ = workloads.comb_batch_numpy(2, [7], 4096, 1.0, 50.0, 120.0, 0.10)
    lines = ["# oracle regression fixture; written by tests/golden/make_golden.py (oracle/ + workloads/ only)",
             "# input: workloads.comb_batch_numpy(2, [7], 4096, 1.0, 50.0, 120.0, 0.10); eqs. 1-4 of PAPER.md:17,33,38,43",
             f"# checksum {workloads.checksum(x)}",
             "# variant bin h_1 h_2 h_4 h_8 h_16 h_32 argmax j_32"]
    for v in ("standard", "max", "freqbin", "greedy"):
        o = oracle.harmonic_sum(x, 32, v, want_jpath=True)
        for n in BINS:
            h = " ".join(f"{o['sums'][0, l, n]:.17g}" for l in range(6))
            lines.append(f"{v} {n} {h} {int(o['argmax'][0, n])} {int(o['jpath'][0, 5, n])}")
    with open(OUT, "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
