"""Writes the stored expected values under tests/golden/ that are NOT the paper's own.

Calls only ``oracle/`` (and the shared seeded input generators): nothing here comes from
the CUDA path.  Run from the repo root:  python tests/golden/make_golden.py
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import awg_workloads as W  # noqa: E402
import oracle  # noqa: E402


def main():
    p = oracle.plan_from_workload(W.config1())
    codes = p.codes(0, 64)
    with open(os.path.join(HERE, "c1_head_codes.txt"), "w") as f:
        f.write("# first 64 int16 codes of BASELINE.json config 1 (16 tones, 560 MS/s, seed 0), oracle/awg_oracle.py\n")
        f.write("# written by tests/golden/make_golden.py; definition: PAPER.md:133 (Eq. 9), 141 (Eq. 10), 332 (Eq. 14)\n")
        f.write("\n".join(str(int(c)) for c in codes) + "\n")


if __name__ == "__main__":
    main()
