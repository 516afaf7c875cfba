"""Writes tests/golden/cfg0_rows.txt: rows of configs[0] (single s-wave boson channel, 10x10 cells, orders 4/4/8)
computed by the CPU oracle alone — a regression fixture for the oracle's arithmetic.  Calls only oracle/ and the
shared input generators; never the CUDA path.  Run from the repository root:  python tests/golden/make_cfg0_rows.py"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle.pm_oracle import Oracle            # noqa: E402
from paper_1508_07441_b200 import inputs      # noqa: E402

CELLS = (0, 37, 55, 99)


def main():
    wl = inputs.config(0)
    o = Oracle()
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg0_rows.txt"), "w") as f:
        f.write("# oracle rows of BASELINE.json configs[0]; written by tests/golden/make_cfg0_rows.py (oracle only)\n")
        f.write("# source_cell column value(hex float) value(decimal)\n")
        for c in CELLS:
            rp, ci, v = o.build_csr(wl, c, c + 1)
            for col, val in zip(ci.tolist(), v.tolist()):
                f.write(f"{c} {col} {float(val).hex()} {val:.17e}\n")


if __name__ == "__main__":
    main()
