"""Writes the stored expected values under tests/golden/ -- calls ONLY oracle/ (never the CUDA path).

Run after the oracle's own pins (tests/test_oracle_*.py) pass:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import refbind as R  # noqa: E402


def main():
    _, ntri, edge = R.mc_table()
    with open(os.path.join(HERE, "mc_ntri.txt"), "w") as f:
        f.write("# triangles per marching-cubes case 0..255 of the oracle's GENERATED table (DESIGN.md D:M-TABLE);\n")
        f.write("# the paper prints only edge_table[8] = 0x80c (PAPER.md line 542), which the table reproduces.\n")
        f.write("# written by tests/golden/make_golden.py from oracle/ only.\n")
        for r in range(16):
            f.write(" ".join(str(int(x)) for x in ntri[16 * r:16 * r + 16]) + "\n")


if __name__ == "__main__":
    main()
