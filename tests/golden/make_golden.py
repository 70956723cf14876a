"""Writes tests/golden/oracle_tiny_samples.txt: a few entries of the oracle's R on config 0
(tiny, seed 0), as a regression anchor for the oracle + input generator pair.

Calls ONLY oracle/ (and the seeded input generator); never the CUDA path.
Run from the repo root:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import ppl_inputs  # noqa: E402

IDX = [(0, 0, 0, 0), (0, 1, 2, 3), (1, 0, 3, 2), (4, 4, 19, 19), (2, 3, 7, 11), (3, 2, 11, 7), (4, 0, 19, 0)]


def main():
    L, t2 = ppl_inputs.make_config("tiny", seed=0)
    R = oracle.bruteforce_direct(L, t2)  # the long-double seven-index sum: the most direct reading of eq. (6)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_tiny_samples.txt")
    with open(out, "w") as f:
        f.write("# R[i,j,a,b] of config 0 (nocc=5,nvirt=20,nchol=60, seed 0) from oracle.bruteforce_direct\n")
        f.write("# (eq. 6, PAPER.md:68, long-double accumulation); written by tests/golden/make_golden.py\n")
        f.write("# columns: i j a b value(hex float) value(repr)\n")
        for (i, j, a, b) in IDX:
            f.write(f"{i} {j} {a} {b} {float(R[i, j, a, b]).hex()} {float(R[i, j, a, b])!r}\n")
        f.write(f"# max|R| = {float(np.abs(R).max())!r}\n")
    print("wrote", out)


if __name__ == "__main__":
    main()
