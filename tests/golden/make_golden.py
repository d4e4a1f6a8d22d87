"""Writes tests/golden/c1_oracle.txt: the CPU oracle's outputs for BASELINE.json configs[0]
(C1: N_d=4, N_m=64, N_t=32, fp64, seed 0), as hexadecimal fp64 so that nothing is lost in text.

    python tests/golden/make_golden.py

Calls only oracle/ and the seeded input generator.  The paper prints no worked numerical example of the
block-Toeplitz matvec (no input/output pair anywhere in PAPER.md), so this directory holds no paper values;
this file pins the oracle's C1 results against accidental change and gives the GPU path a stored target that
never came from the CUDA path.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import toeplitz_plain as op  # noqa: E402
from paper_2501_14911_b200 import synth  # noqa: E402


def main():
    w = synth.CONFIGS["C1"]
    F = synth.block_column(w).numpy()
    m = synth.vector_m(w, k_rhs=1).numpy()
    d = synth.vector_d(w, k_rhs=1).numpy()
    out = {"matvec": op.matvec(F, m), "rmatvec": op.rmatvec(F, d), "normal": op.normal(F, m)}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c1_oracle.txt")
    with open(path, "w") as f:
        f.write("# oracle/toeplitz_plain.py on C1 (BASELINE.json configs[0]); written by tests/golden/make_golden.py\n")
        for name, a in out.items():
            f.write(f"{name} {a.shape[0]} {a.shape[1]}\n")
            for row in a:
                f.write(" ".join(float(x).hex() for x in row) + "\n")
    print(path)


if __name__ == "__main__":
    main()
