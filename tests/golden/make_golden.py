"""Writes tests/golden/c1_oracle.txt and tests/golden/online_oracle.txt: the CPU oracle's outputs for BASELINE.json configs[0]
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

from oracle import online_plain as oo  # noqa: E402
from oracle import toeplitz_plain as op  # noqa: E402
import synth  # noqa: E402


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

    # the online phase (eq 4.13, 4.7, 4.10, 4.11) on the P5 recipe at C1's size, fp64: oracle/online_plain.py only
    import torch
    wo = synth.CONFIGS["P5"].scaled(N_d=4, N_m=64, N_t=32, dtype=torch.float64)
    wq = synth.CONFIGS["Q5"].scaled(N_d=2, N_m=64, N_t=32, dtype=torch.float64)
    Fo = synth.block_column(wo)
    Go = oo.gstar_block_column(Fo.numpy(), synth.prior_gamma(wo).numpy())
    Fq = synth.block_column(wq)
    Gq = oo.gstar_block_column(Fq.numpy(), synth.prior_gamma(wq).numpy())
    Fo, Fq = Fo.numpy(), Fq.numpy()
    nv, d_obs = synth.noise_var(wo).numpy(), synth.vector_d(wo, k_rhs=1).numpy()
    u = synth.vector_m(wo, k_rhs=1).numpy()
    L = oo.cholesky(oo.assemble_K(Fo, Go, nv))
    out = {"chol_solve": oo.chol_solve(L, d_obs.reshape(-1)).reshape(32, 4),
           "map_point": oo.map_point(Fo, Go, nv, L, d_obs),
           "smw_apply": oo.smw_apply(Fo, Go, L, u),
           "d2q": oo.d2q_apply(Fo, Go, nv, L, Fq, 4, d_obs)}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "online_oracle.txt")
    with open(path, "w") as f:
        f.write("# oracle/online_plain.py on the P5/Q5 recipes at N_d=4 (N_q=2), N_m=64, N_t=32 (out_every 4), fp64; "
                "written by tests/golden/make_golden.py\n")
        for name, a in out.items():
            f.write(f"{name} {a.shape[0]} {a.shape[1]}\n")
            for row in a:
                f.write(" ".join(float(x).hex() for x in row) + "\n")
    print(path)


if __name__ == "__main__":
    main()
