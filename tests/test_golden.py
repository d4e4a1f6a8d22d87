"""Stored oracle outputs for C1 (tests/golden/c1_oracle.txt, written by tests/golden/make_golden.py from oracle/
only): the oracle still reproduces them bit for bit (CPU), and the CUDA path matches them within 1e-12 (GPU)."""
import os

import numpy as np
import pytest

from oracle import toeplitz_blocked as ob
from oracle import toeplitz_plain as op
from paper_2501_14911_b200 import synth

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "c1_oracle.txt")


def load_golden():
    out, name, rows = {}, None, []
    with open(GOLD) as f:
        for line in f:
            if line.startswith("#"):
                continue
            t = line.split()
            if t and not t[0].startswith(("0x", "-0x")):
                name, rows = t[0], []
                out[name] = rows
            elif t:
                rows.append([float.fromhex(x) for x in t])
    return {k: np.array(v) for k, v in out.items()}


def c1():
    w = synth.CONFIGS["C1"]
    return synth.block_column(w), synth.vector_m(w, k_rhs=1), synth.vector_d(w, k_rhs=1)


def test_oracle_reproduces_golden_bit_for_bit():
    g = load_golden()
    F, m, d = c1()
    assert g["matvec"].shape == (32, 4) and g["rmatvec"].shape == (32, 64) and g["normal"].shape == (32, 64)
    assert np.array_equal(op.matvec(F.numpy(), m.numpy()), g["matvec"])
    assert np.array_equal(op.rmatvec(F.numpy(), d.numpy()), g["rmatvec"])
    assert np.array_equal(op.normal(F.numpy(), m.numpy()), g["normal"])
    # the blocked build sums in another (fixed) order: rounding-level agreement
    assert np.abs(ob.matvec(F.numpy(), m.numpy()) - g["matvec"]).max() <= 1e-13 * np.abs(g["matvec"]).max()


@pytest.mark.gpu
def test_cuda_path_matches_golden():
    from paper_2501_14911_b200 import binding as tt
    g = load_golden()
    F, m, d = c1()
    plan = tt.Plan(F.cuda())
    try:
        got = {"matvec": plan.matvec(m.cuda()), "rmatvec": plan.rmatvec(d.cuda()), "normal": plan.normal(m.cuda())}
        for k, v in got.items():
            a = v.cpu().numpy()
            assert np.linalg.norm(a - g[k]) <= 1e-12 * np.linalg.norm(g[k]), k
    finally:
        plan.close()
