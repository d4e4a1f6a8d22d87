"""Stored oracle outputs for C1 (tests/golden/c1_oracle.txt, written by tests/golden/make_golden.py from oracle/
only): the oracle still reproduces them bit for bit (CPU), and the CUDA path matches them within 1e-12 (GPU)."""
import os

import numpy as np
import pytest

from oracle import toeplitz_blocked as ob
from oracle import toeplitz_plain as op
import synth
from tests.inputs_online import gstar_column

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "c1_oracle.txt")


GOLD_ONLINE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "online_oracle.txt")


def load_golden(path=GOLD):
    out, name, rows = {}, None, []
    with open(path) as f:
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


def online_case():
    import torch
    from oracle import online_plain as oo
    wo = synth.CONFIGS["P5"].scaled(N_d=4, N_m=64, N_t=32, dtype=torch.float64)
    wq = synth.CONFIGS["Q5"].scaled(N_d=2, N_m=64, N_t=32, dtype=torch.float64)
    F = synth.block_column(wo)
    G = gstar_column(wo, F)
    Fq = synth.block_column(wq)
    nv, d_obs, u = synth.noise_var(wo), synth.vector_d(wo, k_rhs=1), synth.vector_m(wo, k_rhs=1)
    L = oo.cholesky(oo.assemble_K(F.numpy(), G.numpy(), nv.numpy()))
    return F, G, Fq, nv, d_obs, u, L


def test_online_oracle_reproduces_golden():
    from oracle import online_plain as oo
    g = load_golden(GOLD_ONLINE)
    F, G, Fq, nv, d_obs, u, L = online_case()
    Fn, Gn = F.numpy(), G.numpy()
    got = {"chol_solve": oo.chol_solve(L, d_obs.numpy().reshape(-1)).reshape(32, 4),
           "map_point": oo.map_point(Fn, Gn, nv.numpy(), L, d_obs.numpy()),
           "smw_apply": oo.smw_apply(Fn, Gn, L, u.numpy()),
           "d2q": oo.d2q_apply(Fn, Gn, nv.numpy(), L, Fq.numpy(), 4, d_obs.numpy())}
    for k, v in got.items():        # LAPACK / BLAS builds may differ in the last bits: rounding-level agreement
        assert np.linalg.norm(v - g[k]) <= 1e-11 * np.linalg.norm(g[k]), k


@pytest.mark.gpu
def test_cuda_online_path_matches_golden():
    import torch
    from paper_2501_14911_b200 import binding as tt
    g = load_golden(GOLD_ONLINE)
    F, G, Fq, nv, d_obs, u, L = online_case()
    pF, pG, pFq = tt.Plan(F.cuda()), tt.Plan(G.cuda()), tt.Plan(Fq.cuda(), out_every=4)
    chol = tt.Chol(torch.from_numpy(L).cuda())
    mp = tt.MapInference(pF, pG, chol, nv.cuda())
    try:
        work = torch.empty((32, 64), dtype=torch.float64, device="cuda")
        q = torch.empty((8, 2), dtype=torch.float64, device="cuda")
        tt.tt_d2q_apply(mp.handle, pFq.handle, tt.TT_MAP_PAPER, d_obs.cuda(), work, q)
        got = {"chol_solve": chol.solve(d_obs.cuda().reshape(-1)).reshape(32, 4),
               "map_point": mp.infer(d_obs.cuda(), tt.TT_MAP_PAPER), "smw_apply": mp.smw_apply(u.cuda()), "d2q": q}
        for k, v in got.items():
            a = v.cpu().numpy()
            assert np.linalg.norm(a - g[k]) <= 1e-10 * np.linalg.norm(g[k]), k
    finally:
        mp.close(); chol.close(); pF.close(); pG.close(); pFq.close()
