"""The N_m-sharded route ("24 Nvidia A100 GPUs") as far as ONE device allows: the ranks
are emulated one after the other in a single process on cuda:0 - every "rank" owns a plan built on its own p_range slice of
the same block column, exactly what bench.py --parallel shard builds per GPU - and the sum of their partial results stands
in for the all-reduce (the real exchange is covered by tests/test_sharded_gloo.py with two gloo ranks on CPU).  The wrappers
of paper_2501_14911_b200/sharded.py run unchanged; only their `all_reduce` callable is the stand-in.  Compared with the
unsharded plan on the same device and with the oracle."""
import numpy as np
import pytest
import torch

import synth
from oracle import online_plain as oo
from oracle import toeplitz_blocked as ob
from paper_2501_14911_b200 import sharded
from tests.inputs_online import gstar_column

pytestmark = pytest.mark.gpu

TOL = {torch.float64: 1e-12, torch.float32: 1e-5}


@pytest.fixture(scope="module")
def tt():
    from paper_2501_14911_b200 import binding
    binding.lib()
    return binding


def rel(a, b):
    a, b = np.asarray(a, np.float64).ravel(), np.asarray(b, np.float64).ravel()
    return np.linalg.norm(a - b) / np.linalg.norm(b)


class SumOfRanks:
    """Stand-in for the all-reduce: replaces a rank's partial by the sum of what every emulated rank contributed."""

    def __init__(self):
        self.parts, self.total = [], None

    def collect(self, t):
        self.parts.append(t.clone())

    def __call__(self, t):
        if self.total is None:
            self.total = torch.stack(self.parts).sum(0)
        t.copy_(self.total)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32], ids=["f64", "f32"])
@pytest.mark.parametrize("world", [2, 3])
def test_sharded_operator_equals_unsharded_plan_and_oracle(tt, dtype, world):
    w = synth.CONFIGS["C2"].scaled(N_d=5, N_m=9000 + 7, N_t=48, dtype=dtype)     # several GEMV chunks per rank, ragged tail
    F, m, d = synth.block_column(w), synth.vector_m(w, k_rhs=1), synth.vector_d(w, k_rhs=1)
    ranges = [sharded.shard_range(w.N_m, r, world) for r in range(world)]
    plans = [tt.Plan(F[:, :, p0:p1].contiguous().cuda()) for p0, p1 in ranges]
    whole = tt.Plan(F.cuda())
    try:
        red, red_n = SumOfRanks(), SumOfRanks()
        for (p0, p1), pl in zip(ranges, plans):                                 # what every rank contributes
            part = pl.matvec(m[:, p0:p1].contiguous().cuda())
            red.collect(part); red_n.collect(part)
        d_ranks, m_ranks, n_ranks = [], [], []
        for (p0, p1), pl in zip(ranges, plans):                                 # the wrapper itself, per rank
            m_loc = m[:, p0:p1].contiguous().cuda()
            d_ranks.append(sharded.from_plan(pl, all_reduce=red).matvec(m_loc))
            m_ranks.append(sharded.from_plan(pl, all_reduce=red).rmatvec(d.cuda()))
            n_ranks.append(sharded.from_plan(pl, all_reduce=red_n).normal(m_loc))
        got_d = d_ranks[0].cpu().numpy()
        for x in d_ranks[1:]:
            assert torch.equal(x, d_ranks[0])                                   # d is replicated after the exchange
        got_m = torch.cat(m_ranks, dim=1).cpu().numpy()
        got_n = torch.cat(n_ranks, dim=1).cpu().numpy()
        one_d, one_m, one_n = whole.matvec(m.cuda()).cpu().numpy(), whole.rmatvec(d.cuda()).cpu().numpy(), whole.normal(m.cuda()).cpu().numpy()
    finally:
        for pl in plans:
            pl.close()
        whole.close()
    tol = TOL[dtype]
    ref_d, ref_m = ob.matvec(F.numpy(), m.numpy()), ob.rmatvec(F.numpy(), d.numpy())
    ref_n = ob.rmatvec(F.numpy().astype(np.float64), ref_d)
    assert rel(got_d, ref_d) <= tol and rel(got_m, ref_m) <= tol and rel(got_n, ref_n) <= tol
    assert rel(got_d, one_d) <= tol and rel(got_n, one_n) <= tol
    assert np.array_equal(got_m, one_m)        # F^T d needs no exchange: each rank's slice is the unsharded result bit for bit


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32], ids=["f64", "f32"])
def test_sharded_online_phase_equals_oracle(tt, dtype):
    """eq (4.13) and K = Gamma_noise + F G* with the parameter axis split over two emulated ranks."""
    world = 2
    w = synth.CONFIGS["P5"].scaled(N_d=4, N_m=2100, N_t=16, dtype=dtype)
    F = synth.block_column(w)
    G = gstar_column(w, F)
    nv, d_obs = synth.noise_var(w), synth.vector_d(w, k_rhs=1)
    K_ref = oo.assemble_K(F.numpy(), G.numpy(), nv.numpy())
    L = oo.cholesky(K_ref)
    m_ref = oo.map_point(F.numpy(), G.numpy(), nv.numpy(), L, d_obs.numpy(), conv=ob)
    kappa = np.linalg.cond(K_ref)
    ranges = [sharded.shard_range(w.N_m, r, world) for r in range(world)]
    n = w.N_d * w.N_t
    dt = tt.TT_F32 if dtype == torch.float32 else tt.TT_F64
    objs = []
    try:
        mps = []
        for p0, p1 in ranges:
            pF, pG = tt.Plan(F[:, :, p0:p1].contiguous().cuda()), tt.Plan(G[:, :, p0:p1].contiguous().cuda())
            chol = tt.Chol(torch.from_numpy(L).cuda())
            mp = tt.MapInference(pF, pG, chol, nv.cuda())
            objs += [mp, chol, pF, pG]
            mps.append(mp)
        red = SumOfRanks()
        for mp in mps:
            _, b = mp.infer_partial(d_obs.cuda())
            red.collect(b)
        paper = torch.cat([sharded.map_from_binding(mp, all_reduce=red).infer(d_obs.cuda()) for mp in mps], dim=1).cpu().numpy()
        gain = torch.cat([sharded.map_from_binding(mp, all_reduce=red).infer(d_obs.cuda(), gain_form=True) for mp in mps], dim=1).cpu().numpy()
        # K: every rank's F G* without noise, summed, noise added once by the library
        redK = SumOfRanks()
        for p0, p1 in ranges:
            redK.collect(tt.assemble_K_direct(F[:, :, p0:p1].contiguous().cuda(), G[:, :, p0:p1].contiguous().cuda(), None))
        p0, p1 = ranges[0]
        K = sharded.assemble_K_sharded(
            lambda: tt.assemble_K_direct(F[:, :, p0:p1].contiguous().cuda(), G[:, :, p0:p1].contiguous().cuda(), None),
            lambda Kt: tt.tt_K_add_noise(nv.cuda(), n, dt, Kt, Kt.stride(0)), all_reduce=redK).cpu().numpy()
    finally:
        for o in objs:
            o.close()
    u = 1.1e-16 if dtype == torch.float64 else 6e-8
    assert rel(K, K_ref) <= TOL[dtype]
    assert rel(gain, m_ref) <= TOL[dtype] + 8 * 1.1e-16 * kappa
    assert rel(paper, m_ref) <= TOL[dtype] + 8 * u * kappa


def test_bench_shard_branch_runs_nccl_on_one_gpu(tmp_path):
    """bench.py --parallel shard as the driver launches it (torch.distributed.run, one rank per GPU) with ONE rank: NCCL comes
    up, the all-reduce of d runs on the launching stream inside the timed step, and the step takes what the unsharded step
    takes.  configs[1] (C2, 4.3 GB spectrum) keeps it short."""
    import json
    import os
    import socket
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "1", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(root, "bench.py"), "--gpus", "1", "--parallel", "shard", "--config", "C2",
           "--steps", "5", "--warmup", "3", "--no-cpu-baseline", "--no-library-baseline"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=900, cwd=root)
    assert res.returncode == 0, res.stderr[-3000:]
    line = json.loads([l for l in res.stdout.strip().splitlines() if l.startswith("{")][-1])
    assert line["scaling"] == "strong" and line["n_gpus"] == 1
    assert line["exchange"]["collective"].startswith("NCCL") and line["exchange"]["world_size"] == 1
    assert line["exchange"]["bytes"] == 256 * 64 * 8
    assert 0.5 < line["ms_per_step"] < 5.0                      # C2: ~1.4 ms unsharded
