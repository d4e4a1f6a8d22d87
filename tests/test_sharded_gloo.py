"""The N>1 host logic on CPU: two gloo ranks, each holding half of the parameter axis, with the CPU
oracle as the local operator; the all-reduced result must equal the unsharded oracle."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import toeplitz_plain as op
import synth
from paper_2501_14911_b200 import sharded
from tests.inputs_online import gstar_column


def test_shard_range_covers_and_aligns():
    for N_m, world in [(250000, 8), (100, 3), (17, 2), (64, 4), (5, 8), (65536, 7)]:
        ranges = [sharded.shard_range(N_m, r, world) for r in range(world)]
        assert ranges[0][0] == 0 and ranges[-1][1] == N_m
        for (a0, a1), (b0, b1) in zip(ranges, ranges[1:]):
            assert a1 == b0 and a0 <= a1
        assert all(p0 % 16 == 0 for p0, _ in ranges if p0 < N_m)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = synth.CONFIGS["C2"].scaled(N_d=3, N_m=70, N_t=12)
        F, m, d = synth.block_column(w).numpy(), synth.vector_m(w, k_rhs=1).numpy(), synth.vector_d(w, k_rhs=1).numpy()
        p0, p1 = sharded.shard_range(w.N_m, rank, world)
        Fl = F[:, :, p0:p1]
        oper = sharded.ShardedOperator(lambda x: torch.from_numpy(op.matvec(Fl, x.numpy())),
                                       lambda y: torch.from_numpy(op.rmatvec(Fl, y.numpy())))
        got_d = oper.matvec(torch.from_numpy(m[:, p0:p1].copy())).numpy()
        got_m = oper.rmatvec(torch.from_numpy(d)).numpy()
        got_n = oper.normal(torch.from_numpy(m[:, p0:p1].copy())).numpy()
        ref_d, ref_m = op.matvec(F, m), op.rmatvec(F, d)
        ref_n = op.rmatvec(F, ref_d)
        ok = (np.allclose(got_d, ref_d, rtol=0, atol=1e-12 * np.abs(ref_d).max())
              and np.allclose(got_m, ref_m[:, p0:p1], rtol=0, atol=1e-12 * np.abs(ref_m).max())
              and np.allclose(got_n, ref_n[:, p0:p1], rtol=0, atol=1e-11 * np.abs(ref_n).max()))
        # the online phase (eq 4.13) on the same two ranks: replicated K-solve, sharded G* and F
        from oracle import online_plain as oo
        wo = synth.CONFIGS["P5"].scaled(N_d=3, N_m=70, N_t=12, dtype=torch.float64)
        Fo = synth.block_column(wo)
        Go = gstar_column(wo, Fo).numpy()
        Fo = Fo.numpy()
        nv, dob = synth.noise_var(wo).numpy(), synth.vector_d(wo, k_rhs=1).numpy()
        Lc = oo.cholesky(oo.assemble_K(Fo, Go, nv))
        m_ref = oo.map_point(Fo, Go, nv, Lc, dob)
        Fl2, Gl2 = Fo[:, :, p0:p1], Go[:, :, p0:p1]
        solve = lambda b: oo.chol_solve(Lc, b.reshape(-1)).reshape(b.shape)
        st = {}

        def partial(dd):                                   # the oracle as the local first half
            st["y"] = dd.numpy() / nv
            return torch.from_numpy(op.matvec(Fl2, op.rmatvec(Gl2, st["y"])))

        finish = lambda b: torch.from_numpy(op.rmatvec(Gl2, st["y"] - solve(b.numpy())))
        gain = lambda dd: torch.from_numpy(op.rmatvec(Gl2, solve(dd.numpy())))
        smap = sharded.ShardedMapInference(partial, finish, gain)
        for gain in (False, True):
            got = smap.infer(torch.from_numpy(dob), gain_form=gain).numpy()
            ok = ok and np.allclose(got, m_ref[:, p0:p1], rtol=0, atol=1e-10 * np.abs(m_ref).max())
        # K = Gamma_noise + F G* assembled from the ranks' parameter slices: one all-reduce, the noise added once
        K_ref = oo.assemble_K(Fo, Go, nv)
        def add_noise(K):        # on a GPU: binding.tt_K_add_noise; here the test adds the diagonal itself
            K.view(-1)[:: K.shape[0] + 1] += torch.from_numpy(nv).reshape(-1)

        K_sh = sharded.assemble_K_sharded(lambda: torch.from_numpy(oo.assemble_K(Fl2, Gl2, np.zeros_like(nv))), add_noise).numpy()
        ok = ok and np.allclose(K_sh, K_ref, rtol=0, atol=1e-12 * np.abs(K_ref).max())
        with open(os.path.join(out_dir, f"rank{rank}.ok"), "w") as f:
            f.write("1" if ok else "0")
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_gloo_ranks_equal_unsharded_oracle(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    for r in range(world):
        with open(tmp_path / f"rank{r}.ok") as f:
            assert f.read() == "1", f"rank {r} disagrees with the unsharded oracle"
