"""GPU parity for the operator with its output on a coarser time grid (tt_plan_create_coarse; the p2q map of
PAPER.md:140-162, 381, 405; reading R19) against oracle/toeplitz_plain.matvec_decimated / rmatvec_decimated.
Same bar as the p2o map: relative L2 <= 1e-12 (fp64), <= 1e-5 (fp32)."""
import numpy as np
import pytest
import torch

from oracle import toeplitz_blocked as ob
from oracle import toeplitz_plain as op
import synth

pytestmark = pytest.mark.gpu
TOL = {torch.float64: 1e-12, torch.float32: 1e-5}


@pytest.fixture(scope="module")
def tt():
    from paper_2501_14911_b200 import binding
    binding.lib()
    return binding


def rel(a, b):
    a = np.asarray(a, dtype=np.float64).ravel()
    b = np.asarray(b, dtype=np.float64).ravel()
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / (nb if nb > 0 else 1.0)


# (N_q, N_m, N_t, out_every): the paper's ratio 10, ragged tiles, r = N_t (a single output step), r = 1
SHAPES = [(2, 70, 20, 10), (3, 1000, 50, 5), (1, 33, 12, 12), (4, 2100, 36, 2), (16, 300, 100, 10), (2, 40, 15, 1)]


@pytest.mark.parametrize("N_q,N_m,N_t,r", SHAPES)
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("layout", [0, 1])
def test_coarse_output(tt, N_q, N_m, N_t, r, dtype, layout):
    w = synth.CONFIGS["C2"].scaled(N_d=N_q, N_m=N_m, N_t=N_t, dtype=dtype)
    F, m = synth.block_column(w), synth.vector_m(w, k_rhs=1)
    q = synth.vector_d(w.scaled(N_t=N_t // r), k_rhs=1)
    ref_q = op.matvec_decimated(F.numpy(), m.numpy(), r)
    ref_m = op.rmatvec_decimated(F.numpy(), q.numpy(), r)
    ref_n = op.rmatvec_decimated(F.numpy(), ref_q, r)
    lay = (lambda t: t.t().contiguous()) if layout == 1 else (lambda t: t)
    unlay = (lambda t: t.t()) if layout == 1 else (lambda t: t)
    plan = tt.Plan(F.cuda(), layout=layout, out_every=r)
    try:
        got_q = unlay(plan.matvec(lay(m).cuda())).cpu().numpy()
        got_m = unlay(plan.rmatvec(lay(q).cuda())).cpu().numpy()
        got_n = unlay(plan.normal(lay(m).cuda())).cpu().numpy()
    finally:
        plan.close()
    assert got_q.shape == (N_t // r, N_q)
    assert rel(got_q, ref_q) <= TOL[dtype]
    assert rel(got_m, ref_m) <= TOL[dtype]
    assert rel(got_n, ref_n) <= TOL[dtype]


@pytest.mark.parametrize("layout", [0, 1])
def test_coarse_output_batched(tt, layout):
    N_q, N_m, N_t, r, k = 3, 500, 40, 4, 5
    w = synth.CONFIGS["C4"].scaled(N_d=N_q, N_m=N_m, N_t=N_t)
    F = synth.block_column(w)
    M = synth.vector_m(w, k_rhs=k)                               # [N_t, N_m, k]
    Q = synth.vector_d(w.scaled(N_t=N_t // r), k_rhs=k)          # [N_t/r, N_q, k]
    ref_Q = op.matvec_decimated(F.numpy(), M.numpy(), r)
    ref_M = op.rmatvec_decimated(F.numpy(), Q.numpy(), r)
    lay = (lambda t: t.permute(2, 1, 0).contiguous()) if layout == 1 else (lambda t: t)
    unlay = (lambda t: t.permute(2, 1, 0)) if layout == 1 else (lambda t: t)
    plan = tt.Plan(F.cuda(), layout=layout, k_max=k, out_every=r)
    try:
        got_Q = unlay(plan.matvec_batched(lay(M).cuda())).cpu().numpy()
        got_M = unlay(plan.rmatvec_batched(lay(Q).cuda())).cpu().numpy()
    finally:
        plan.close()
    assert rel(got_Q, ref_Q) <= 1e-12 and rel(got_M, ref_M) <= 1e-12


def test_coarse_errors(tt):
    w = synth.CONFIGS["C1"]
    F = synth.block_column(w).cuda()
    for bad in (0, 3, 64):            # 32 steps: 3 does not divide, 64 > N_t
        with pytest.raises(tt.TTError) as ei:
            tt.Plan(F, out_every=bad)
        assert ei.value.status == -2  # TT_ERR_SHAPE


def test_p2q_full_size_whole_vector(tt):
    """The paper's p2q shape (N_q = 16, N_m = 263169, N_t = 500, N_t^q = 50), in the launch
    configuration bench.py --config Q5 times: q = S F_q m over all 800 QoIs and m' = F_q^T S^T q over all 131 584 500
    parameters against the blocked oracle (reading R19: fine-grid result sampled at the end of every r-th step; exact
    transpose with zeros at the unsampled steps), the block column streamed to the host in sensor slabs."""
    import time
    w = synth.CONFIGS["Q5"]
    free, _ = torch.cuda.mem_get_info()
    if free < 40 * (1 << 30):
        pytest.skip("needs 40 GiB of free device memory")
    r = 10
    F = synth.block_column(w, device="cuda")
    m = synth.vector_m(w, device="cuda")
    q = synth.vector_d(w.scaled(N_t=w.N_t // r), device="cuda")
    plan = tt.Plan(F, out_every=r)
    try:
        got_q, got_m = plan.matvec(m), plan.rmatvec(q)
        torch.cuda.synchronize()
    finally:
        plan.close()
    lhs = float((got_q.double() * q.double()).sum())
    rhs = float((m.double() * got_m.double()).sum())
    assert abs(lhs - rhs) <= 1e-5 * float(got_q.double().norm() * q.double().norm())
    mh, qh = m.cpu().numpy(), q.cpu().numpy()
    zq = np.zeros((w.N_t, w.N_d), dtype=np.float32)
    zq[r - 1::r] = qh                                               # S^T q
    ref_q = np.empty((w.N_t // r, w.N_d))
    ref_m = np.zeros((w.N_t, w.N_m))
    t0 = time.perf_counter()
    for s0 in range(0, w.N_d, 4):
        slab = F[:, s0:s0 + 4, :].contiguous().cpu().numpy()
        ref_q[:, s0:s0 + 4] = ob.matvec(slab, mh)[r - 1::r]         # S (F m)
        ref_m += ob.rmatvec(slab, np.ascontiguousarray(zq[:, s0:s0 + 4]))
    e_q, e_m = rel(got_q.cpu().numpy(), ref_q), rel(got_m.cpu().numpy(), ref_m)
    print(f"Q5 whole-vector rel-L2 vs the oracle (oracle {time.perf_counter() - t0:.0f} s): S F_q m {e_q:.2e}  F_q^T S^T q {e_m:.2e} (tol 1e-05)")
    assert e_q <= 1e-5 and e_m <= 1e-5
    gm = got_m.cpu().numpy()
    for p0 in range(0, w.N_m, 8192):
        assert rel(gm[:, p0:p0 + 8192], ref_m[:, p0:p0 + 8192]) <= 1e-5, f"parameters {p0}.."
