"""GPU parity: the CUDA path, called through the C ABI (libtt.so via the ctypes binding),
against the CPU oracle (oracle/), element by element on the same seeded inputs.

Bar (BASELINE.json north_star): relative L2 error over the whole output vector
  <= 1e-12 for fp64/complex128,  <= 1e-5 for fp32/complex64.
"""
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


def workload(base, N_d, N_m, N_t, dtype=None):
    w = synth.CONFIGS[base].scaled(N_d=N_d, N_m=N_m, N_t=N_t)
    if dtype is not None:
        w = w.scaled(dtype=dtype)
    return w


def inputs(w):
    F = synth.block_column(w)
    m = synth.vector_m(w, k_rhs=1)
    d = synth.vector_d(w, k_rhs=1)
    return F, m, d


# (base recipe, N_d, N_m, N_t): C1 as given; shrunken copies of C2..C5 that still span several
# FFT tiles (32 series), several GEMV chunks (2048) and ragged tails; odd / prime-factor N_t.
SHAPES = [
    ("C1", 4, 64, 32),
    ("C1", 3, 5, 7),
    ("C1", 1, 1, 1),
    ("C1", 2, 3, 1),
    ("C1", 1, 4, 6),
    ("C1", 4, 1, 5),
    ("C1", 5, 100, 15),
    ("C1", 3, 70, 35),
    ("C1", 2, 33, 21),
    ("C1", 2, 40, 49),
    ("C2", 7, 1000, 50),
    ("C2", 64, 4099, 64),
    ("C2", 16, 6000, 256),
    ("C3", 10, 5000, 400),
    ("C3", 100, 2500, 100),
    ("C4", 8, 4500, 512),
    ("C5", 20, 3000, 400),
    ("C5", 3, 2049, 500),
    ("C2", 2, 17, 900),
]


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32], ids=["f64", "f32"])
@pytest.mark.parametrize("base,N_d,N_m,N_t", SHAPES)
def test_matvec_rmatvec_normal_vs_oracle(tt, base, N_d, N_m, N_t, dtype):
    w = workload(base, N_d, N_m, N_t, dtype)
    F, m, d = inputs(w)
    plan = tt.Plan(F.cuda())
    try:
        got_d = plan.matvec(m.cuda()).cpu().numpy()
        got_m = plan.rmatvec(d.cuda()).cpu().numpy()
        got_n = plan.normal(m.cuda()).cpu().numpy()
    finally:
        plan.close()
    orc = op if N_t * N_t * N_d * N_m < 2e6 else ob
    ref_d = orc.matvec(F.numpy(), m.numpy())
    ref_m = orc.rmatvec(F.numpy(), d.numpy())
    ref_n = orc.rmatvec(F.numpy().astype(np.float64), ref_d)
    tol = TOL[dtype]
    assert rel(got_d, ref_d) <= tol
    assert rel(got_m, ref_m) <= tol
    assert rel(got_n, ref_n) <= tol


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32], ids=["f64", "f32"])
def test_host_block_column_equals_device_block_column(tt, dtype):
    w = workload("C2", 9, 700, 48, dtype)
    F, m, _ = inputs(w)
    p1, p2 = tt.Plan(F.cuda()), tt.Plan(F)  # device pointer / pageable host pointer
    try:
        assert torch.equal(p1.spectrum(), p2.spectrum())
        assert torch.equal(p1.matvec(m.cuda()), p2.matvec(m.cuda()))
    finally:
        p1.close(); p2.close()


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32], ids=["f64", "f32"])
def test_spectrum_pins(tt, dtype):
    """Fhat against what the mathematics fixes: DC and Nyquist bins, Parseval, a naive O(L^2) DFT."""
    w = workload("C2", 3, 37, 20, dtype)
    F = synth.block_column(w)
    plan = tt.Plan(F.cuda())
    try:
        S = plan.spectrum().cpu().numpy().astype(np.complex128)
    finally:
        plan.close()
    Fn = F.numpy().astype(np.float64)
    N_t = w.N_t
    L = 2 * N_t
    tol = 1e-13 if dtype == torch.float64 else 2e-7
    scale = np.abs(Fn).sum(axis=0).max()
    assert np.abs(S[0] - Fn.sum(axis=0)).max() <= tol * scale
    sign = (-1.0) ** np.arange(N_t)
    assert np.abs(S[N_t] - np.tensordot(sign, Fn, axes=(0, 0))).max() <= tol * scale
    assert np.abs(S[0].imag).max() == 0.0 and np.abs(S[N_t].imag).max() == 0.0
    wts = np.full(N_t + 1, 2.0); wts[0] = wts[-1] = 1.0
    lhs = np.tensordot(wts, np.abs(S) ** 2, axes=(0, 0))
    rhs = L * (Fn ** 2).sum(axis=0)
    assert np.abs(lhs - rhs).max() <= 50 * tol * rhs.max()
    k = np.arange(N_t)
    for (s, p) in [(0, 0), (2, 36), (1, 17)]:
        for om in [1, 7, N_t - 1]:
            naive = np.sum(Fn[:, s, p] * np.exp(-2j * np.pi * om * k / L))
            assert abs(S[om, s, p] - naive) <= tol * scale


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32], ids=["f64", "f32"])
def test_impulse_returns_block_column(tt, dtype):
    """m = e_(j0,p0) => d_i = F_{i-j0}[:,p0] for i >= j0, ~0 before (causality); adjoint with the
    impulse at the LAST step returns F_{N_t-1-j}[s0,:] (catches keeping the wrong half)."""
    w = workload("C1", 4, 64, 32, dtype)
    F = synth.block_column(w)
    Fn = F.numpy().astype(np.float64)
    N_t, N_d, N_m = F.shape
    tol = TOL[dtype]
    plan = tt.Plan(F.cuda())
    try:
        j0, p0 = 5, 17
        m = torch.zeros((N_t, N_m), dtype=dtype); m[j0, p0] = 1.0
        d = plan.matvec(m.cuda()).cpu().numpy().astype(np.float64)
        expect = np.zeros((N_t, N_d)); expect[j0:] = Fn[: N_t - j0, :, p0]
        assert np.linalg.norm(d - expect) <= tol * np.linalg.norm(expect)
        assert np.abs(d[:j0]).max() <= tol * np.abs(Fn).max()
        i0, s0 = N_t - 1, 2
        dd = torch.zeros((N_t, N_d), dtype=dtype); dd[i0, s0] = 1.0
        mm = plan.rmatvec(dd.cuda()).cpu().numpy().astype(np.float64)
        expect = Fn[::-1][:, s0, :]  # m'_j = F_{i0-j}[s0,:]
        assert np.linalg.norm(mm - expect) <= tol * np.linalg.norm(expect)
    finally:
        plan.close()


# Transform lengths that walk every kind of pass sequence of the FFT kernels: no pass (1), a single pass (first = last:
# 2, 3, 4, 8, 25), an odd last radix (9, 27, 125, 343, 625), an even one whose upper output half is dead code
# (686 = 7*7*7*2, 1000, 1024), and three- and four-pass plans; 37 series leave a ragged last tile of 5.
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32], ids=["f64", "f32"])
@pytest.mark.parametrize("N_t", [2, 3, 4, 8, 9, 25, 27, 125, 343, 625, 686, 1000, 1024])
def test_fft_pass_sequences_vs_oracle(tt, N_t, dtype):
    w = workload("C2", 2, 37, N_t, dtype)
    F, m, d = inputs(w)
    plan = tt.Plan(F.cuda())
    try:
        got_d = plan.matvec(m.cuda()).cpu().numpy()
        got_m = plan.rmatvec(d.cuda()).cpu().numpy()
    finally:
        plan.close()
    orc = op if N_t * N_t * 2 * 37 < 2e6 else ob
    tol = TOL[dtype]
    assert rel(got_d, orc.matvec(F.numpy(), m.numpy())) <= tol
    assert rel(got_m, orc.rmatvec(F.numpy(), d.numpy())) <= tol


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32], ids=["f64", "f32"])
def test_adjoint_identity_linearity_shift_on_gpu(tt, dtype):
    w = workload("C5", 6, 777, 60, dtype)
    F, m, d = inputs(w)
    tol = TOL[dtype]
    plan = tt.Plan(F.cuda())
    try:
        mc, dc = m.cuda(), d.cuda()
        Fm = plan.matvec(mc).double()
        Ftd = plan.rmatvec(dc).double()
        lhs = float((Fm * dc.double()).sum()); rhs = float((mc.double() * Ftd).sum())
        assert abs(lhs - rhs) <= tol * float(Fm.norm() * dc.double().norm())
        # linearity
        m2 = synth.vector_m(w.scaled(seed=w.seed + 100), k_rhs=1).cuda()
        comb = plan.matvec((2.0 * mc - 3.0 * m2)).double()
        sep = 2.0 * Fm - 3.0 * plan.matvec(m2).double()
        assert float((comb - sep).norm()) <= tol * float(sep.norm())
        # shift equivariance (block Toeplitz): delaying m by tau delays d by tau
        tau = 7
        ms = torch.zeros_like(mc); ms[tau:] = mc[:-tau]
        ds = plan.matvec(ms).double()
        assert float((ds[tau:] - Fm[:-tau]).norm()) <= tol * float(Fm.norm())
        assert float(ds[:tau].abs().max()) <= tol * float(Fm.abs().max())
        # normal operator: <m, F^T F m> = |F m|^2
        n = plan.normal(mc).double()
        assert abs(float((mc.double() * n).sum()) - float(Fm.norm() ** 2)) <= tol * float(Fm.norm() ** 2)
    finally:
        plan.close()


def test_exact_integer_case(tt):
    """Small-integer F and m: every sum is exact in fp64, so the fp64 GPU result rounds to the exact integers."""
    rng = np.random.default_rng(5)
    F = torch.from_numpy(rng.integers(-3, 4, size=(16, 3, 50)).astype(np.float64))
    m = torch.from_numpy(rng.integers(-3, 4, size=(16, 50)).astype(np.float64))
    plan = tt.Plan(F.cuda())
    try:
        d = plan.matvec(m.cuda()).cpu().numpy()
    finally:
        plan.close()
    ref = op.matvec(F.numpy(), m.numpy())
    assert np.array_equal(np.rint(d), ref)
    assert np.abs(d - ref).max() < 1e-9


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32], ids=["f64", "f32"])
@pytest.mark.parametrize("k", [1, 3, 8, 32])
def test_batched_columns_equal_oracle(tt, dtype, k):
    w = workload("C4", 6, 300, 32, dtype)
    F = synth.block_column(w)
    M = synth.vector_m(w, k_rhs=k).reshape(w.N_t, w.N_m, k)
    D = synth.vector_d(w, k_rhs=k).reshape(w.N_t, w.N_d, k)
    plan = tt.Plan(F.cuda(), k_max=32)
    try:
        gd = plan.matvec_batched(M.cuda()).cpu().numpy()
        gm = plan.rmatvec_batched(D.cuda()).cpu().numpy()
    finally:
        plan.close()
    rd = op.matvec(F.numpy(), M.numpy())
    rm = op.rmatvec(F.numpy(), D.numpy())
    tol = TOL[dtype]
    for r in range(k):
        assert rel(gd[..., r], rd[..., r]) <= tol
        assert rel(gm[..., r], rm[..., r]) <= tol


@pytest.mark.parametrize("N_d,N_m,N_t,k", [(70, 5000, 16, 5), (130, 4500, 12, 33), (64, 8192, 64, 32),
                                            (9, 257, 20, 17), (3, 31, 6, 40)])
def test_dmma_gemm_path_shapes(tt, N_d, N_m, N_t, k):
    """fp64 k-RHS path (batched FFTs + per-frequency DMMA GEMMs): ragged sensor blocks (N_d not a multiple
    of 64, > 64), several p-splits, N_m not a multiple of 256, k not a multiple of 8 and k > 32."""
    w = workload("C4", N_d, N_m, N_t, torch.float64)
    F = synth.block_column(w)
    M = synth.vector_m(w, k_rhs=k)
    D = synth.vector_d(w, k_rhs=k)
    plan = tt.Plan(F.cuda(), k_max=k)
    try:
        gd = plan.matvec_batched(M.cuda()).cpu().numpy()
        gm = plan.rmatvec_batched(D.cuda()).cpu().numpy()
        one_d = plan.matvec(M[..., 1].contiguous().cuda()).cpu().numpy()
        one_m = plan.rmatvec(D[..., 1].contiguous().cuda()).cpu().numpy()
    finally:
        plan.close()
    cols = sorted({0, 1, k // 2, k - 1})
    for r in cols:
        assert rel(gd[..., r], ob.matvec(F.numpy(), M[..., r].contiguous().numpy())) <= 1e-12
        assert rel(gm[..., r], ob.rmatvec(F.numpy(), D[..., r].contiguous().numpy())) <= 1e-12
    # column r of the batched result equals the single-vector result on column r (include/tt.h)
    assert rel(gd[..., 1], one_d) <= 1e-13 and rel(gm[..., 1], one_m) <= 1e-13


@pytest.mark.parametrize("N_d,N_m,N_t,k", [(70, 5000, 16, 5), (130, 4500, 12, 33), (64, 8192, 64, 32), (49, 2049, 20, 32),
                                            (9, 257, 20, 17), (3, 31, 6, 40), (200, 700, 8, 7), (16, 3001, 10, 2)])
@pytest.mark.parametrize("layout", [0, 1])
def test_fp32_gemm_path_shapes(tt, N_d, N_m, N_t, k, layout):
    """fp32 k-RHS path (batched FFTs + per-frequency complex64 FMA GEMMs, tt_gemm32.cu): every sensor-tile variant
    (N_d <= 32, <= 64, > 64, > 128), ragged tiles, several p-splits, odd N_m, odd k, k > 32, both layouts."""
    w = workload("C4", N_d, N_m, N_t, torch.float32)
    F = synth.block_column(w)
    M = synth.vector_m(w, k_rhs=k)
    D = synth.vector_d(w, k_rhs=k)
    lay = (lambda t: t.permute(2, 1, 0).contiguous()) if layout == 1 else (lambda t: t)
    unlay = (lambda t: t.permute(2, 1, 0)) if layout == 1 else (lambda t: t)
    plan = tt.Plan(F.cuda(), layout=layout, k_max=k)
    try:
        gd = unlay(plan.matvec_batched(lay(M).cuda())).cpu().numpy()
        gm = unlay(plan.rmatvec_batched(lay(D).cuda())).cpu().numpy()
    finally:
        plan.close()
    for r in sorted({0, 1, k // 2, k - 1}):
        assert rel(gd[..., r], ob.matvec(F.numpy(), M[..., r].contiguous().numpy())) <= 1e-5
        assert rel(gm[..., r], ob.rmatvec(F.numpy(), D[..., r].contiguous().numpy())) <= 1e-5


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32], ids=["f64", "f32"])
def test_space_major_layout(tt, dtype):
    """TT_SPACE_MAJOR (time contiguous, the 'm (64x32)' shapes of BASELINE.json) gives the same numbers."""
    w = workload("C1", 4, 64, 32, dtype)
    F, m, d = inputs(w)
    plan = tt.Plan(F.cuda(), layout=tt.TT_SPACE_MAJOR, k_max=2)
    try:
        gd = plan.matvec(m.t().contiguous().cuda()).cpu().numpy().T
        gm = plan.rmatvec(d.t().contiguous().cuda()).cpu().numpy().T
        M = synth.vector_m(w, k_rhs=2)                      # [N_t, N_m, 2]
        gD = plan.matvec_batched(M.permute(2, 1, 0).contiguous().cuda()).cpu().numpy()  # [2, N_d, N_t]
    finally:
        plan.close()
    tol = TOL[dtype]
    assert rel(gd, op.matvec(F.numpy(), m.numpy())) <= tol
    assert rel(gm, op.rmatvec(F.numpy(), d.numpy())) <= tol
    rD = op.matvec(F.numpy(), M.numpy())
    assert rel(np.transpose(gD, (2, 1, 0)), rD) <= tol


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32], ids=["f64", "f32"])
def test_host_vector_calls(tt, dtype):
    w = workload("C3", 5, 1200, 40, dtype)
    F, m, d = inputs(w)
    plan = tt.Plan(F.cuda())
    try:
        mh, dh = m.pin_memory(), d.pin_memory()
        d_out = torch.empty_like(d).pin_memory()
        m_out = torch.empty_like(m).pin_memory()
        n_out = torch.empty_like(m).pin_memory()
        tt.tt_matvec_host(plan.handle, mh, d_out)
        tt.tt_rmatvec_host(plan.handle, dh, m_out)
        tt.tt_normal_host(plan.handle, mh, n_out)
        torch.cuda.synchronize()
        assert torch.equal(d_out, plan.matvec(m.cuda()).cpu())
        assert torch.equal(m_out, plan.rmatvec(d.cuda()).cpu())
        assert torch.equal(n_out, plan.normal(m.cuda()).cpu())
    finally:
        plan.close()


@pytest.mark.parametrize("n_ranges,growth", [(0, 0), (3, 0), (8, 160), (8, 60), (5, 100), (32, 400), (1, 0)])
def test_host_vector_calls_graded_ranges(tt, n_ranges, growth):
    """The pipelined *_host calls cut the parameter axis into a geometric sequence of ranges (tt_api.cu host_ranges): whatever
    the number of ranges and their ratio, and in either direction of the sequence, the result is the device call's bit for bit
    (N_d = 20 and N_d = 90: the planner's own choice is 8 graded ranges for the first, 16 equal ones for the second; 9 units of
    2048 parameters to distribute)."""
    for N_d in (20, 90):
        w = workload("C3", N_d, 16384 + 7, 40, torch.float32)
        F, m, d = inputs(w)
        plan = tt.Plan(F.cuda())
        try:
            ref_d, ref_m, ref_n = plan.matvec(m.cuda()).cpu(), plan.rmatvec(d.cuda()).cpu(), plan.normal(m.cuda()).cpu()
            tt.tt_debug_set("host_chunks", n_ranges)
            tt.tt_debug_set("host_growth", growth)
            mh, dh = m.pin_memory(), d.pin_memory()
            d_out, m_out, n_out = torch.empty_like(d).pin_memory(), torch.empty_like(m).pin_memory(), torch.empty_like(m).pin_memory()
            tt.tt_matvec_host(plan.handle, mh, d_out)
            tt.tt_rmatvec_host(plan.handle, dh, m_out)
            tt.tt_normal_host(plan.handle, mh, n_out)
            torch.cuda.synchronize()
            assert torch.equal(d_out, ref_d) and torch.equal(m_out, ref_m) and torch.equal(n_out, ref_n)
        finally:
            tt.tt_debug_set("host_chunks", 0)
            tt.tt_debug_set("host_growth", 0)
            plan.close()


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32], ids=["f64", "f32"])
@pytest.mark.parametrize("base,N_d,N_m,N_t", SHAPES)
def test_rmatvec_producer_consumer_mode_is_bit_identical(tt, base, N_d, N_m, N_t, dtype):
    """F^T d with B3 as a concurrent consumer of B2 (tt_api.cu run_rmatvec: group-major B2 grid with per-tile counters,
    persistent consumer CTAs on the plan's stream, spectrum handed over in the L2 and dropped there, clean-up launch for
    tiles the consumers did not reach) against the plain two-launch sequence, forced on at every test shape - the planner
    itself only takes it from ~14 GB of spectrum: tt_rmatvec and tt_normal bit for bit, for small and large groups, few
    and many consumers, with and without the discard.  (Shapes whose FFT tile is not a whole number of 128-byte lines
    fall back to the two launches inside the library: equal by construction.)"""
    w = workload(base, N_d, N_m, N_t, dtype)
    F, m, d = inputs(w)
    plan = tt.Plan(F.cuda())
    try:
        tt.tt_debug_set("l2r_mb", 0)
        ref_m, ref_n = plan.rmatvec(d.cuda()), plan.normal(m.cuda())
        for mb, ctas, discard in ((1, 3, 1), (1, 40, 1), (64, 7, 1), (2, 148, 0)):
            tt.tt_debug_set("l2r_mb", mb)
            tt.tt_debug_set("l2r_ctas", ctas)
            tt.tt_debug_set("l2r_discard", discard)
            for _ in range(2):
                assert torch.equal(plan.rmatvec(d.cuda()), ref_m), (mb, ctas, discard)
                assert torch.equal(plan.normal(m.cuda()), ref_n), (mb, ctas, discard)
    finally:
        tt.tt_debug_set("l2r_mb", -1)
        tt.tt_debug_set("l2r_ctas", 0)
        tt.tt_debug_set("l2r_discard", 1)
        plan.close()


def test_rmatvec_producer_consumer_mode_survives_serialised_kernels(tt):
    """The consumer kernel is an accelerator, not a dependency: when kernels cannot run side by side (here
    CUDA_LAUNCH_BLOCKING=1 in a child process; a profiler that serialises launches does the same) the consumers give up
    after 50 ms without a producer, and the regular B3 launch behind B2 transforms every tile - same bits, only slower."""
    import os
    import subprocess
    import sys
    code = (
        "import torch, synth\n"
        "from paper_2501_14911_b200 import binding as tt\n"
        "w = synth.CONFIGS['C3'].scaled(N_d=7, N_m=3000, N_t=400)\n"
        "F, d = synth.block_column(w).cuda(), synth.vector_d(w, k_rhs=1).cuda()\n"
        "plan = tt.Plan(F)\n"
        "tt.tt_debug_set('l2r_mb', 0)\n"
        "ref = plan.rmatvec(d)\n"
        "tt.tt_debug_set('l2r_mb', 1); tt.tt_debug_set('l2r_ctas', 16)\n"
        "out = plan.rmatvec(d)\n"
        "torch.cuda.synchronize()\n"
        "assert torch.equal(out, ref)\n"
        "print('serialised ok')\n"
    )
    env = dict(os.environ, CUDA_LAUNCH_BLOCKING="1")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    res = subprocess.run([sys.executable, "-c", code], cwd=root, env=env, capture_output=True, text=True, timeout=600)
    assert res.returncode == 0 and "serialised ok" in res.stdout, res.stdout + res.stderr


def test_error_codes(tt):
    import ctypes
    L = tt.lib()
    F = torch.zeros((11, 2, 3), dtype=torch.float64, device="cuda")
    out = ctypes.c_void_p()
    st = torch.cuda.current_stream().cuda_stream

    def create(N_d, N_m, N_t, dtype=tt.TT_F64, layout=0, k=1, ptr=F.data_ptr()):
        return L.tt_plan_create(ctypes.byref(out), N_d, N_m, N_t, dtype, layout, k, ptr, st)

    assert tt.tt_status_string(create(2, 3, 11)) == "TT_ERR_UNSUPPORTED_NT"
    assert tt.tt_status_string(create(2, 3, 4000)) == "TT_ERR_UNSUPPORTED_NT"
    assert tt.tt_status_string(create(0, 3, 8)) == "TT_ERR_SHAPE"
    assert tt.tt_status_string(create(2, -1, 8)) == "TT_ERR_SHAPE"
    assert tt.tt_status_string(create(2, 3, 8, dtype=7)) == "TT_ERR_DTYPE"
    assert tt.tt_status_string(create(2, 3, 8, layout=9)) == "TT_ERR_LAYOUT"
    assert tt.tt_status_string(create(2, 3, 8, k=0)) == "TT_ERR_K"
    assert tt.tt_status_string(create(2, 3, 8, ptr=None)) == "TT_ERR_NULL"
    assert out.value is None
    plan = tt.Plan(F[:10].contiguous(), k_max=2)
    try:
        v = torch.zeros((10, 3), dtype=torch.float64, device="cuda")
        assert tt.tt_status_string(L.tt_normal(plan.handle, v.data_ptr(), v.data_ptr(), st)) == "TT_ERR_ALIAS"
        assert tt.tt_status_string(L.tt_matvec(plan.handle, None, v.data_ptr(), st)) == "TT_ERR_NULL"
        assert tt.tt_status_string(L.tt_matvec_batched(plan.handle, 3, v.data_ptr(), v.data_ptr(), st)) == "TT_ERR_K"
        assert plan.device_bytes > 0
    finally:
        plan.close()
    L.tt_plan_destroy(None)  # NULL-safe


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32], ids=["f64", "f32"])
@pytest.mark.parametrize("layout", [0, 1])
def test_normal_batched(tt, dtype, layout):
    """tt_normal_batched: F^T (F M) for k columns, each column equal to the single-vector normal operator of the oracle."""
    N_d, N_m, N_t, k = 5, 700, 24, 6
    w = workload("C4", N_d, N_m, N_t, dtype)
    F = synth.block_column(w)
    M = synth.vector_m(w, k_rhs=k)
    lay = (lambda t: t.permute(2, 1, 0).contiguous()) if layout == 1 else (lambda t: t)
    unlay = (lambda t: t.permute(2, 1, 0)) if layout == 1 else (lambda t: t)
    plan = tt.Plan(F.cuda(), layout=layout, k_max=8)
    try:
        Md = lay(M).cuda()
        out = torch.empty_like(Md)
        tt.tt_normal_batched(plan.handle, k, Md, out)
        got = unlay(out).cpu().numpy()
        with pytest.raises(tt.TTError):
            tt.tt_normal_batched(plan.handle, k, Md, Md)
        with pytest.raises(tt.TTError):
            tt.tt_normal_batched(plan.handle, 9, Md, out)
    finally:
        plan.close()
    for r in range(k):
        assert rel(got[..., r], ob.rmatvec(F.numpy(), ob.matvec(F.numpy(), M[..., r].contiguous().numpy()))) <= TOL[dtype]
