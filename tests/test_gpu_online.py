"""GPU parity for the online phase: the triangular solves with the Cholesky
factor of K, the assembly of K = Gamma_noise + F G* and the MAP point of eq (4.13), called through the
C ABI and compared with oracle/online_plain.py on the same seeded inputs.

Tolerances (relative L2 over the whole output; DESIGN.md section 11 derives them):
  * triangular solves, fp64: 1e-12 on factors whose diagonal blocks are well conditioned;
  * K: 1e-12 (fp64 plans) / 1e-5 (fp32 plans) relative to ||K||_F  (n matvec pairs, the matvec bar);
  * m_map with the ORACLE's factor L uploaded (so that only the online arithmetic is compared):
      gain form  G* K^{-1} d_obs            : matvec bar (1e-12 / 1e-5) + 8 u64 kappa(K) for the fp64 solve;
      paper form (I - G* K^{-1} F) G* y     : rounding of a = G* y and b = F a is amplified by the solve,
                                              bound  8 u kappa(K)  with u the unit roundoff of the plan dtype.
"""
import numpy as np
import pytest
import torch

from oracle import online_plain as oo
from oracle import toeplitz_plain as op
import synth
from tests.inputs_online import gstar_column

pytestmark = pytest.mark.gpu

U = {torch.float64: 1.1e-16, torch.float32: 6.0e-8}
BAR = {torch.float64: 1e-12, torch.float32: 1e-5}


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


def random_factor(n, seed):
    """A lower-triangular matrix with the profile of a Cholesky factor: positive diagonal, decaying off-diagonal."""
    rng = np.random.default_rng(seed)
    L = np.tril(rng.standard_normal((n, n))) / np.sqrt(max(n, 1))
    L[np.arange(n), np.arange(n)] = rng.uniform(1.0, 2.0, n)
    return L


# ---------------------------------------------------------------------------- triangular solves
@pytest.mark.parametrize("n", [1, 2, 63, 64, 65, 130, 200, 1000, 4097])
@pytest.mark.parametrize("where", ["device", "host"])
def test_trsv_and_solve(tt, n, where):
    L = random_factor(n, n)
    b = np.random.default_rng(n + 1).standard_normal(n)
    Lt = torch.from_numpy(L)
    # garbage in the upper triangle must be ignored
    Lt = Lt + torch.triu(torch.full((n, n), 7.0, dtype=torch.float64), diagonal=1)
    chol = tt.Chol(Lt.cuda() if where == "device" else Lt)
    try:
        bd = torch.from_numpy(b).cuda()
        y = chol.trsv(bd).cpu().numpy()
        x = chol.trsv(bd, transposed=True).cpu().numpy()
        z = chol.solve(bd).cpu().numpy()
        z2 = chol.solve(bd).cpu().numpy()
    finally:
        chol.close()
    assert rel(y, oo.forward_substitution(L, b)) <= 1e-12
    assert rel(x, oo.back_substitution_T(L, b)) <= 1e-12
    assert rel(z, oo.chol_solve(L, b)) <= 1e-12
    assert np.array_equal(z, z2)            # fixed summation order: bit-reproducible


def test_trsv_pitch_alias_and_errors(tt):
    n = 150
    L = random_factor(n, 5)
    big = torch.zeros((n, n + 9), dtype=torch.float64)
    big[:, :n] = torch.from_numpy(L)
    chol = tt.Chol(big.cuda()[:, :n])                      # row pitch n + 9
    try:
        b = torch.from_numpy(np.random.default_rng(1).standard_normal(n)).cuda()
        ref = oo.chol_solve(L, b.cpu().numpy())
        x = b.clone()
        tt.tt_chol_solve(chol.handle, x, x)                # in place
        assert rel(x.cpu().numpy(), ref) <= 1e-12
        assert chol.device_bytes >= 8 * n * n // 2
    finally:
        chol.close()
    bad = torch.from_numpy(L.copy())
    bad[77, 77] = 0.0
    with pytest.raises(tt.TTError) as ei:
        tt.Chol(bad.cuda())
    assert ei.value.status == -11                           # TT_ERR_NOT_SPD
    bad[77, 77] = float("nan")
    with pytest.raises(tt.TTError):
        tt.Chol(bad)
    with pytest.raises(tt.TTError):
        tt.tt_chol_create(0, torch.zeros(1, dtype=torch.float64).cuda())


def test_trsv_nan_rhs_terminates(tt):
    # a NaN right-hand side must flow through (and not be mistaken for the 'not yet computed' pattern)
    n = 300
    chol = tt.Chol(torch.from_numpy(random_factor(n, 9)).cuda())
    try:
        b = torch.zeros(n, dtype=torch.float64)
        b[5] = float("nan")
        sentinel = np.array([0x7FF4A5A5DEADBEEF], dtype=np.uint64).view(np.float64)[0]
        b[70] = float(sentinel)
        x = chol.solve(b.cuda())
        torch.cuda.synchronize()
        assert torch.isnan(x).any()
    finally:
        chol.close()


# ---------------------------------------------------------------------------- K and the MAP point
def online_inputs(N_d, N_m, N_t, dtype):
    w = synth.CONFIGS["P5"].scaled(N_d=N_d, N_m=N_m, N_t=N_t, dtype=dtype)
    F = synth.block_column(w)
    G = gstar_column(w, F)
    nv = synth.noise_var(w)
    d_obs = synth.vector_d(w, k_rhs=1)
    return w, F, G, nv, d_obs


ONLINE_SHAPES = [(3, 40, 12), (6, 400, 50), (5, 1000, 35), (1, 64, 20), (4, 2100, 16)]


@pytest.mark.parametrize("N_d,N_m,N_t", ONLINE_SHAPES)
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("k_max", [1, 8, 16, 32])      # 16, 32: the fp32 groups take the tcgen05 GEMMs, the ragged last group the FMA ones
def test_assemble_K(tt, N_d, N_m, N_t, dtype, k_max):
    w, F, G, nv, _ = online_inputs(N_d, N_m, N_t, dtype)
    K_ref = oo.assemble_K(F.numpy(), G.numpy(), nv.numpy())
    pF, pG = tt.Plan(F.cuda(), k_max=k_max), tt.Plan(G.cuda(), k_max=k_max)
    try:
        K = tt.assemble_K(pF, pG, nv.cuda()).cpu().numpy()
        n = N_d * N_t
        part = torch.full((n, n + 3), -1.0, dtype=torch.float64, device="cuda")      # a column range, pitched output
        c0, nc = n // 3, min(n - n // 3, 11)
        tt.tt_assemble_K(pF.handle, pG.handle, nv.cuda(), c0, nc, part, n + 3)
        part = part.cpu().numpy()
    finally:
        pF.close(); pG.close()
    assert rel(K, K_ref) <= BAR[dtype]
    assert rel(K, K.T) <= 2 * BAR[dtype]
    assert rel(part[:, c0:c0 + nc], K_ref[:, c0:c0 + nc]) <= BAR[dtype]
    assert (part[:, :c0] == -1.0).all() and (part[:, c0 + nc:] == -1.0).all()


# n = N_t N_d spans one tile (36), ragged second tiles (300, 350), the order of a diagonal block larger than a tile (N_d = 150);
# N_m spans less than one shared-memory stage (5), ragged stages (1000, 2100) and more than one fp32 chunk of 8192 (9000).
DIRECT_SHAPES = ONLINE_SHAPES + [(7, 9000, 30), (3, 33, 100), (150, 70, 2), (2, 5, 3), (1, 1, 1), (10, 257, 35)]


@pytest.mark.parametrize("N_d,N_m,N_t", DIRECT_SHAPES)
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_assemble_K_direct(tt, N_d, N_m, N_t, dtype):
    """tt_assemble_K_direct (one GEMM of the block columns + running sums down the block diagonals) against the oracle's
    column-by-column K = Gamma_noise + F G* (PAPER.md:296, 306)."""
    w, F, G, nv, _ = online_inputs(N_d, N_m, N_t, dtype)
    K_ref = oo.assemble_K(F.numpy(), G.numpy(), nv.numpy())
    n = N_d * N_t
    buf = torch.full((n, n + 3), -1.0, dtype=torch.float64, device="cuda")             # pitched output
    tt.tt_assemble_K_direct(F.cuda(), G.cuda(), nv.cuda(), N_d, N_m, N_t, tt.TT_F32 if dtype == torch.float32 else tt.TT_F64,
                            buf, n + 3)
    buf = buf.cpu().numpy()
    K = buf[:, :n]
    assert (buf[:, n:] == -1.0).all()
    assert rel(K, K_ref) <= BAR[dtype]
    assert np.array_equal(K, K.T)                                                      # the upper triangle is a copy
    # the noise sits on the diagonal only: the same call with twice the noise moves exactly the diagonal
    K2 = tt.assemble_K_direct(F.cuda(), G.cuda(), (2 * nv).cuda()).cpu().numpy()
    off = ~np.eye(n, dtype=bool)
    assert np.array_equal(K2[off], K[off])
    assert np.allclose(np.diag(K2) - np.diag(K), nv.numpy().reshape(n).astype(np.float64), rtol=1e-6, atol=0)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_assemble_K_direct_agrees_with_column_by_column(tt, dtype):
    N_d, N_m, N_t = 6, 700, 40
    w, F, G, nv, _ = online_inputs(N_d, N_m, N_t, dtype)
    pF, pG = tt.Plan(F.cuda(), k_max=8), tt.Plan(G.cuda(), k_max=8)
    try:
        K_cols = tt.assemble_K(pF, pG, nv.cuda()).cpu().numpy()
    finally:
        pF.close(); pG.close()
    K_dir = tt.assemble_K_direct(F.cuda(), G.cuda(), nv.cuda()).cpu().numpy()
    assert rel(K_dir, K_cols) <= 2 * BAR[dtype]


def test_assemble_K_direct_validation(tt):
    F = torch.zeros((4, 2, 8), dtype=torch.float32, device="cuda")
    nv = torch.ones((4, 2), dtype=torch.float32, device="cuda")
    K = torch.zeros((8, 8), dtype=torch.float64, device="cuda")
    L = tt.lib()
    st = torch.cuda.current_stream().cuda_stream
    assert L.tt_assemble_K_direct(None, F.data_ptr(), nv.data_ptr(), 2, 8, 4, tt.TT_F32, K.data_ptr(), 8, st) == -1      # TT_ERR_NULL
    assert L.tt_assemble_K_direct(F.data_ptr(), F.data_ptr(), nv.data_ptr(), 2, 8, 4, 7, K.data_ptr(), 8, st) == -3   # TT_ERR_DTYPE
    assert L.tt_assemble_K_direct(F.data_ptr(), F.data_ptr(), nv.data_ptr(), 2, 8, 4, tt.TT_F32, K.data_ptr(), 7, st) == -2   # TT_ERR_SHAPE (ldk < n)
    assert L.tt_assemble_K_direct(F.data_ptr(), F.data_ptr(), nv.data_ptr(), 0, 8, 4, tt.TT_F32, K.data_ptr(), 8, st) == -2   # TT_ERR_SHAPE


@pytest.mark.parametrize("N_d,N_m,N_t", ONLINE_SHAPES)
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("layout", [0, 1])
def test_map_point(tt, N_d, N_m, N_t, dtype, layout):
    w, F, G, nv, d_obs = online_inputs(N_d, N_m, N_t, dtype)
    Fn, Gn, nvn, dn = F.numpy(), G.numpy(), nv.numpy(), d_obs.numpy()
    K = oo.assemble_K(Fn, Gn, nvn)
    L = oo.cholesky(K)
    m_ref = oo.map_point(Fn, Gn, nvn, L, dn)
    ev = np.linalg.eigvalsh(K)
    kappa = ev[-1] / ev[0]
    pF, pG = tt.Plan(F.cuda(), layout=layout), tt.Plan(G.cuda(), layout=layout)
    chol = tt.Chol(torch.from_numpy(L).cuda())
    lay = (lambda t: t.t().contiguous()) if layout == 1 else (lambda t: t)
    unlay = (lambda t: t.t()) if layout == 1 else (lambda t: t)
    mp = tt.MapInference(pF, pG, chol, lay(nv).cuda())
    try:
        m_paper = unlay(mp.infer(lay(d_obs).cuda(), tt.TT_MAP_PAPER)).cpu().numpy()
        m_gain = unlay(mp.infer(lay(d_obs).cuda(), tt.TT_MAP_GAIN)).cpu().numpy()
        mg = tt.MapInference(None, pG, chol, lay(nv).cuda())       # gain form needs no F
        m_gain2 = unlay(mg.infer(lay(d_obs).cuda(), tt.TT_MAP_GAIN)).cpu().numpy()
        with pytest.raises(tt.TTError):
            mg.infer(lay(d_obs).cuda(), tt.TT_MAP_PAPER)
        mg.close()
    finally:
        mp.close(); chol.close(); pF.close(); pG.close()
    e_gain, e_paper = rel(m_gain, m_ref), rel(m_paper, m_ref)
    print(f"map {N_d}x{N_m}x{N_t} {dtype} layout {layout}: kappa(K) {kappa:.1f}  gain {e_gain:.2e}  paper {e_paper:.2e}")
    assert e_gain <= BAR[dtype] + 8 * U[torch.float64] * kappa
    assert e_paper <= 8 * U[dtype] * kappa + BAR[dtype]
    assert np.array_equal(m_gain, m_gain2)
    # the MAP point solves eq (2.12): F* Gn^{-1} (d - F m) = Gamma_prior^{-1} m, checked through the oracle operators
    g = synth.prior_gamma(w).numpy()
    lhs = op.rmatvec(Fn, (dn - op.matvec(Fn, m_gain)) / nvn)
    assert rel(lhs, m_gain / g[None, :]) <= 1e3 * (BAR[dtype] + 8 * U[dtype] * kappa)


def test_map_mismatch_errors(tt):
    w, F, G, nv, d_obs = online_inputs(3, 40, 12, torch.float64)
    pF, pG = tt.Plan(F.cuda()), tt.Plan(G[:, :2].contiguous().cuda())
    chol = tt.Chol(torch.eye(7, dtype=torch.float64).cuda())
    try:
        with pytest.raises(tt.TTError) as ei:
            tt.MapInference(pF, pG, chol, nv.cuda())
        assert ei.value.status == -12                       # TT_ERR_MISMATCH (plans)
        with pytest.raises(tt.TTError) as ei:
            tt.MapInference(None, pF, chol, nv.cuda())
        assert ei.value.status == -12                       # factor order != N_d N_t
        with pytest.raises(tt.TTError):
            tt.assemble_K(pF, pG, nv.cuda())
    finally:
        chol.close(); pF.close(); pG.close()


def _guarded(shape, dtype):
    """An output tensor surrounded by 4096-element canary zones (compute-sanitizer is not available on the pool)."""
    n = int(np.prod(shape))
    buf = torch.full((n + 8192,), -7.0, dtype=dtype, device="cuda")
    return buf, buf[4096:4096 + n].view(shape)


def test_outputs_stay_inside_their_buffers(tt):
    """Every kernel that writes a caller's vector, at ragged shapes: the bytes before and after the output are untouched."""
    for dtype in (torch.float32, torch.float64):
        N_d, N_m, N_t, k = 5, 1001, 35, 7
        w = synth.CONFIGS["P5"].scaled(N_d=N_d, N_m=N_m, N_t=N_t, dtype=dtype)
        F = synth.block_column(w)
        G = gstar_column(w, F)
        nv = synth.noise_var(w)
        L = oo.cholesky(oo.assemble_K(F.numpy(), G.numpy(), nv.numpy()))
        pF, pG = tt.Plan(F.cuda(), k_max=k), tt.Plan(G.cuda(), k_max=k)
        chol = tt.Chol(torch.from_numpy(L).cuda())
        mp = tt.MapInference(pF, pG, chol, nv.cuda())
        bufs = []
        try:
            m, d = synth.vector_m(w, k_rhs=1).cuda(), synth.vector_d(w, k_rhs=1).cuda()
            M, D = synth.vector_m(w, k_rhs=k).cuda(), synth.vector_d(w, k_rhs=k).cuda()
            for shape, call in (((N_t, N_d), lambda o: tt.tt_matvec(pF.handle, m, o)),
                                ((N_t, N_m), lambda o: tt.tt_rmatvec(pF.handle, d, o)),
                                ((N_t, N_m), lambda o: tt.tt_normal(pF.handle, m, o)),
                                ((N_t, N_d, k), lambda o: tt.tt_matvec_batched(pF.handle, k, M, o)),
                                ((N_t, N_m, k), lambda o: tt.tt_rmatvec_batched(pF.handle, k, D, o)),
                                ((N_t, N_m), lambda o: tt.tt_map_infer(mp.handle, tt.TT_MAP_PAPER, d, o)),
                                ((N_t, N_m), lambda o: tt.tt_map_infer(mp.handle, tt.TT_MAP_GAIN, d, o))):
                buf, out = _guarded(shape, dtype)
                call(out)
                bufs.append((buf, out.numel()))
            b64 = torch.randn(N_d * N_t, dtype=torch.float64, device="cuda")
            for tr in (None, False, True):
                buf, out = _guarded((N_d * N_t,), torch.float64)
                tt.tt_chol_solve(chol.handle, b64, out) if tr is None else tt.tt_chol_trsv(chol.handle, tr, b64, out)
                bufs.append((buf, out.numel()))
            torch.cuda.synchronize()
        finally:
            mp.close(); chol.close(); pF.close(); pG.close()
        for buf, n in bufs:
            assert (buf[:4096] == -7.0).all() and (buf[4096 + n:] == -7.0).all()
            assert torch.isfinite(buf[4096:4096 + n]).all()


def test_K_direct_fp32_slab_sums_meet_in_fp64(tt):
    """The fp32 path of tt_assemble_K_direct walks the parameter axis in slabs (8192 parameters by default) whose sums meet in fp64 in K:
    with the developer knob `kd_slab` the same call takes 1, 3 and 32 slabs (the last one ragged: N_m = 2021 is not a multiple of the
    32-parameter K-block, and the rows of the block columns are not 16-byte aligned) - every variant within the bar of the oracle, and
    close to each other (the slab boundaries only change where fp32 running sums are handed to fp64)."""
    N_d, N_m, N_t = 6, 2021, 30
    w = synth.CONFIGS["P5"].scaled(N_d=N_d, N_m=N_m, N_t=N_t, dtype=torch.float32)
    F = synth.block_column(w)
    G = gstar_column(w, F)
    nv = synth.noise_var(w)
    ref = oo.assemble_K(F.numpy(), G.numpy(), nv.numpy())
    got = {}
    try:
        for slab in (0, 704, 64):
            tt.tt_debug_set("kd_slab", slab)
            got[slab] = tt.assemble_K_direct(F.cuda(), G.cuda(), nv.cuda()).cpu().numpy()
    finally:
        tt.tt_debug_set("kd_slab", 0)
    for slab, K in got.items():
        assert rel(K, ref) <= 1e-5, (slab, rel(K, ref))
        assert np.array_equal(K, K.T)
    assert rel(got[64], got[0]) <= 2e-6 and rel(got[704], got[0]) <= 2e-6


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_K_direct_stays_inside_its_matrix(tt, dtype):
    """tt_assemble_K_direct (fp32: the tcgen05 kernel, whose 128 x 256 tiles overhang a ragged n on both sides; fp64: DMMA)
    into a matrix with a row pitch larger than n, canary zones before and after: the pad columns of every row and the zones
    keep their values, every entry of K is written."""
    N_d, N_m, N_t = 7, 333, 41                       # n = 287: two tile rows, two tile columns, both ragged
    w = synth.CONFIGS["P5"].scaled(N_d=N_d, N_m=N_m, N_t=N_t, dtype=dtype)
    F = synth.block_column(w)
    G = gstar_column(w, F)
    nv = synth.noise_var(w)
    n, ldk = N_d * N_t, N_d * N_t + 37
    buf, K = _guarded((n, ldk), torch.float64)
    K[:, :n] = float("nan")
    tt.tt_assemble_K_direct(F.cuda(), G.cuda(), nv.cuda(), N_d, N_m, N_t, tt.TT_F32 if dtype == torch.float32 else tt.TT_F64, K, ldk)
    torch.cuda.synchronize()
    assert (buf[:4096] == -7.0).all() and (buf[4096 + n * ldk:] == -7.0).all()
    assert (K[:, n:] == -7.0).all()
    assert torch.isfinite(K[:, :n]).all()
    ref = oo.assemble_K(F.numpy(), G.numpy(), nv.numpy())
    assert rel(K[:, :n].cpu().numpy(), ref) <= (1e-12 if dtype == torch.float64 else 1e-5)


def test_map_two_halves_equal_the_whole(tt):
    """tt_map_infer_partial + tt_map_infer_finish (the split at the sharded path's all-reduce) == tt_map_infer."""
    from paper_2501_14911_b200 import sharded
    w, F, G, nv, d_obs = online_inputs(4, 700, 24, torch.float32)
    L = oo.cholesky(oo.assemble_K(F.numpy(), G.numpy(), nv.numpy()))
    pF, pG, chol = tt.Plan(F.cuda()), tt.Plan(G.cuda()), tt.Chol(torch.from_numpy(L).cuda())
    mp = tt.MapInference(pF, pG, chol, nv.cuda())
    try:
        whole = mp.infer(d_obs.cuda(), tt.TT_MAP_PAPER).cpu()
        a, b = mp.infer_partial(d_obs.cuda())
        halves = mp.infer_finish(b, a).cpu()
        sm = sharded.map_from_binding(mp)                      # world size 1: no collective
        via = sm.infer(d_obs.cuda()).cpu()
        gain = sm.infer(d_obs.cuda(), gain_form=True).cpu()
        ref_gain = mp.infer(d_obs.cuda(), tt.TT_MAP_GAIN).cpu()
    finally:
        mp.close(); chol.close(); pF.close(); pG.close()
    assert torch.equal(whole, halves) and torch.equal(whole, via) and torch.equal(gain, ref_gain)


def test_apply_calls_are_cuda_graph_capturable(tt):
    """No allocation, no host synchronisation after plan creation: the whole online step (and the plain matvec pair)
    can be captured once in a CUDA graph and replayed - what a launch-bound small problem (C1: 7 launches) wants."""
    w, F, G, nv, d_obs = online_inputs(4, 64, 32, torch.float64)
    L = oo.cholesky(oo.assemble_K(F.numpy(), G.numpy(), nv.numpy()))
    pF, pG, chol = tt.Plan(F.cuda()), tt.Plan(G.cuda()), tt.Chol(torch.from_numpy(L).cuda())
    mp = tt.MapInference(pF, pG, chol, nv.cuda())
    try:
        d_in = d_obs.cuda().clone()
        m_in = synth.vector_m(w, k_rhs=1).cuda()
        out_map = torch.empty((w.N_t, w.N_m), dtype=torch.float64, device="cuda")
        out_d = torch.empty((w.N_t, w.N_d), dtype=torch.float64, device="cuda")
        out_m = torch.empty_like(out_map)
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            for _ in range(2):                                    # warm-up outside the capture
                tt.tt_map_infer(mp.handle, tt.TT_MAP_PAPER, d_in, out_map, s)
        s.synchronize()
        ref_map = out_map.clone()
        tt.tt_debug_set("l2r_mb", 1)                              # F^T d in producer / consumer mode (forked plan stream) too
        tt.tt_debug_set("l2r_ctas", 8)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=s):
            tt.tt_matvec(pF.handle, m_in, out_d, s)
            tt.tt_rmatvec(pF.handle, out_d, out_m, s)
            tt.tt_map_infer(mp.handle, tt.TT_MAP_PAPER, d_in, out_map, s)
        out_map.zero_(); out_d.zero_(); out_m.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(out_map, ref_map)
        d_in.mul_(2.0)                                            # new data, same graph
        graph.replay()
        torch.cuda.synchronize()
        assert rel(out_map.cpu().numpy(), 2.0 * ref_map.cpu().numpy()) <= 1e-13
        assert rel(out_m.cpu().numpy(), op.rmatvec(F.numpy(), op.matvec(F.numpy(), m_in.cpu().numpy()))) <= 1e-12
    finally:
        tt.tt_debug_set("l2r_mb", -1)
        tt.tt_debug_set("l2r_ctas", 0)
        mp.close(); chol.close(); pF.close(); pG.close()


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("layout", [0, 1])
def test_pipelined_host_calls_equal_device_calls(tt, dtype, layout):
    """The *_host calls move the parameter-sized vector range by range (16 ranges of the parameter axis) on a copy stream
    while the kernels of the neighbouring range run; the result must be bit-identical to the device-pointer calls.
    N_m = 40007 gives ten non-empty ranges (4096 parameters each) with a ragged last one."""
    N_d, N_m, N_t, r = 3, 40007, 20, 2
    w = synth.CONFIGS["P5"].scaled(N_d=N_d, N_m=N_m, N_t=N_t, dtype=dtype)
    F = synth.block_column(w)
    G = gstar_column(w, F)
    nv, d_obs = synth.noise_var(w), synth.vector_d(w, k_rhs=1)
    m = synth.vector_m(w, k_rhs=1)
    lay = (lambda t: t.t().contiguous()) if layout == 1 else (lambda t: t)
    mh, dh = lay(m).pin_memory(), lay(d_obs).pin_memory()
    pF, pG = tt.Plan(F.cuda(), layout=layout), tt.Plan(G.cuda(), layout=layout)
    pC = tt.Plan(F.cuda(), layout=layout, out_every=r)
    n = N_d * N_t
    Lf = torch.eye(n, dtype=torch.float64) * 3.0 + torch.tril(torch.full((n, n), 0.01, dtype=torch.float64), -1)
    chol = tt.Chol(Lf.cuda())
    mp = tt.MapInference(pF, pG, chol, lay(nv).cuda())
    try:
        for plan, dvec in ((pF, dh), (pC, lay(d_obs[: N_t // r]).pin_memory())):
            d_dev = plan.matvec(mh.cuda())
            m_dev = plan.rmatvec(dvec.cuda())
            n_dev = plan.normal(mh.cuda())
            d_host = torch.empty_like(d_dev, device="cpu").pin_memory()
            m_host = torch.empty_like(m_dev, device="cpu").pin_memory()
            n_host = torch.empty_like(n_dev, device="cpu").pin_memory()
            tt.tt_matvec_host(plan.handle, mh, d_host)
            tt.tt_rmatvec_host(plan.handle, dvec, m_host)
            tt.tt_normal_host(plan.handle, mh, n_host)
            tt.tt_rmatvec_host(plan.handle, dvec, m_host)            # back to back: staging reuse is ordered
            torch.cuda.synchronize()
            assert torch.equal(d_host, d_dev.cpu()) and torch.equal(m_host, m_dev.cpu()) and torch.equal(n_host, n_dev.cpu())
        for form in (tt.TT_MAP_PAPER, tt.TT_MAP_GAIN):
            ref = mp.infer(dh.cuda(), form).cpu()
            out = torch.empty_like(ref).pin_memory()
            tt.tt_map_infer_host(mp.handle, form, dh, out)
            torch.cuda.synchronize()
            assert torch.equal(out, ref)
    finally:
        mp.close(); chol.close(); pF.close(); pG.close(); pC.close()


def test_trsv_repeated_launches_are_stable(tt):
    """The chain kernels spin on self-flagging data: 300 back-to-back solves (no host synchronisation in between, the
    flags are re-armed by the pre-step of every call) must all terminate and return the same bits."""
    n = 2500
    L = random_factor(n, 3)
    chol = tt.Chol(torch.from_numpy(L).cuda())
    try:
        b = torch.from_numpy(np.random.default_rng(2).standard_normal(n)).cuda()
        first = chol.solve(b).clone()
        outs = [torch.empty_like(b) for _ in range(4)]
        for it in range(300):
            tt.tt_chol_solve(chol.handle, b, outs[it % 4])
            if it % 3 == 0:
                tt.tt_chol_trsv(chol.handle, bool(it % 2), b, outs[(it + 1) % 4])
                tt.tt_chol_solve(chol.handle, b, outs[(it + 1) % 4])
        torch.cuda.synchronize()
        for o in outs:
            assert torch.equal(o, first)
    finally:
        chol.close()


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("layout", [0, 1])
def test_smw_operator(tt, dtype, layout):
    """(I - G* K^{-1} F) u, eq (4.7) / (4.8): the posterior covariance action for u = Gamma_prior v, against the oracle
    (which is pinned to the dense inverse Hessian)."""
    N_d, N_m, N_t = 5, 1000, 35
    w, F, G, nv, _ = online_inputs(N_d, N_m, N_t, dtype)
    Fn, Gn = F.numpy(), G.numpy()
    K = oo.assemble_K(Fn, Gn, nv.numpy())
    L = oo.cholesky(K)
    ev = np.linalg.eigvalsh(K)
    kappa = ev[-1] / ev[0]
    v = synth.vector_m(w, k_rhs=1)
    u = (v.double() * synth.prior_gamma(w)[None, :]).to(dtype)           # Gamma_prior v, rounded once: the input of both sides
    ref = oo.smw_apply(Fn, Gn, L, u.numpy())
    lay = (lambda t: t.t().contiguous()) if layout == 1 else (lambda t: t)
    unlay = (lambda t: t.t()) if layout == 1 else (lambda t: t)
    pF, pG = tt.Plan(F.cuda(), layout=layout), tt.Plan(G.cuda(), layout=layout)
    chol = tt.Chol(torch.from_numpy(L).cuda())
    mp = tt.MapInference(pF, pG, chol, lay(nv).cuda())
    try:
        ud = lay(u).cuda()
        got = unlay(mp.smw_apply(ud)).cpu().numpy()
        with pytest.raises(tt.TTError) as ei:
            tt.tt_smw_apply(mp.handle, ud, ud)
        assert ei.value.status == -7                                      # TT_ERR_ALIAS
    finally:
        mp.close(); chol.close(); pF.close(); pG.close()
    # u - G* K^{-1} F u: the correction is O(1) of u here, both terms carry the matvec bar; the solve amplifies by kappa
    assert rel(got, ref) <= BAR[dtype] + 8 * U[dtype] * kappa


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_phase3_compositions(tt, dtype):
    """eq (4.10) Gamma_post(q) v and eq (4.11)/(4.14) q_map = Q d_obs through the p2q plans on a coarser output grid."""
    N_d, N_q, N_m, N_t, r = 4, 3, 600, 30, 5
    w, F, G, nv, d_obs = online_inputs(N_d, N_m, N_t, dtype)
    wq = synth.CONFIGS["Q5"].scaled(N_d=N_q, N_m=N_m, N_t=N_t, dtype=dtype)
    Fq = synth.block_column(wq)
    Gq = gstar_column(wq, Fq)
    v = synth.vector_d(wq.scaled(N_t=N_t // r), k_rhs=1)
    Fn, Gn, nvn = F.numpy(), G.numpy(), nv.numpy()
    K = oo.assemble_K(Fn, Gn, nvn)
    L = oo.cholesky(K)
    ev = np.linalg.eigvalsh(K)
    kappa = ev[-1] / ev[0]
    ref_pq = oo.post_cov_q_apply(Fn, Gn, L, Fq.numpy(), Gq.numpy(), r, v.numpy())
    ref_q = oo.d2q_apply(Fn, Gn, nvn, L, Fq.numpy(), r, d_obs.numpy())
    pF, pG = tt.Plan(F.cuda()), tt.Plan(G.cuda())
    pFq, pGq = tt.Plan(Fq.cuda(), out_every=r), tt.Plan(Gq.cuda(), out_every=r)
    chol = tt.Chol(torch.from_numpy(L).cuda())
    mp = tt.MapInference(pF, pG, chol, nv.cuda())
    try:
        work = torch.empty((2, N_t, N_m), dtype=dtype, device="cuda")
        out = torch.empty((N_t // r, N_q), dtype=dtype, device="cuda")
        tt.tt_postcov_q_apply(mp.handle, pFq.handle, pGq.handle, v.cuda(), work, out)
        got_pq = out.cpu().numpy()
        got_q = {}
        for form in (tt.TT_MAP_PAPER, tt.TT_MAP_GAIN):
            tt.tt_d2q_apply(mp.handle, pFq.handle, form, d_obs.cuda(), work, out)
            got_q[form] = out.cpu().numpy()
        with pytest.raises(tt.TTError) as ei:                       # a p2q plan of another parameter dimension
            bad = tt.Plan(Fq[:, :, :500].contiguous().cuda(), out_every=r)
            try:
                tt.tt_d2q_apply(mp.handle, bad.handle, tt.TT_MAP_GAIN, d_obs.cuda(), work, out)
            finally:
                bad.close()
        assert ei.value.status == -12
    finally:
        mp.close(); chol.close(); pF.close(); pG.close(); pFq.close(); pGq.close()
    tol = BAR[dtype] + 8 * U[dtype] * kappa
    assert rel(got_pq, ref_pq) <= tol
    assert rel(got_q[tt.TT_MAP_PAPER], ref_q) <= tol and rel(got_q[tt.TT_MAP_GAIN], ref_q) <= BAR[dtype] + 8 * U[torch.float64] * kappa


@pytest.mark.parametrize("N_d,N_q,N_m,N_t,r", [(4, 3, 600, 30, 5), (2, 5, 130, 12, 1), (3, 2, 70, 40, 10), (1, 1, 9, 6, 3)])
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_qoi_direct(tt, N_d, N_q, N_m, N_t, r, dtype):
    """tt_qoi_direct: the dense data-to-QoI map Q (eq 4.11) and the dense QoI posterior covariance (eq 4.10) from block columns,
    against the oracle's operator forms applied to every unit vector."""
    w, F, G, nv, _ = online_inputs(N_d, N_m, N_t, dtype)
    wq = synth.CONFIGS["Q5"].scaled(N_d=N_q, N_m=N_m, N_t=N_t, dtype=dtype)
    Fq = synth.block_column(wq)
    Gq = gstar_column(wq, Fq)
    Fn, Gn, nvn, Fqn, Gqn = F.numpy(), G.numpy(), nv.numpy(), Fq.numpy(), Gq.numpy()
    K = oo.assemble_K(Fn, Gn, nvn)
    L = oo.cholesky(K)
    ev = np.linalg.eigvalsh(K)
    kappa = ev[-1] / ev[0]
    n, nq = N_t * N_d, (N_t // r) * N_q
    Q_ref = np.empty((nq, n))
    for c in range(n):
        e = np.zeros(n); e[c] = 1.0
        Q_ref[:, c] = oo.d2q_apply(Fn, Gn, nvn, L, Fqn, r, e.reshape(N_t, N_d)).reshape(nq)
    C_ref = np.empty((nq, nq))
    for c in range(nq):
        e = np.zeros(nq); e[c] = 1.0
        C_ref[:, c] = oo.post_cov_q_apply(Fn, Gn, L, Fqn, Gqn, r, e.reshape(N_t // r, N_q)).reshape(nq)
    chol = tt.Chol(torch.from_numpy(L).cuda())
    try:
        Q, C = tt.qoi_direct(Fq.cuda(), Gq.cuda(), G.cuda(), r, chol)
        Q, C = Q.cpu().numpy(), C.cpu().numpy()
        bad = tt.Chol(torch.eye(n + 1, dtype=torch.float64).cuda())
        try:
            with pytest.raises(tt.TTError) as ei:
                tt.qoi_direct(Fq.cuda(), Gq.cuda(), G.cuda(), r, bad)
            assert ei.value.status == -12                               # TT_ERR_MISMATCH: factor of another order
        finally:
            bad.close()
    finally:
        chol.close()
    tol = BAR[dtype] + 8 * U[dtype] * kappa
    assert rel(Q, Q_ref) <= tol
    assert rel(C, C_ref) <= tol
    assert rel(C, C.T) <= tol


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_assemble_K_space_major(tt, dtype):
    """K's ordering is row = i*N_d + s whatever the plans' layout: unit vectors and results of TT_SPACE_MAJOR plans are permuted."""
    N_d, N_m, N_t = 3, 200, 14
    w, F, G, nv, _ = online_inputs(N_d, N_m, N_t, dtype)
    K_ref = oo.assemble_K(F.numpy(), G.numpy(), nv.numpy())
    for k_max in (1, 5):
        pF, pG = tt.Plan(F.cuda(), layout=1, k_max=k_max), tt.Plan(G.cuda(), layout=1, k_max=k_max)
        try:
            K = tt.assemble_K(pF, pG, nv.t().contiguous().cuda()).cpu().numpy()
        finally:
            pF.close(); pG.close()
        assert rel(K, K_ref) <= BAR[dtype]
