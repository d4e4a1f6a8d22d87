"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

C2 (fp64, 4.3 GB spectrum) is compared element by element over the whole output.  At C3 / C5
(80 / 64 GB spectra) the oracle's O(N_t^2 N_d N_m) cost forbids that, so the CUDA outputs are
compared on slices the oracle can compute from a slice of the block column -- whole time
series d[:, s] of single sensors (needs F[:, s, :]) and whole series m'[:, p0:p1] of parameter
ranges (needs F[:, :, p0:p1]) -- in relative L2 over each slice, plus properties that hold at
any size (adjoint identity, <m, F^T F m> = |F m|^2).  The inputs are drawn once on the device
(the 40 GB column would take minutes on the host) and the very same bytes are copied to the
host for the oracle.
"""
import numpy as np
import pytest
import torch

from oracle import toeplitz_blocked as ob
from paper_2501_14911_b200 import synth

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
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def need_memory(gb):
    free, _ = torch.cuda.mem_get_info()
    if free < gb * (1 << 30):
        pytest.skip(f"needs {gb} GiB of free device memory")


def test_c2_full_elementwise(tt):
    w = synth.CONFIGS["C2"]
    need_memory(12)
    F = synth.block_column(w, device="cuda")
    m, d = synth.vector_m(w, device="cuda"), synth.vector_d(w, device="cuda")
    plan = tt.Plan(F)
    try:
        got_d, got_m, got_n = plan.matvec(m).cpu().numpy(), plan.rmatvec(d).cpu().numpy(), plan.normal(m).cpu().numpy()
    finally:
        plan.close()
    Fh, mh, dh = F.cpu().numpy(), m.cpu().numpy(), d.cpu().numpy()
    del F
    ref_d = ob.matvec(Fh, mh)
    ref_m = ob.rmatvec(Fh, dh)
    ref_n = ob.rmatvec(Fh, ref_d)
    assert rel(got_d, ref_d) <= 1e-12
    assert rel(got_m, ref_m) <= 1e-12
    assert rel(got_n, ref_n) <= 1e-12


@pytest.mark.parametrize("cfg", ["C3", "C5"])
def test_paper_scale_slices_and_properties(tt, cfg):
    w = synth.CONFIGS[cfg]
    need_memory(150)
    tol = TOL[w.dtype]
    F = synth.block_column(w, device="cuda")
    m, d = synth.vector_m(w, device="cuda", k_rhs=1), synth.vector_d(w, device="cuda", k_rhs=1)
    sensors = [0, w.N_d // 2 + 1, w.N_d - 1]
    p_ranges = [(0, 48), (w.N_m // 3 + 5, w.N_m // 3 + 37), (w.N_m - 33, w.N_m)]
    F_rows = {s: F[:, s:s + 1, :].contiguous().cpu().numpy() for s in sensors}
    F_cols = {pr: F[:, :, pr[0]:pr[1]].contiguous().cpu().numpy() for pr in p_ranges}
    plan = tt.Plan(F)
    del F
    torch.cuda.empty_cache()
    try:
        Fm = plan.matvec(m)
        Ftd = plan.rmatvec(d)
        FtFm = plan.normal(m)
        torch.cuda.synchronize()
    finally:
        plan.close()
    mh, dh = m.cpu().numpy(), d.cpu().numpy()
    Fm_h, Ftd_h, FtFm_h = Fm.cpu().numpy(), Ftd.cpu().numpy(), FtFm.cpu().numpy()

    # F m on whole single-sensor series
    for s in sensors:
        ref = ob.matvec(F_rows[s], mh)[:, 0]
        assert rel(Fm_h[:, s], ref) <= tol, f"F m, sensor {s}"
    # F^T d and F^T (F m) on whole parameter-range series; the normal operator is checked against the
    # oracle applied to the (already checked) device result of F m
    for pr in p_ranges:
        ref = ob.rmatvec(F_cols[pr], dh)
        assert rel(Ftd_h[:, pr[0]:pr[1]], ref) <= tol, f"F^T d, parameters {pr}"
        ref_n = ob.rmatvec(F_cols[pr].astype(np.float64), Fm_h.astype(np.float64))
        assert rel(FtFm_h[:, pr[0]:pr[1]], ref_n) <= tol, f"F^T F m, parameters {pr}"
    # properties at full size (fp64 dot products of the device results)
    lhs = float((Fm.double() * d.double()).sum())
    rhs = float((m.double() * Ftd.double()).sum())
    scale = float(Fm.double().norm() * d.double().norm())
    assert abs(lhs - rhs) <= tol * scale                       # <F m, d> = <m, F^T d>
    q = float((m.double() * FtFm.double()).sum())
    n2 = float(Fm.double().norm() ** 2)
    assert abs(q - n2) <= 10 * tol * n2                        # <m, F^T F m> = |F m|^2


def test_c4_krhs_slices(tt):
    """configs[3]: fp64, k = 32 right-hand sides through the DMMA GEMM path, at full size (34 GB spectrum).
    Whole time series of sampled (sensor, column) and (parameter range, column) pairs against the oracle."""
    w = synth.CONFIGS["C4"]
    need_memory(110)
    k = w.k_rhs
    F = synth.block_column(w, device="cuda")
    M, D = synth.vector_m(w, device="cuda"), synth.vector_d(w, device="cuda")   # [N_t, N_m, k], [N_t, N_d, k]
    sensors, cols = [0, w.N_d - 1], [0, 13, k - 1]
    p_ranges = [(0, 40), (w.N_m - 24, w.N_m)]
    F_rows = {s: F[:, s:s + 1, :].contiguous().cpu().numpy() for s in sensors}
    F_cols = {pr: F[:, :, pr[0]:pr[1]].contiguous().cpu().numpy() for pr in p_ranges}
    plan = tt.Plan(F, k_max=k)
    del F
    torch.cuda.empty_cache()
    try:
        FM = plan.matvec_batched(M)
        FtD = plan.rmatvec_batched(D)
        torch.cuda.synchronize()
    finally:
        plan.close()
    for r in cols:
        m_r = M[..., r].contiguous().cpu().numpy()
        d_r = D[..., r].contiguous().cpu().numpy()
        for s in sensors:
            ref = ob.matvec(F_rows[s], m_r)[:, 0]
            assert rel(FM[:, s, r].cpu().numpy(), ref) <= 1e-12, f"F M, sensor {s}, column {r}"
        for pr in p_ranges:
            ref = ob.rmatvec(F_cols[pr], d_r)
            assert rel(FtD[:, pr[0]:pr[1], r].cpu().numpy(), ref) <= 1e-12, f"F^T D, parameters {pr}, column {r}"
    # adjoint identity over all columns at once: <F M, D> = <M, F^T D>
    lhs, rhs = float((FM * D).sum()), float((M * FtD).sum())
    assert abs(lhs - rhs) <= 1e-12 * float(FM.norm() * D.norm())


# ------------------------------------------------------------------------------------------------
# Online phase at sizes beyond tests/test_gpu_online.py
# ------------------------------------------------------------------------------------------------
def test_online_medium_true_K(tt):
    """Everything real at a size that spans several tiles of every kernel (2 GEMV chunks, 10 blocks of the
    triangular solves): K assembled by the GPU against the oracle's K, then m_map (both forms) with the ORACLE's
    Cholesky factor against the oracle's eq (4.13)."""
    from oracle import online_plain as oo
    for dtype in (torch.float64, torch.float32):
        w = synth.CONFIGS["P5"].scaled(N_d=8, N_m=4160, N_t=80, dtype=dtype)
        F = synth.block_column(w)
        G = synth.gstar_block_column(w, F)
        nv, d_obs = synth.noise_var(w), synth.vector_d(w, k_rhs=1)
        Fn, Gn = F.numpy(), G.numpy()
        K_ref = oo.assemble_K(Fn, Gn, nv.numpy())
        L = oo.cholesky(K_ref)
        m_ref = oo.map_point(Fn, Gn, nv.numpy(), L, d_obs.numpy(), conv=ob)
        ev = np.linalg.eigvalsh(K_ref)
        kappa = ev[-1] / ev[0]
        pF, pG = tt.Plan(F.cuda(), k_max=16), tt.Plan(G.cuda(), k_max=16)
        chol = tt.Chol(torch.from_numpy(L))          # host factor: goes through the slab path
        mp = tt.MapInference(pF, pG, chol, nv.cuda())
        try:
            K = tt.assemble_K(pF, pG, nv.cuda()).cpu().numpy()
            m_paper = mp.infer(d_obs.cuda(), tt.TT_MAP_PAPER).cpu().numpy()
            m_gain = mp.infer(d_obs.cuda(), tt.TT_MAP_GAIN).cpu().numpy()
        finally:
            mp.close(); chol.close(); pF.close(); pG.close()
        u = 1.1e-16 if dtype == torch.float64 else 6e-8
        print(f"online medium {dtype}: kappa {kappa:.0f}  K {rel(K, K_ref):.2e}  gain {rel(m_gain, m_ref):.2e}  "
              f"paper {rel(m_paper, m_ref):.2e}")
        assert rel(K, K_ref) <= TOL[dtype]
        assert rel(m_gain, m_ref) <= TOL[dtype] + 8 * 1.1e-16 * kappa
        assert rel(m_paper, m_ref) <= TOL[dtype] + 8 * u * kappa


def test_online_p5_full_size_sampled(tt):
    """The paper's own shape (N_d=49, N_m=263169, N_t=500: 131 584 500 parameters, 24 500 data), in the launch
    configuration `bench.py --config P5 --online` times: the K-solve against the oracle over the whole vector, and
    m_map = G* K^{-1} d_obs (gain form) on sampled outputs the oracle computes one by one from single columns
    G[:, :, p] of the block column.  The factor is the seeded stand-in the bench uses."""
    from oracle import online_plain as oo
    from oracle import toeplitz_plain as op
    w = synth.CONFIGS["P5"]
    need_memory(120)
    n = w.N_d * w.N_t
    L = synth.factor_standin(n, w.seed, device="cuda")
    chol = tt.Chol(L)
    L_h = L.cpu().numpy()
    del L
    d_obs = synth.vector_d(w, device="cuda", k_rhs=1)
    d_np = d_obs.cpu().numpy().astype(np.float64)
    z_ref = oo.chol_solve(L_h, d_np.reshape(n))
    z = chol.solve(torch.from_numpy(d_np.reshape(n)).cuda()).cpu().numpy()
    assert rel(z, z_ref) <= 1e-12
    chol_h = tt.Chol(torch.from_numpy(L_h))       # the same factor from HOST memory: five 1 GiB slabs of block rows
    try:
        z_h = chol_h.solve(torch.from_numpy(d_np.reshape(n)).cuda()).cpu().numpy()
    finally:
        chol_h.close()
    assert np.array_equal(z_h, z)
    del L_h
    G = synth.block_column(w, device="cuda")
    synth.gstar_block_column(w, G, out=G)
    rng = np.random.default_rng(5)
    ps = sorted(set(int(p) for p in rng.integers(0, w.N_m, 12)) | {0, w.N_m - 1})
    cols = {p: G[:, :, p:p + 1].cpu().numpy() for p in ps}
    pG = tt.Plan(G)
    del G
    torch.cuda.empty_cache()
    mp = tt.MapInference(None, pG, chol, synth.noise_var(w, device="cuda"))
    try:
        m_map = mp.infer(d_obs, tt.TT_MAP_GAIN)
        got = {p: m_map[:, p].cpu().numpy() for p in ps}
        scale = float(m_map.double().pow(2).mean().sqrt())
    finally:
        mp.close(); pG.close(); chol.close()
    zr = z_ref.reshape(w.N_t, w.N_d)
    for p in ps:
        ref = np.array([op.rmatvec_entry(cols[p], zr, j, 0) for j in range(0, w.N_t, 7)])
        err = np.linalg.norm(got[p][::7] - ref) / max(np.linalg.norm(ref), 1e-3 * scale * np.sqrt(len(ref)))
        assert err <= 1e-5, (p, err)


def test_K_assembly_p5_full_size_sampled(tt):
    """tt_assemble_K at the paper's shape in the configuration `bench.py --config P5 --online --k-batch 16` times
    (fp32 plans, batches of 16 unit vectors through the batched FFTs and the complex64 GEMMs): 16 columns of K, sampled
    entries against oracle/online_plain.K_entry computed from single sensor rows of the block columns."""
    from oracle import online_plain as oo
    w = synth.CONFIGS["P5"]
    need_memory(160)
    n = w.N_d * w.N_t
    F = synth.block_column(w, device="cuda")
    rows_F = {s: F[:, s, :].cpu().numpy() for s in (0, 17, 48)}
    pF = tt.Plan(F, k_max=16)
    synth.gstar_block_column(w, F, out=F)
    cols = [(3, 5), (250, 17), (499, 48)]                      # (time step, sensor) of sampled columns of K
    rows_G = {s2: F[:, s2, :].cpu().numpy() for _, s2 in cols}
    pG = tt.Plan(F, k_max=16)
    del F
    torch.cuda.empty_cache()
    nv = synth.noise_var(w, device="cuda")
    try:
        got = {}
        K = torch.zeros((n, n), dtype=torch.float64, device="cuda")
        for i2, s2 in cols:
            c = i2 * w.N_d + s2
            c0 = min(c - c % 16, n - 16)
            tt.tt_assemble_K(pF.handle, pG.handle, nv, c0, 16, K, n)
            got[(i2, s2)] = K[:, c].cpu().numpy()
        del K
    finally:
        pF.close(); pG.close()
    nvh = nv.cpu().numpy().astype(np.float64)
    for (i2, s2), col in got.items():
        scale = np.sqrt(np.mean(col ** 2))
        for i, s in ((0, 0), (i2, 17), (min(i2 + 40, w.N_t - 1), 48), (w.N_t - 1, 0), (i2, s2)):
            if (i, s) == (i2, s2):
                rows = rows_F.get(s)
                if rows is None:
                    continue
                ref = oo.K_entry(rows, rows_G[s2], i, i2, nvh[i, s])
            else:
                ref = oo.K_entry(rows_F[s], rows_G[s2], i, i2)
            assert abs(col[i * w.N_d + s] - ref) <= 1e-5 * max(abs(ref), scale), ((i, s), (i2, s2), col[i * w.N_d + s], ref)


def test_K_direct_p5_full_size_sampled(tt):
    """tt_assemble_K_direct at the paper's shape (fp32 block columns of 25.8 GB each, n = 24 500): the whole K in one call, as
    `bench.py --config P5 --online` times it; sampled entries against oracle/online_plain.K_entry, exact symmetry, and
    the noise on the diagonal."""
    from oracle import online_plain as oo
    w = synth.CONFIGS["P5"]
    need_memory(70)
    n = w.N_d * w.N_t
    F = synth.block_column(w, device="cuda")
    G = synth.gstar_block_column(w, F)
    nv = synth.noise_var(w, device="cuda")
    K = torch.full((n, n), float("nan"), dtype=torch.float64, device="cuda")
    tt.tt_assemble_K_direct(F, G, nv, w.N_d, w.N_m, w.N_t, tt.TT_F32, K, n)
    torch.cuda.synchronize()
    rows_F = {s: F[:, s, :].cpu().numpy() for s in (0, 17, 48)}
    rows_G = {s: G[:, s, :].cpu().numpy() for s in (5, 17, 48)}
    del F, G
    assert bool(torch.isfinite(K).all())
    for r0 in range(0, n, 4900):                                   # K == K^T bit for bit, slab by slab
        assert bool((K[r0:r0 + 4900, :] == K[:, r0:r0 + 4900].t()).all())
    nvh = nv.cpu().numpy().astype(np.float64)
    scale = float(K[:: 97, :: 89].pow(2).mean().sqrt())
    pairs = [((0, 0), (3, 5)), ((3, 17), (3, 5)), ((43, 48), (3, 5)), ((499, 0), (3, 5)),
             ((250, 17), (250, 17)), ((290, 48), (250, 17)), ((0, 0), (250, 17)), ((499, 0), (250, 17)),
             ((499, 48), (499, 48)), ((499, 17), (499, 48)), ((127, 0), (499, 48)), ((2, 48), (1, 48)), ((261, 17), (262, 5))]
    for (i, s), (i2, s2) in pairs:
        ref = oo.K_entry(rows_F[s], rows_G[s2], i, i2, nvh[i, s] if (i, s) == (i2, s2) else 0.0)
        got = float(K[i * w.N_d + s, i2 * w.N_d + s2])
        assert abs(got - ref) <= 1e-5 * max(abs(ref), scale), ((i, s), (i2, s2), got, ref)


def test_online_fp64_full_parameter_dimension(tt):
    """The fp64 path (complex128 spectrum) at the paper's full parameter and time dimensions (N_m = 263169, N_t = 500) with
    8 sensors - the configuration of `bench.py --config P5 --online --f64` with fewer sensors, block column handed over as a
    HOST pointer: m_map = G* K^{-1} d_obs on sampled outputs against the oracle, bar 1e-12 of the rms."""
    from oracle import online_plain as oo
    from oracle import toeplitz_plain as op
    w = synth.CONFIGS["P5"].scaled(N_d=8, dtype=torch.float64)
    need_memory(40)
    n = w.N_d * w.N_t
    G_h = torch.empty((w.N_t, w.N_d, w.N_m), dtype=torch.float64)
    for s0 in range(0, w.N_d, 4):
        slab = synth.block_column(w, device="cuda", s_range=(s0, s0 + 4))
        synth.gstar_block_column(w, slab, out=slab)
        G_h[:, s0:s0 + 4, :] = slab.cpu()
        del slab
    pG = tt.Plan(G_h)                                              # host pointer: streamed through 1 GiB slabs
    ps = (0, 131072, w.N_m - 1)
    cols = {p: G_h[:, :, p:p + 1].numpy().copy() for p in ps}
    del G_h
    L = synth.factor_standin(n, w.seed, device="cuda")
    chol = tt.Chol(L)
    L_h = L.cpu().numpy()
    del L
    d_obs = synth.vector_d(w, device="cuda", k_rhs=1)
    mp = tt.MapInference(None, pG, chol, synth.noise_var(w, device="cuda"))
    try:
        m_map = mp.infer(d_obs, tt.TT_MAP_GAIN)
        scale = float(m_map.pow(2).mean().sqrt())
        got = {p: m_map[::25, p].cpu().numpy() for p in ps}
    finally:
        mp.close(); chol.close(); pG.close()
    z = oo.chol_solve(L_h, d_obs.cpu().numpy().reshape(n)).reshape(w.N_t, w.N_d)
    for p in ps:
        ref = np.array([op.rmatvec_entry(cols[p], z, j, 0) for j in range(0, w.N_t, 25)])
        assert np.abs(got[p] - ref).max() <= 1e-12 * scale, p
