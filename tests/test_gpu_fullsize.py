"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

C2, C3, C5 (4.3 / 80 / 64 GB spectra) are compared with the oracle over the WHOLE output vector
(SURVEY.md 8(c)); C4 over whole columns of the k-RHS result.  At C3 / C5 / C4 the block column is
drawn once on the device (the 40 GB column would take minutes on the host) and streamed to the host
oracle in sensor slabs - the very same bytes on both sides - which costs about two minutes of
oracle time per config on the box's 16 host cores.  On top: properties that hold at any size
(adjoint identity, <m, F^T F m> = |F m|^2) and bit-equality of the pipelined *_host calls.
"""
import numpy as np
import pytest
import torch

from oracle import toeplitz_blocked as ob
import synth
from tests.inputs_online import gstar_column

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
    import gc
    gc.collect()
    torch.cuda.empty_cache()          # blocks cached by torch for an earlier test count as used otherwise
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


def _slab_sensors(w, target_bytes=2 << 30):
    """Sensors per slab of the block column so that one slab F[:, s0:s1, :] is about target_bytes on the host."""
    es = 4 if w.dtype == torch.float32 else 8
    return max(1, min(w.N_d, int(target_bytes // (w.N_t * w.N_m * es))))


def _whole_vector(tt, cfg):
    """F m, F^T d and F^T F m of config `cfg` at full size against the oracle over EVERY output ("over the
    whole output vector"; eq 2.5; "exact up to rounding error").

    The block column stays on the device and is streamed to the host in sensor slabs F[:, s0:s1, :]: each slab gives
    complete rows d[:, s0:s1] of oracle.matvec and one term of oracle.rmatvec, accumulated in fp64 (the sum over sensors
    of the definition, split at slab boundaries).  The normal operator's reference has the oracle on both halves:
    rmatvec(F, matvec(F, m)), the intermediate kept in fp64.  The *_host calls (pipelined over 8 graded or 16 equal parameter ranges, whose
    boundaries only exist at this size) must reproduce the device-pointer calls bit for bit."""
    import time
    w = synth.CONFIGS[cfg]
    es = 4 if w.dtype == torch.float32 else 8
    need_memory(int(3.1 * w.N_t * w.N_d * w.N_m * es / 2**30) + 8)      # block column + its complex spectrum + vectors
    tol = TOL[w.dtype]
    F = synth.block_column(w, device="cuda")
    m, d = synth.vector_m(w, device="cuda", k_rhs=1), synth.vector_d(w, device="cuda", k_rhs=1)
    plan = tt.Plan(F)
    try:
        Fm, Ftd, FtFm = plan.matvec(m), plan.rmatvec(d), plan.normal(m)
        torch.cuda.synchronize()
        m_h, d_h = m.cpu().pin_memory(), d.cpu().pin_memory()
        d_o, m_o, n_o = torch.empty_like(d_h).pin_memory(), torch.empty_like(m_h).pin_memory(), torch.empty_like(m_h).pin_memory()
        tt.tt_matvec_host(plan.handle, m_h, d_o)
        tt.tt_rmatvec_host(plan.handle, d_h, m_o)
        tt.tt_normal_host(plan.handle, m_h, n_o)
        torch.cuda.synchronize()
    finally:
        plan.close()
    Fm_h, Ftd_h, FtFm_h = Fm.cpu(), Ftd.cpu(), FtFm.cpu()
    assert torch.equal(d_o, Fm_h) and torch.equal(m_o, Ftd_h) and torch.equal(n_o, FtFm_h), "host-vector calls differ from device calls"
    del m_o, n_o, d_o
    # properties at full size (fp64 dot products of the device results)
    lhs, rhs = float((Fm.double() * d.double()).sum()), float((m.double() * Ftd.double()).sum())
    assert abs(lhs - rhs) <= tol * float(Fm.double().norm() * d.double().norm())          # <F m, d> = <m, F^T d>
    q, n2 = float((m.double() * FtFm.double()).sum()), float(Fm.double().norm() ** 2)
    assert abs(q - n2) <= tol * n2                                                        # <m, F^T F m> = |F m|^2
    del Fm, Ftd, FtFm
    torch.cuda.empty_cache()

    mh, dh = m_h.numpy(), d_h.numpy()
    ref_d = np.empty((w.N_t, w.N_d), dtype=np.float64)
    ref_m = np.zeros((w.N_t, w.N_m), dtype=np.float64)
    ref_n = np.zeros((w.N_t, w.N_m), dtype=np.float64)
    ns = _slab_sensors(w)
    t0 = time.perf_counter()
    for s0 in range(0, w.N_d, ns):
        s1 = min(w.N_d, s0 + ns)
        slab = F[:, s0:s1, :].contiguous().cpu().numpy()
        ref_d[:, s0:s1] = ob.matvec(slab, mh)
        ref_m += ob.rmatvec(slab, np.ascontiguousarray(dh[:, s0:s1]))
        ref_n += ob.rmatvec(slab.astype(np.float64), np.ascontiguousarray(ref_d[:, s0:s1]))
        del slab
    t_oracle = time.perf_counter() - t0
    e_d, e_m, e_n = rel(Fm_h.numpy(), ref_d), rel(Ftd_h.numpy(), ref_m), rel(FtFm_h.numpy(), ref_n)
    print(f"{cfg} whole-vector rel-L2 vs the oracle ({w.N_t * w.N_d} + 2 x {w.N_t * w.N_m} outputs, oracle {t_oracle:.0f} s on "
          f"{ob.num_threads()} threads): F m {e_d:.2e}  F^T d {e_m:.2e}  F^T F m {e_n:.2e}  (tol {tol:g})")
    assert e_d <= tol, f"F m: {e_d}"
    assert e_m <= tol, f"F^T d: {e_m}"
    assert e_n <= tol, f"F^T F m: {e_n}"
    # no output may hide behind the norm of the others: every sensor series and every block of 4096 parameters on its own
    for s in range(w.N_d):
        assert rel(Fm_h[:, s].numpy(), ref_d[:, s]) <= tol, f"F m, sensor {s}"
    got_m, got_n = Ftd_h.numpy(), FtFm_h.numpy()
    for p0 in range(0, w.N_m, 4096):
        sl = slice(p0, min(w.N_m, p0 + 4096))
        assert rel(got_m[:, sl], ref_m[:, sl]) <= tol, f"F^T d, parameters {p0}.."
        assert rel(got_n[:, sl], ref_n[:, sl]) <= tol, f"F^T F m, parameters {p0}.."


def test_c3_whole_vector(tt):
    """BASELINE.json configs[2], the config the metric is quoted on: 100 x 250000 x 400, complex64 spectrum of 80 GB."""
    _whole_vector(tt, "C3")


def test_c5_whole_vector(tt):
    """BASELINE.json configs[4]: the normal operator at 200 x 100000 x 400."""
    _whole_vector(tt, "C5")


def test_c4_krhs_whole_columns(tt):
    """configs[3]: fp64, k = 32 right-hand sides through the DMMA GEMM path, at full size (34 GB spectrum): columns 0, 13 and 31
    of F M and of F^T D over EVERY sensor and EVERY parameter against the oracle (one column at a time, block column streamed
    in sensor slabs), the remaining columns through the adjoint identity over all 32 at once."""
    import time
    w = synth.CONFIGS["C4"]
    need_memory(110)
    k = w.k_rhs
    F = synth.block_column(w, device="cuda")
    M, D = synth.vector_m(w, device="cuda"), synth.vector_d(w, device="cuda")   # [N_t, N_m, k], [N_t, N_d, k]
    cols = [0, 13, k - 1]
    plan = tt.Plan(F, k_max=k)
    try:
        FM = plan.matvec_batched(M)
        FtD = plan.rmatvec_batched(D)
        torch.cuda.synchronize()
    finally:
        plan.close()
    lhs, rhs = float((FM * D).sum()), float((M * FtD).sum())
    assert abs(lhs - rhs) <= 1e-12 * float(FM.norm() * D.norm())                # <F M, D> = <M, F^T D>, all columns
    got_d = {r: FM[..., r].contiguous().cpu().numpy() for r in cols}
    got_m = {r: FtD[..., r].contiguous().cpu().numpy() for r in cols}
    m_r = {r: M[..., r].contiguous().cpu().numpy() for r in cols}
    d_r = {r: D[..., r].contiguous().cpu().numpy() for r in cols}
    del FM, FtD, M, D
    torch.cuda.empty_cache()
    ref_d = {r: np.empty((w.N_t, w.N_d)) for r in cols}
    ref_m = {r: np.zeros((w.N_t, w.N_m)) for r in cols}
    ns = _slab_sensors(w)
    t0 = time.perf_counter()
    for s0 in range(0, w.N_d, ns):
        s1 = min(w.N_d, s0 + ns)
        slab = F[:, s0:s1, :].contiguous().cpu().numpy()
        for r in cols:
            ref_d[r][:, s0:s1] = ob.matvec(slab, m_r[r])
            ref_m[r] += ob.rmatvec(slab, np.ascontiguousarray(d_r[r][:, s0:s1]))
        del slab
    errs = [(rel(got_d[r], ref_d[r]), rel(got_m[r], ref_m[r])) for r in cols]
    print(f"C4 k-RHS whole columns {cols} rel-L2 vs the oracle (oracle {time.perf_counter() - t0:.0f} s): "
          + "  ".join(f"[F M {a:.2e}, F^T D {b:.2e}]" for a, b in errs))
    for r, (a, b) in zip(cols, errs):
        assert a <= 1e-12, f"F M, column {r}: {a}"
        assert b <= 1e-12, f"F^T D, column {r}: {b}"
        for s in range(w.N_d):
            assert rel(got_d[r][:, s], ref_d[r][:, s]) <= 1e-12, f"F M, sensor {s}, column {r}"


def test_p5_quarter_krhs_fp32_whole_columns(tt):
    """The fp32 k-RHS path (3xTF32 GEMMs on tcgen05, tt_gemm32_umma.cu) at the paper's sensor and time counts (49 sensors, 500
    steps, 501 frequencies) and a quarter of its parameters (65 792: 13 GB spectrum, 2056 K-blocks per frequency, 514 parameter
    tiles): columns 0 and 31 of F M and of F^T D over every sensor and every parameter against the oracle, all 32 columns through
    the adjoint identity.  (P5 with k = 32 is not a BASELINE.json config: this is the size the oracle does in half a minute.)"""
    import time
    w = synth.CONFIGS["P5"].scaled(N_m=65792, k_rhs=32)
    need_memory(60)
    k = w.k_rhs
    F = synth.block_column(w, device="cuda")
    M, D = synth.vector_m(w, device="cuda"), synth.vector_d(w, device="cuda")   # [N_t, N_m, k], [N_t, N_d, k]
    cols = [0, k - 1]
    plan = tt.Plan(F, k_max=k)
    try:
        FM = plan.matvec_batched(M)
        FtD = plan.rmatvec_batched(D)
        torch.cuda.synchronize()
    finally:
        plan.close()
    lhs, rhs = float((FM.double() * D.double()).sum()), float((M.double() * FtD.double()).sum())
    assert abs(lhs - rhs) <= 1e-5 * float(FM.double().norm() * D.double().norm())   # <F M, D> = <M, F^T D>, all columns
    got_d = {r: FM[..., r].contiguous().cpu().numpy() for r in cols}
    got_m = {r: FtD[..., r].contiguous().cpu().numpy() for r in cols}
    m_r = {r: M[..., r].contiguous().cpu().numpy() for r in cols}
    d_r = {r: D[..., r].contiguous().cpu().numpy() for r in cols}
    del FM, FtD, M, D
    torch.cuda.empty_cache()
    Fh = F.cpu().numpy()
    del F
    t0 = time.perf_counter()
    errs = []
    for r in cols:
        ref_d, ref_m = ob.matvec(Fh, m_r[r]), ob.rmatvec(Fh, d_r[r])
        errs.append((rel(got_d[r], ref_d), rel(got_m[r], ref_m)))
        for s in range(w.N_d):
            assert rel(got_d[r][:, s], ref_d[:, s]) <= 1e-5, f"F M, sensor {s}, column {r}"
        for p0 in range(0, w.N_m, 4096):
            assert rel(got_m[r][:, p0:p0 + 4096], ref_m[:, p0:p0 + 4096]) <= 1e-5, f"F^T D, parameters {p0}.., column {r}"
    print(f"P5/4 fp32 k-RHS whole columns {cols} rel-L2 vs the oracle (oracle {time.perf_counter() - t0:.0f} s): "
          + "  ".join(f"[F M {a:.2e}, F^T D {b:.2e}]" for a, b in errs))
    for r, (a, b) in zip(cols, errs):
        assert a <= 1e-5 and b <= 1e-5, f"column {r}: {a}, {b}"


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
        G = gstar_column(w, F)
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


def test_online_p5_full_size_whole_vector(tt):
    """The paper's own shape (N_d=49, N_m=263169, N_t=500: 131 584 500 parameters, 24 500 data), in the launch
    configuration `bench.py --config P5 --online` times: the K-solve against the oracle over the whole vector, and
    m_map = G* K^{-1} d_obs (gain form, eq 4.13 by reading R16) over ALL 131 584 500 parameters against the oracle's
    G* z = rmatvec(G, z), the block column of G* streamed to the host in sensor slabs.  The factor is the seeded
    stand-in the tests use at this order."""
    import time
    from oracle import online_plain as oo
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
    synth.scaled_block_column(w, G, out=G)
    pG = tt.Plan(G)
    mp = tt.MapInference(None, pG, chol, synth.noise_var(w, device="cuda"))
    try:
        m_map = mp.infer(d_obs, tt.TT_MAP_GAIN)
        got = m_map.cpu().numpy()
    finally:
        mp.close(); pG.close(); chol.close()
    del m_map
    torch.cuda.empty_cache()
    zr = z_ref.reshape(w.N_t, w.N_d)
    ref = np.zeros((w.N_t, w.N_m))
    t0 = time.perf_counter()
    for s0 in range(0, w.N_d, 4):
        s1 = min(w.N_d, s0 + 4)
        slab = G[:, s0:s1, :].contiguous().cpu().numpy()
        ref += ob.rmatvec(slab.astype(np.float64), np.ascontiguousarray(zr[:, s0:s1]))
        del slab
    err = rel(got, ref)
    print(f"P5 online, gain form, whole m_map ({w.N_t * w.N_m} parameters) rel-L2 vs the oracle (oracle {time.perf_counter() - t0:.0f} s): {err:.2e} (tol 1e-05)")
    assert err <= 1e-5
    for p0 in range(0, w.N_m, 8192):
        assert rel(got[:, p0:p0 + 8192], ref[:, p0:p0 + 8192]) <= 1e-5, f"parameters {p0}.."


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
    synth.scaled_block_column(w, F, out=F)
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
    G = synth.scaled_block_column(w, F)
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
        synth.scaled_block_column(w, slab, out=slab)
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
