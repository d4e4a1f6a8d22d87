#!/usr/bin/env python
"""bench.py - ms per F.m and F^T.d at ~1e8 parameters, and achieved HBM GB/s vs the B200 peak.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C3] [--impl ours|reference]

A "step" is one pass of the whole hot path: d = F m (kernels A1, A2, A3) followed by
m' = F^T d (B1, B2, B3) on the BASELINE.json configs[2] workload (C3: N_d=100, N_m=250000,
N_t=400, fp32 vectors, complex64 spectrum of 80.2 GB), synthetic seeded inputs resident in HBM.
The JSON line carries
  value      ms per step (one F.m plus one F^T.d), device time, max over ranks, / n_gpus
  e2e        the same through tt_matvec_host / tt_rmatvec_host with pinned HOST vectors
             (H2D of the input and D2H of the result inside the timed region)
  roofline   the dominant kernel (the per-frequency matvec that streams Fhat): algorithmic
             bytes per launch / its mean launch duration, measured live with CUDA events
             recorded by the library on the launching stream, vs MEASURED_PEAKS.json
  cpu_baseline  the CPU oracle (oracle/, as it stands) timed on this box's host cores on a
             bounded sample of the same workload, extrapolated by the MAC count
Multi-GPU: the north star is a one-GPU path (no sharding, no collectives): --gpus N runs N
independent replicas ("replicas only"), timed as the max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import synth  # noqa: E402

METRIC = "ms per F·m and F^T·d at ~1e8 params; achieved HBM GB/s vs B200 peak"
NOMINAL_HBM_GBS = 8000.0     # north_star's "~8 TB/s"
FALLBACK_HBM_GBS = 6650.0    # B200_PROFILING.md fallback
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the newest committed `ncu --set full`
# capture of each config.  A figure is only quoted when the plan built in THIS run describes its kernels (tt_plan_describe)
# with the line the capture's summary records; otherwise `traffic` is null and the line says why.
NCU_TRAFFIC = {
    "C3": {"bytes": 81.003854e9 + 23.052e6, "profile": "profiles/r2_c3_ncu_full.md",
           "kernel": "A2 gemv_fwd_kernel<float,8> grid=(62,401) block=512 smem=32768 chunk=4096"},
}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return json.load(f), "measured"
    except OSError:
        return {"hbm_gbs": FALLBACK_HBM_GBS}, "fallback"


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
            time.sleep(0.3)
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *exc):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


# One sample shape for BOTH CPU legs (cpu_baseline of the default run, --impl reference): the first SAMPLE_SENSORS sensors x
# the first SAMPLE_PARAMS parameters x all N_t steps of the config's own block column - about 1.5 s of oracle time per
# F.m + F^T.d pair on 16 host cores at C3.  The full step is that time x N_d*N_m / (sample sensors x sample parameters): the
# oracle's cost is exactly proportional to both counts (independent dot products), and the line says so ("extrapolated").
SAMPLE_SENSORS, SAMPLE_PARAMS = 8, 75000


def sample_shape(w):
    return min(w.N_d, SAMPLE_SENSORS), min(w.N_m, SAMPLE_PARAMS)


def oracle_sample(F_s, m_s, d_s):
    """Times the CPU oracle (blocked C build) on a sample; returns (seconds matvec, seconds rmatvec, threads)."""
    from oracle import toeplitz_blocked as ob
    ob.build()
    t0 = time.perf_counter(); ob.matvec(F_s, m_s); t1 = time.perf_counter()
    ob.rmatvec(F_s, d_s); t2 = time.perf_counter()
    return t1 - t0, t2 - t1, ob.num_threads()


def sample_text(w, ns, npar, dt, scale, reps):
    return (f"oracle/toeplitz_blocked.c (direct O(N_t^2) block convolution, fp64) on sensors 0..{ns - 1} x parameters 0..{npar - 1} "
            f"x all {w.N_t} steps of the same workload: {dt:.2f} s per F.m + F^T.d pair (mean of {reps}), "
            f"x {scale:.1f} = N_d*N_m/(sample){' * k' if w.k_rhs > 1 else ''} to the full step")


def cpu_baseline(w, sample, target_s=12.0):
    """sample = (F_s [N_t,ns,npar], m_s [N_t,npar], d_s [N_t,ns]) numpy, the shape of sample_shape(w)."""
    F_s, m_s, d_s = sample
    ns, npar = F_s.shape[1], F_s.shape[2]
    ta, tb, thr = oracle_sample(F_s, m_s, d_s)            # warms the library and the caches
    reps = int(max(1, min(20, round(target_s / max(1e-3, ta + tb)))))
    acc_a = acc_b = 0.0
    for _ in range(reps):
        ta, tb, thr = oracle_sample(F_s, m_s, d_s)
        acc_a += ta; acc_b += tb
    ta, tb = acc_a / reps, acc_b / reps
    scale = (w.N_d * w.N_m) / float(ns * npar) * w.k_rhs   # k-RHS: the oracle does the columns one by one
    return {
        "value": (ta + tb) * scale * 1e3, "unit": "ms", "cores": thr, "kind": "oracle",
        "sample": sample_text(w, ns, npar, ta + tb, scale, reps), "extrapolated": True, "scale": scale,
        "sample_ms": (ta + tb) * 1e3, "matvec_ms": ta * scale * 1e3, "rmatvec_ms": tb * scale * 1e3,
        "note": "reported baseline (the oracle as it stands, O(N_t^2)), not the optimisation target",
    }


def cpu_fft_baseline(w, F_s, m, d_s, threads):
    """The paper's own ALGORITHM on the host cores (FFT along time, one matvec per frequency, inverse FFT),
    restated with library calls (torch.fft = pocketfft/MKL, torch.einsum) - a comparison row like the cuFFT + cuBLAS one, never
    part of libtt and not the oracle.  The spectrum of a SENSOR SLAB of the block column (all parameters, all steps) is
    computed untimed (plan cost); timed: rfft of the whole parameter vector, the per-frequency matvec against the slab's
    spectrum, irfft.  The matvec part streams the slab once and is scaled by N_d / (slab sensors); the FFT of m is not scaled."""
    torch.set_num_threads(threads)
    N_t, ns, N_m = F_s.shape
    L2 = 2 * N_t
    Fh = torch.fft.rfft(F_s.to(torch.float64), n=L2, dim=0).to(torch.complex64 if F_s.dtype == torch.float32 else torch.complex128)

    def fwd():
        t0 = time.perf_counter()
        mh = torch.fft.rfft(m, n=L2, dim=0)                         # [n_f, N_m]
        t1 = time.perf_counter()
        dh = torch.einsum("wsp,wp->ws", Fh, mh)
        t2 = time.perf_counter()
        torch.fft.irfft(dh, n=L2, dim=0)[:N_t]
        return t1 - t0, t2 - t1, time.perf_counter() - t2

    def adj():
        t0 = time.perf_counter()
        dh = torch.fft.rfft(d_s, n=L2, dim=0)                        # [n_f, ns]
        t1 = time.perf_counter()
        mh = torch.einsum("wsp,ws->wp", Fh.conj(), dh)
        t2 = time.perf_counter()
        torch.fft.irfft(mh, n=L2, dim=0)[:N_t]
        return t1 - t0, t2 - t1, time.perf_counter() - t2

    fwd(); adj()
    f, a = fwd(), adj()
    scale = w.N_d / float(ns)
    ms_f = (f[0] + f[1] * scale + f[2]) * 1e3
    ms_a = (a[0] + a[1] * scale + a[2]) * 1e3
    return {"value": ms_f + ms_a, "unit": "ms", "cores": threads, "kind": "cpu restatement of the FFT algorithm (torch.fft + einsum)",
            "matvec_ms": ms_f, "rmatvec_ms": ms_a, "extrapolated": True, "scale": scale,
            "sample": (f"spectrum of sensors 0..{ns - 1} (all {N_m} parameters, {N_t} steps) precomputed untimed; timed: rfft of m "
                       f"{f[0] * 1e3:.0f} ms, per-frequency matvec on the slab {f[1] * 1e3:.0f} ms (x {scale:.1f} = N_d/{ns}), irfft; "
                       f"adjoint: matvec on the slab {a[1] * 1e3:.0f} ms (x {scale:.1f}), irfft of the parameter vector {a[2] * 1e3:.0f} ms"),
            "note": "comparison row, not the oracle: the same method as libtt on the host cores (ADVICE r1)"}


def run_reference(args, w):
    """--impl reference: the oracle on the host cores, each step one bounded sample (the shape cpu_baseline uses), same metric."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    ns, npar = sample_shape(w)
    F_s = synth.block_column(w, s_range=(0, ns), p_range=(0, npar)).numpy()
    m_s = synth.vector_m(w.scaled(N_m=npar), k_rhs=1).numpy()
    d_s = synth.vector_d(w.scaled(N_d=ns), k_rhs=1).numpy()
    thr = 0
    for _ in range(args.warmup):
        _, _, thr = oracle_sample(F_s, m_s, d_s)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _, _, thr = oracle_sample(F_s, m_s, d_s)
    dt = (time.perf_counter() - t0) / args.steps
    scale = (w.N_d * w.N_m) / float(ns * npar) * w.k_rhs
    ms = dt * scale * 1e3
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": ms, "unit": "ms", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": config_dict(w, args),
        "cpu_baseline": {"value": ms, "unit": "ms", "cores": thr, "kind": "oracle",
                         "sample": sample_text(w, ns, npar, dt, scale, args.steps), "extrapolated": True, "scale": scale,
                         "sample_ms": dt * 1e3},
        "e2e": {"value": ms, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))
    return 0


def config_dict(w, args, cfg_name=None):
    return {"workload": f"{w.name}: N_d={w.N_d}, N_m={w.N_m}, N_t={w.N_t} ({w.n_params:.3g} parameters), "
                        f"{'fp32 vectors / complex64 spectrum' if w.dtype == torch.float32 else 'fp64 / complex128'}"
                        + (f", k={w.k_rhs} right-hand sides" if w.k_rhs > 1 else ""),
            "baseline_config": cfg_name or args.config,
            "step": "one F.m (A1,A2,A3) + one F^T.d (B1,B2,B3)" if w.k_rhs == 1
                    else f"one batched F.M + one batched F^T.D, k={w.k_rhs} (batched FFTs + per-frequency "
                         f"{'complex64 FMA' if w.dtype == torch.float32 else 'DMMA'} GEMMs)",
            "layout": "time-major",
            "out_every": getattr(args, "r_out", 1),
            "parallelism": (f"N_m sharded over {args.gpus} rank(s), one all-reduce of d per F.m" if args.parallel == "shard"
                            else "single GPU" if args.gpus == 1 else "replicas only"),
            "l2": "inputs larger than L2 (Fhat streamed once per op; no flush needed)"}


def kd_roofline(w, n, seconds, peaks):
    """tt_assemble_K_direct is a dense contraction: bound "tensor".  fp32 block columns run on tcgen05 kind::tf32 with three MMAs
    per product (hi/lo split), so the tensor work is 3 x the algorithmic flops; the tf32 peak is the measured bf16 figure of
    MEASURED_PEAKS.json x the guide's nominal tf32/bf16 ratio (1.1 / 2.25 PFLOP/s) - the sustained one: the call runs ~0.8 s under
    the power cap."""
    flops = float(n) * (n + 1) * w.N_m                 # lower triangle incl. diagonal, 2 flop per multiply-add
    if w.dtype != torch.float32:
        return {"bound": "tensor", "kernel": "kd_gemm_dmma_kernel (mma.sync m8n8k4 f64)", "achieved": flops / seconds * 1e-12,
                "unit": "TFLOP/s", "peak": None, "frac": None, "peak_kind": "FP64 DMMA: see the C4 leg of the default run (tt_probe_dmma)"}
    bf16 = peaks.get("bf16_tflops_sustained") or peaks.get("bf16_tflops")
    peak = bf16 * (1.1 / 2.25) if bf16 else None
    ach = 3.0 * flops / seconds * 1e-12
    return {"bound": "tensor", "kernel": "kd_umma_kernel (tcgen05.mma kind::tf32, 3 MMAs per fp32 product)", "achieved": ach,
            "unit": "TFLOP/s", "peak": peak, "frac": ach / peak if peak else None, "effective_fp32_TFLOPs": flops / seconds * 1e-12,
            "peak_kind": "MEASURED_PEAKS.json bf16_tflops_sustained x nominal tf32/bf16 ratio 1.1/2.25" if bf16 else "no measured peak",
            "tensor_flops_per_call": 3.0 * flops, "traffic": None,
            "ncu": "profiles/r2_kdirect_ncu_full.md: tensor pipe active 73.6 % of the cycles at N_m x 0.02"}


ONLINE_METRIC = "ms per online MAP inference, eq (4.13): m_map from d_obs (G*, F, K-solve, G*)"


def run_online(args, w):
    """--online: the online phase at the paper's own shape (P5: PAPER.md:370-381).

    Inputs of the online phase, all resident in HBM before the timed region: the spectra of F and of
    G* = Gamma_prior F* (synthetic block columns, synth.py), diag(Gamma_noise), and a Cholesky factor of the order
    of K (n = N_d N_t).  The factor is a seeded stand-in (synth.factor_standin): assembling the true K takes n
    matvec pairs; `--k-cols` columns of it ARE assembled with tt_assemble_K and timed.
    A step = one tt_map_infer in the paper's form (G*, F, two triangular solves, G*).
    """
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    from paper_2501_14911_b200 import binding as tt
    tt.lib()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    es = 4 if w.dtype == torch.float32 else 8
    n = w.N_d * w.N_t
    kb = max(1, args.k_batch)
    t0 = time.perf_counter()
    F = synth.block_column(w, device=dev)
    # K = Gamma_noise + F G* in one call from the two block columns (tt_assemble_K_direct), while both are resident
    G = synth.scaled_block_column(w, F)
    nv0 = synth.noise_var(w, device=dev)
    Kd = torch.empty((n, n), dtype=torch.float64, device=dev)
    tiny = (slice(0, 2), slice(0, min(w.N_d, 2)), slice(0, 64))
    tt.assemble_K_direct(F[tiny].contiguous(), G[tiny].contiguous(), nv0[:2, : min(w.N_d, 2)].contiguous())   # first-launch costs
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    tt.tt_assemble_K_direct(F, G, nv0, w.N_d, w.N_m, w.N_t, tt.TT_F32 if w.dtype == torch.float32 else tt.TT_F64, Kd, n)
    e1.record()
    torch.cuda.synchronize()
    s_direct = e0.elapsed_time(e1) * 1e-3
    kd_c0 = min(n // 2, n - min(n, args.k_cols))
    Kd_cols = Kd[:, kd_c0:kd_c0 + min(n, args.k_cols)].clone()       # compared below with the column-by-column route
    kd_sym = bool((Kd[: min(n, 4096)] == Kd[:, : min(n, 4096)].t()).all())
    # With all of K in hand the factor can be the real one: Cholesky by the library (cuSOLVER through torch; the paper's offline
    # factorisation is a library call too), libtt's triangular solves on it, checked by a residual.  If this K
    # (fp32 products) is not numerically SPD the seeded stand-in below is used and the line says so.
    true_K, chol, L_h = {"used": False}, None, None
    try:
        tc0 = time.perf_counter()
        L = torch.linalg.cholesky(Kd, upper=True).t()   # K = U^T U: cuSOLVER's column-major U is a row-major L
        L = L if L.stride(1) == 1 else L.contiguous()
        torch.cuda.synchronize()
        t_chol = time.perf_counter() - tc0
        chol = tt.Chol(L)
        L_h = L.cpu().numpy() if not args.no_cpu_baseline else None
        del L
        b_chk = torch.randn(n, dtype=torch.float64, device=dev)
        x_chk = chol.solve(b_chk)
        true_K = {"used": True, "cholesky_s_cusolver": t_chol,
                  "residual_of_tt_chol_solve": float((Kd @ x_chk - b_chk).norm() / b_chk.norm()),
                  "what": "L = chol(K) of the K assembled by tt_assemble_K_direct; |K x - b| / |b| for x = tt_chol_solve(b), b ~ N(0, I)"}
        v = torch.randn(n, dtype=torch.float64, device=dev)
        for _ in range(30):                              # power iteration: lambda_max(K); lambda_min(K) >= min(Gamma_noise)
            v = Kd @ v
            lam = float(v.norm())
            v /= lam
        true_K["cond_estimate"] = lam / float(nv0.min())
        true_K["cond_what"] = "lambda_max(K) by power iteration / min diag(Gamma_noise) (a lower bound of lambda_min: F G* is PSD)"
        del b_chk, x_chk, v
    except Exception as exc:
        true_K = {"used": False, "why": f"{type(exc).__name__}: {exc}"[:200]}
        if chol is not None:
            chol.close()
        chol, L_h = None, None
    del Kd, nv0
    torch.cuda.empty_cache()                         # libtt allocates with cudaMalloc: hand torch's cached blocks back first
    # --phase3: the dense Q and Gamma_post(q) from block columns (tt_qoi_direct), while G's block column is resident
    qoi_direct = None
    if args.phase3 and true_K["used"]:
        wq0 = synth.CONFIGS["Q5"]
        Fq0 = synth.block_column(wq0, device=dev)
        Gq0 = synth.scaled_block_column(wq0, Fq0)
        torch.cuda.empty_cache()
        torch.cuda.synchronize()
        tq0 = time.perf_counter()
        Q_dense, C_dense = tt.qoi_direct(Fq0, Gq0, G, 10, chol)
        torch.cuda.synchronize()
        qoi_direct = {"seconds": time.perf_counter() - tq0}
        del Fq0, Gq0
        torch.cuda.empty_cache()
    pF = tt.Plan(F, k_max=kb)
    del F
    torch.cuda.empty_cache()
    pG = tt.Plan(G, k_max=kb)
    F_s = None
    if not args.no_cpu_baseline:
        F_s = G[:, : min(w.N_d, 4), : min(w.N_m, SAMPLE_PARAMS)].contiguous().cpu().numpy()   # sample of G for the CPU leg
    del G
    torch.cuda.empty_cache()
    nv = synth.noise_var(w, device=dev)
    d_obs = synth.vector_d(w, device=dev, k_rhs=1)
    if chol is None:
        L = synth.factor_standin(n, w.seed, device=dev)
        chol = tt.Chol(L)
        L_h = L.cpu().numpy() if not args.no_cpu_baseline else None
        del L
    torch.cuda.empty_cache()
    mp = tt.MapInference(pF, pG, chol, nv)
    torch.cuda.synchronize()
    t_setup = time.perf_counter() - t0

    stream = torch.cuda.Stream(device=dev)
    m_map = torch.empty((w.N_t, w.N_m), dtype=w.dtype, device=dev)
    b64 = torch.randn(n, dtype=torch.float64, device=dev)
    x64 = torch.empty_like(b64)

    def time_op(fn, k):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record(stream)
        for _ in range(k):
            fn()
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / k

    paper = lambda: tt.tt_map_infer(mp.handle, tt.TT_MAP_PAPER, d_obs, m_map, stream)
    gain = lambda: tt.tt_map_infer(mp.handle, tt.TT_MAP_GAIN, d_obs, m_map, stream)
    for _ in range(args.warmup):
        paper(); gain()
    if true_K["used"]:   # with the factor of the true K the two forms of eq (4.13) are the same vector (reading R16)
        paper()
        stream.synchronize()          # the calls run on `stream`, the clone and the norms on torch's current stream
        m_p = m_map.clone()
        torch.cuda.synchronize()
        gain()
        stream.synchronize()
        true_K["paper_form_vs_gain_form_rel_l2"] = float((m_p - m_map).norm() / m_map.norm())
        true_K["paper_form_note"] = ("eq (4.13) as written forms z = y - K^-1 (F G* y): the roundings of the two matvecs (relative u of "
                                     "the plan dtype) are amplified by cond(K) before the subtraction, the gain form G* K^-1 d has no "
                                     "such cancellation (DESIGN.md section 11, tolerances: bar + 8 u cond(K))")
        del m_p
    with ClockSampler(0) as clocks:
        ms_paper = time_op(paper, args.steps)
    ms_gain = time_op(gain, args.steps)
    ms_solve = time_op(lambda: tt.tt_chol_solve(chol.handle, b64, x64, stream), 4 * args.steps)
    ms_fwd = time_op(lambda: tt.tt_chol_trsv(chol.handle, False, b64, x64, stream), 4 * args.steps)
    ms_bwd = time_op(lambda: tt.tt_chol_trsv(chol.handle, True, b64, x64, stream), 4 * args.steps)
    m_tmp = torch.empty_like(m_map)
    d_tmp = torch.empty_like(d_obs)
    ms_G = time_op(lambda: tt.tt_rmatvec(pG.handle, d_obs, m_tmp, stream), args.steps)
    ms_F = time_op(lambda: tt.tt_matvec(pF.handle, m_tmp, d_tmp, stream), args.steps)
    ms_smw = time_op(lambda: tt.tt_smw_apply(mp.handle, m_tmp, m_map, stream), args.steps)   # (I - G* K^-1 F) u, eq (4.7)/(4.8)
    del m_tmp

    # end to end with HOST vectors: d_obs in (98 KB), m_map out (526 MB)
    d_h = d_obs.cpu().pin_memory()
    m_h = torch.empty((w.N_t, w.N_m), dtype=w.dtype).pin_memory()
    tt.tt_map_infer_host(mp.handle, tt.TT_MAP_PAPER, d_h, m_h, stream)
    stream.synchronize()
    n_e2e = max(2, min(args.steps, 5))
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        tt.tt_map_infer_host(mp.handle, tt.TT_MAP_PAPER, d_h, m_h, stream)
    stream.synchronize()
    ms_e2e = (time.perf_counter() - t0) * 1e3 / n_e2e

    # Phase 3 actions (eq 4.10, 4.11) through the p2q plans of the paper's shape (N_q = 16, every 10th step), --phase3
    phase3 = None
    if args.phase3:
        wq = synth.CONFIGS["Q5"]
        r = 10
        Fq = synth.block_column(wq, device=dev)
        pFq = tt.Plan(Fq, out_every=r)
        synth.scaled_block_column(wq, Fq, out=Fq)
        pGq = tt.Plan(Fq, out_every=r)
        del Fq
        torch.cuda.empty_cache()
        vq = synth.vector_d(wq.scaled(N_t=wq.N_t // r), device=dev, k_rhs=1)
        qout = torch.empty_like(vq)
        work = torch.empty((2, w.N_t, w.N_m), dtype=w.dtype, device=dev)
        ms_pq = time_op(lambda: tt.tt_postcov_q_apply(mp.handle, pFq.handle, pGq.handle, vq, work, qout, stream), args.steps)
        ms_q = time_op(lambda: tt.tt_d2q_apply(mp.handle, pFq.handle, tt.TT_MAP_PAPER, d_obs, work, qout, stream), args.steps)
        ms_qg = time_op(lambda: tt.tt_d2q_apply(mp.handle, pFq.handle, tt.TT_MAP_GAIN, d_obs, work, qout, stream), args.steps)
        nq = wq.N_d * (wq.N_t // r)
        phase3 = {"postcov_q_action_ms": ms_pq, "all_columns_s": ms_pq * nq * 1e-3, "d2q_action_ms": ms_q,
                  "d2q_action_gain_form_ms": ms_qg, "n_qoi": nq,
                  "paper_timing_context": "PAPER.md:421-423: 48 ms per Gamma_post(q) action (38.4 s for 800), 56 ms per Q action, 24 A100"}
        if qoi_direct is not None:   # the dense matrices against the operator actions of the same run
            stream.synchronize()
            q_act = qout.double().reshape(-1).clone()                                 # tt_d2q_apply, gain form, of d_obs
            q_mat = Q_dense @ d_obs.double().reshape(-1)
            tt.tt_postcov_q_apply(mp.handle, pFq.handle, pGq.handle, vq, work, qout, stream)
            stream.synchronize()
            c_act = qout.double().reshape(-1)
            c_mat = C_dense @ vq.double().reshape(-1)
            qoi_direct.update({
                "what": "tt_qoi_direct: dense Q (800 x 24 500) and Gamma_post(q) (800 x 800) from the block columns of F_q, G_q and G "
                        "and the factor of K: two rectangular direct Toeplitz products, 800 K-solves, one GEMM; no matvecs",
                "Q_times_d_obs_vs_tt_d2q_apply_rel_l2": float((q_mat - q_act).norm() / q_act.norm()),
                "postcov_times_v_vs_tt_postcov_q_apply_rel_l2": float((c_mat - c_act).norm() / c_act.norm()),
                "postcov_symmetry_defect": float((C_dense - C_dense.t()).norm() / C_dense.norm()),
                "by_actions_s": (ms_pq + ms_qg) * nq * 1e-3,
                "paper_timing_context": "PAPER.md:421-423: 800 actions each: 38.4 s (Gamma_post(q)) + ~45 s (Q), 24 A100"})
            phase3["qoi_direct"] = qoi_direct
            del Q_dense, C_dense
        pFq.close(); pGq.close()
        del work
        torch.cuda.empty_cache()
        args.k_cols = min(args.k_cols, 4)

    # K assembly: a bounded number of columns, extrapolated like the paper does (n x time per column)
    kcols = min(n, args.k_cols)
    c0 = min(n // 2, n - kcols)
    Kbuf = torch.zeros((n, n), dtype=torch.float64, device=dev)
    tt.tt_assemble_K(pF.handle, pG.handle, nv, c0, min(kb, kcols), Kbuf, n, stream)   # warm-up: one batch (scratch, first launches)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    tt.tt_assemble_K(pF.handle, pG.handle, nv, c0, kcols, Kbuf, n, stream)
    torch.cuda.synchronize()
    s_cols = time.perf_counter() - t0
    Kd = Kbuf[c0:c0 + kcols, c0:c0 + kcols]
    sym = float((Kd - Kd.t()).abs().max() / Kd.abs().max())      # K is symmetric: its diagonal block must be
    direct_vs_cols = None
    if args.phase3 is False and c0 == kd_c0 and kcols == Kd_cols.shape[1]:
        direct_vs_cols = float((Kbuf[:, c0:c0 + kcols] - Kd_cols).norm() / Kd_cols.norm())
    del Kbuf, Kd, Kd_cols

    peaks, peak_kind = measured_peaks()
    peak = float(peaks.get("hbm_gbs", FALLBACK_HBM_GBS))
    lt_bytes = 64 * 64 * 8 * ((n + 63) // 64) * ((n + 63) // 64 - 1) // 2
    n_f, ldp = w.N_t + 1, (w.N_m + 15) // 16 * 16
    fhat_bytes = n_f * w.N_d * ldp * 2 * es
    vec = w.N_t * w.N_m * es
    out = {
        "metric": ONLINE_METRIC, "value": ms_paper, "unit": "ms", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_paper, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32 matvecs / f64 K-solve" if w.dtype == torch.float32 else "f64", "data": "synthetic",
        "config": {"workload": f"{w.name}: N_d={w.N_d}, N_m={w.N_m}, N_t={w.N_t} ({w.n_params:.4g} parameters, "
                               f"{n} data), online phase of PAPER.md:343-350",
                   "step": "tt_map_infer TT_MAP_PAPER: y = Gn^-1 d, a = G* y, b = F a, c = K^-1 b (two triangular solves), "
                           "m_map = G* (y - c)",
                   "factor": ("Cholesky factor of the true K = Gamma_noise + F G* (tt_assemble_K_direct, then cuSOLVER potrf)"
                              if true_K["used"] else
                              "seeded stand-in of order n (synth.factor_standin); timing is value independent"),
                   "l2": "inputs larger than L2 (two 52 GB spectra + 2.4 GB factor streamed per step)"},
        "e2e": {"value": ms_e2e, "unit": "ms", "h2d_bytes_per_step": n * es, "d2h_bytes_per_step": w.N_t * w.N_m * es,
                "steps": n_e2e, "api": "tt_map_infer_host, pinned host vectors"},
        "gpu_launches": (3 * 3 + 1 + 4 + 3) * args.steps,   # 2 x G* (3 each), F (4), 4 solve kernels, 3 element-wise
        "clocks": clocks.summary(),
        "roofline": {"bound": "hbm", "kernel": "trsv_fwd_kernel + trsv_bwd_kernel (the two triangular solves of the K-solve)",
                     "achieved": 2 * lt_bytes / (ms_solve * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                     "frac": 2 * lt_bytes / (ms_solve * 1e-3) / 1e9 / peak, "traffic": None,
                     "peak_kind": f"{peak_kind} copy bandwidth (MEASURED_PEAKS.json hbm_gbs)",
                     "algorithmic_bytes_per_solve": 2 * lt_bytes, "ms_per_solve": ms_solve,
                     "forward_ms": ms_fwd, "backward_ms": ms_bwd, "chain_steps": (n + 63) // 64,
                     "note": "latency chain of n/64 block steps on top of the stream; see DESIGN.md section 11"},
        "ops": {"map_paper_form_ms": ms_paper, "map_gain_form_ms": ms_gain, "Gstar_ms": ms_G, "F_ms": ms_F,
                "K_solve_ms": ms_solve, "smw_operator_ms": ms_smw,
                "smw_context": "(I - G* K^-1 F) u = the posterior covariance action of eq (4.7) without the prior solve; "
                               "PAPER.md:409: 11 + 11 + 20 ms on 24 A100 (+ 84 ms prior solve)",
                "paper_form_GBs": (3 * (fhat_bytes + vec) + 2 * lt_bytes) / (ms_paper * 1e-3) / 1e9,
                "gain_form_GBs": (fhat_bytes + vec + 2 * lt_bytes) / (ms_gain * 1e-3) / 1e9,
                "paper_timing_context": "PAPER.md:436-438: ~53 ms on 24 A100 (11 ms per G*/F, 20 ms K-solve)"},
        "factor": true_K,
        "K_assembly_direct": {"seconds": s_direct, "what": "tt_assemble_K_direct: all of K from the two block columns, one real GEMM "
                              "(lower triangle) + running sums down the block diagonals + mirror; no matvecs",
                              "multiply_adds": n * (n + 1) // 2 * w.N_m,
                              "TFLOPs": n * (n + 1) * w.N_m / s_direct * 1e-12,
                              "roofline": kd_roofline(w, n, s_direct, peaks),
                              "upper_equals_lower_transposed": kd_sym,
                              "rel_diff_vs_column_by_column": direct_vs_cols,
                              "paper_timing_context": "PAPER.md:407: 24 500 x 0.022 s ~ 9 min on 24 A100 (column by column)"},
        "K_assembly": {"columns_timed": kcols, "k_batch": kb, "s_per_column": s_cols / kcols,
                       "extrapolated_total_s": s_cols / kcols * n, "symmetry_defect_of_the_diagonal_block": sym,
                       "paper_timing_context": "PAPER.md:407: 24 500 x 0.022 s ~ 9 min on 24 A100"},
        "phase3": phase3,
        "setup": {"seconds": t_setup, "plan_bytes": pF.device_bytes + pG.device_bytes, "chol_bytes": chol.device_bytes},
    }
    if not args.no_cpu_baseline:
        from oracle import online_plain as oo
        from oracle import toeplitz_blocked as ob
        ob.build()
        d_np = d_obs.cpu().numpy()
        t0 = time.perf_counter(); z = oo.chol_solve(L_h, d_np.reshape(n).astype("float64")); t_solve = time.perf_counter() - t0
        ns, npar = F_s.shape[1], F_s.shape[2]
        zz = z.reshape(w.N_t, w.N_d)[:, :ns].copy()
        ob.rmatvec(F_s, zz)
        t0 = time.perf_counter(); ob.rmatvec(F_s, zz); t_g = time.perf_counter() - t0
        scale = (w.N_d * w.N_m) / float(ns * npar)
        out["cpu_baseline"] = {
            "value": (t_solve + 3 * t_g * scale) * 1e3, "unit": "ms", "cores": ob.num_threads(), "kind": "oracle",
            "sample": (f"oracle/online_plain.chol_solve at full order n={n} ({t_solve:.2f} s, numpy substitution loops) + 3 x "
                       f"oracle/toeplitz_blocked block convolution timed on {ns} sensors x {npar} parameters x {w.N_t} steps "
                       f"({t_g:.2f} s), scaled by {scale:.1f}"),
            "note": "reported baseline, not the optimisation target"}
    mp.close(); chol.close(); pF.close(); pG.close()
    print(json.dumps(out))
    return 0


def run_online_f64(args, w):
    """--online --f64: the gain form m_map = G* K^{-1} d_obs in the paper's own storage precision (fp64) at its
    own shape.  The complex128 spectrum of G* is 103 GB, so one B200 holds G* and the factor but not F as well (the form of
    eq 4.13 as written needs two GPUs: paper_2501_14911_b200/sharded.py); the 51.6 GB fp64 block column is drawn sensor slab
    by sensor slab on the device, kept in host memory and handed to tt_plan_create as a HOST pointer (streamed through 1 GiB)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    from paper_2501_14911_b200 import binding as tt
    tt.lib()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    w = w.scaled(dtype=torch.float64)
    n = w.N_d * w.N_t
    # all of K in fp64 from the two fp64 block columns (2 x 51.6 GB at P5), before the 103 GB spectrum is built
    F = synth.block_column(w, device=dev)
    G = synth.scaled_block_column(w, F)
    nv0 = synth.noise_var(w, device=dev)
    Kd = torch.empty((n, n), dtype=torch.float64, device=dev)
    tiny = (slice(0, 2), slice(0, min(w.N_d, 2)), slice(0, 64))
    tt.assemble_K_direct(F[tiny].contiguous(), G[tiny].contiguous(), nv0[:2, : min(w.N_d, 2)].contiguous())   # first-launch costs
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    tt.tt_assemble_K_direct(F, G, nv0, w.N_d, w.N_m, w.N_t, tt.TT_F64, Kd, n)
    e1.record()
    torch.cuda.synchronize()
    s_direct = e0.elapsed_time(e1) * 1e-3
    kd_sym = bool((Kd[: min(n, 4096)] == Kd[:, : min(n, 4096)].t()).all())
    del F, G, nv0
    torch.cuda.empty_cache()
    # With K itself in hand the factor is the real one: Cholesky by the library (cuSOLVER through torch - the paper's own
    # offline factorisation is a library call too), then libtt's triangular solves on it, checked by a residual.
    true_K = {"used": False}
    chol = None
    try:
        tc0 = time.perf_counter()
        L = torch.linalg.cholesky(Kd, upper=True).t()   # K = U^T U: L = U^T; cuSOLVER's column-major U is a row-major L
        L = L if L.stride(1) == 1 else L.contiguous()
        torch.cuda.synchronize()
        t_chol = time.perf_counter() - tc0
        chol = tt.Chol(L)
        del L
        b_chk = torch.randn(n, dtype=torch.float64, device=dev)
        x_chk = chol.solve(b_chk)
        res = float((Kd @ x_chk - b_chk).norm() / b_chk.norm())
        true_K = {"used": True, "cholesky_s_cusolver": t_chol, "residual_of_tt_chol_solve": res,
                  "what": "L = chol(K) of the K assembled above; |K x - b| / |b| for x = tt_chol_solve(b), b ~ N(0, I)"}
        del b_chk, x_chk
    except Exception as exc:   # K not numerically SPD, or no memory for the factorisation: report it, time with the stand-in
        true_K = {"used": False, "why": f"{type(exc).__name__}: {exc}"[:200]}
        if chol is not None:
            chol.close()
            chol = None
    del Kd
    torch.cuda.empty_cache()
    t0 = time.perf_counter()
    G_h = torch.empty((w.N_t, w.N_d, w.N_m), dtype=torch.float64).pin_memory()
    for s0 in range(0, w.N_d, 4):
        s1 = min(w.N_d, s0 + 4)
        slab = synth.block_column(w, device=dev, s_range=(s0, s1))
        synth.scaled_block_column(w, slab, out=slab)
        G_h[:, s0:s1, :] = slab.cpu()
        del slab
    torch.cuda.empty_cache()
    t_gen = time.perf_counter() - t0
    t0 = time.perf_counter()
    pG = tt.Plan(G_h)
    torch.cuda.synchronize()
    t_plan = time.perf_counter() - t0
    del G_h
    nv = synth.noise_var(w, device=dev)
    d_obs = synth.vector_d(w, device=dev, k_rhs=1)
    if chol is None:
        L = synth.factor_standin(n, w.seed, device=dev)
        chol = tt.Chol(L)
        del L
    torch.cuda.empty_cache()
    mp = tt.MapInference(None, pG, chol, nv)
    stream = torch.cuda.Stream(device=dev)
    m_map = torch.empty((w.N_t, w.N_m), dtype=torch.float64, device=dev)

    def time_op(fn, k):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record(stream)
        for _ in range(k):
            fn()
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / k

    gain = lambda: tt.tt_map_infer(mp.handle, tt.TT_MAP_GAIN, d_obs, m_map, stream)
    for _ in range(args.warmup):
        gain()
    with ClockSampler(0) as clocks:
        ms_gain = time_op(gain, args.steps)
    b64 = torch.randn(n, dtype=torch.float64, device=dev)
    ms_solve = time_op(lambda: tt.tt_chol_solve(chol.handle, b64, b64, stream), 4 * args.steps)
    ms_G = time_op(lambda: tt.tt_rmatvec(pG.handle, d_obs, m_map, stream), args.steps)
    peaks, peak_kind = measured_peaks()
    peak = float(peaks.get("hbm_gbs", FALLBACK_HBM_GBS))
    ghat = (w.N_t + 1) * w.N_d * ((w.N_m + 15) // 16 * 16) * 16
    lt_bytes = 64 * 64 * 8 * ((n + 63) // 64) * ((n + 63) // 64 - 1) // 2
    out = {
        "metric": "ms per online MAP inference in fp64, gain form m_map = G* K^-1 d_obs", "value": ms_gain, "unit": "ms",
        "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_gain, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{w.name} in fp64: N_d={w.N_d}, N_m={w.N_m}, N_t={w.N_t}, complex128 spectrum of G* {ghat / 1e9:.1f} GB",
                   "step": "tt_map_infer TT_MAP_GAIN: K-solve (two triangular solves) + one G* action",
                   "factor": ("Cholesky factor of the true K = Gamma_noise + F G* (tt_assemble_K_direct, then cuSOLVER potrf)"
                              if true_K["used"] else "seeded stand-in of order n (synth.factor_standin)"),
                   "l2": "inputs larger than L2"},
        "gpu_launches": 9 * args.steps, "clocks": clocks.summary(),
        "roofline": {"bound": "hbm", "kernel": "gemv_adj_kernel<double> (B2 of the G* action)",
                     "achieved": (ghat + 2 * lt_bytes + w.N_t * w.N_m * 8) / (ms_gain * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                     "frac": (ghat + 2 * lt_bytes + w.N_t * w.N_m * 8) / (ms_gain * 1e-3) / 1e9 / peak, "traffic": None,
                     "peak_kind": f"{peak_kind} copy bandwidth; achieved = (|Ghat| + 2 |Lt| + |m_map|) / step time"},
        "ops": {"map_gain_form_ms": ms_gain, "Gstar_ms": ms_G, "K_solve_ms": ms_solve,
                "parity": "tests/test_gpu_fullsize.py::test_online_fp64_full_parameter_dimension (sampled outputs vs the oracle)",
                "paper_timing_context": "PAPER.md:436-438: ~53 ms on 24 A100 for eq (4.13) as written, fp64 storage"},
        "K_assembly_direct": {"seconds": s_direct, "what": "tt_assemble_K_direct, TT_F64: all of K from the two fp64 block columns "
                              "(DMMA GEMM of the lower triangle + running sums down the block diagonals + mirror)",
                              "multiply_adds": n * (n + 1) // 2 * w.N_m, "TFLOPs": n * (n + 1) * w.N_m / s_direct * 1e-12,
                              "upper_equals_lower_transposed": kd_sym,
                              "parity": "tests/test_gpu_online.py::test_assemble_K_direct (fp64: 1e-12 against the oracle)",
                              "paper_timing_context": "PAPER.md:407: 24 500 x 0.022 s ~ 9 min on 24 A100 (column by column, fp64)"},
        "factor": true_K,
        "setup": {"block_column_generation_s": t_gen, "plan_create_from_host_s": t_plan,
                  "device_bytes": pG.device_bytes + chol.device_bytes},
    }
    mp.close(); chol.close(); pG.close()
    print(json.dumps(out))
    return 0


class Ctx:
    def __init__(self, **kw):
        self.__dict__.update(kw)


def measure(ctx, args, w, cfg_name, *, steps, warmup, headline):
    """One config through the C ABI on this rank's GPU: the timed step (F.m + F^T.d, or the k-RHS pair), per-op times,
    the roofline object of SURVEY.md 8(d) and - for the headline config only - e2e, bandwidth probes, the library
    comparison row and the CPU legs.  Returns the JSON object (rank 0 prints it)."""
    tt, dev, dist, rank, world = ctx.tt, ctx.dev, ctx.dist, ctx.rank, ctx.world
    es = 4 if w.dtype == torch.float32 else 8

    # ---- inputs, resident in HBM ----------------------------------------------------------
    t0 = time.perf_counter()
    shard = args.parallel == "shard"
    K = w.k_rhs                                   # > 1: the k-RHS batched calls (C4)
    w_full = w
    if shard:
        from paper_2501_14911_b200 import sharded
        p0, p1 = sharded.shard_range(w.N_m, rank, world)
        F = synth.block_column(w, device=dev, p_range=(p0, p1))
        m = synth.vector_m(w, device=dev)[:, p0:p1].contiguous()
        w = w.scaled(N_m=p1 - p0)                 # byte counts below are this rank's
    else:
        F = synth.block_column(w, device=dev)
        m = synth.vector_m(w, device=dev)         # [N_t, N_m] or [N_t, N_m, K]
    r_out = args.out_every or (10 if cfg_name == "Q5" else 1)
    args.r_out = r_out
    d = synth.vector_d(w.scaled(N_t=w.N_t // r_out), device=dev)
    torch.cuda.synchronize()
    t_gen = time.perf_counter() - t0
    lib_baseline = headline and K == 1 and world == 1 and r_out == 1 and not args.no_library_baseline
    cpu_legs = headline and rank == 0 and world == 1 and not args.no_cpu_baseline

    sample = fft_sample = None
    if cpu_legs:   # the CPU legs' samples: the same bytes, copied from the device before the column is freed
        ns, npar = sample_shape(w)
        m1 = m if K == 1 else m[..., 0]
        d1 = d if K == 1 else d[..., 0]
        if r_out > 1:                       # the oracle applies F^T to S^T d: zeros at the steps that are not sampled
            up = torch.zeros((w.N_t,) + tuple(d1.shape[1:]), dtype=d1.dtype, device=d1.device)
            up[r_out - 1::r_out] = d1
            d1 = up
        sample = (F[:, :ns, :npar].contiguous().cpu().numpy(), m1[:, :npar].contiguous().cpu().numpy(),
                  d1[:, :ns].contiguous().cpu().numpy())
        if K == 1 and r_out == 1:
            nsf = min(w.N_d, 4)
            fft_sample = (F[:, :nsf, :].contiguous().cpu(), m1.cpu(), d1[:, :nsf].contiguous().cpu())

    t0 = time.perf_counter()
    plan = tt.Plan(F, k_max=K, out_every=r_out)
    torch.cuda.synchronize()
    t_plan = time.perf_counter() - t0
    del F
    torch.cuda.empty_cache()

    stream = torch.cuda.Stream(device=dev)
    d_out = torch.empty_like(d)
    m_out = torch.empty_like(m)
    h = plan.handle
    describe = tt.tt_plan_describe(h)

    if K == 1:
        op_fwd = lambda: tt.tt_matvec(h, m, d_out, stream)
        op_adj = lambda: tt.tt_rmatvec(h, d, m_out, stream)
        tag_fwd, tag_adj = tt.TT_OP_MATVEC, tt.TT_OP_RMATVEC
    else:
        op_fwd = lambda: tt.tt_matvec_batched(h, K, m, d_out, stream)
        op_adj = lambda: tt.tt_rmatvec_batched(h, K, d, m_out, stream)
        tag_fwd, tag_adj = tt.TT_OP_MATVEC_BATCHED, tt.TT_OP_RMATVEC_BATCHED

    if shard and dist is not None:  # F.m = local partial + the path's one exchange step; F^T.d needs no collective
        local_fwd = op_fwd

        def op_fwd():
            local_fwd()
            with torch.cuda.stream(stream):
                dist.all_reduce(d_out, op=dist.ReduceOp.SUM)

    def step():
        op_fwd()
        op_adj()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x: float) -> float:
        if dist is None:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    with torch.cuda.stream(stream):
        for _ in range(warmup):
            step()
    barrier()

    # ---- timed region: device-resident ------------------------------------------------------
    tt.tt_plan_set_profiling(h, True)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(ctx.local_rank) as clocks:
        barrier()
        ev0.record(stream)
        for _ in range(steps):
            step()
        ev1.record(stream)
        barrier()
    ms_step = max_over_ranks(ev0.elapsed_time(ev1) / steps)
    fwd = tt.tt_plan_stage_ms(h, tag_fwd)
    adj = tt.tt_plan_stage_ms(h, tag_adj)
    tt.tt_plan_set_profiling(h, False)

    # ---- separate ms per F.m and per F^T.d (same launch configuration) -----------------------
    def time_op(fn, n):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record(stream)
        for _ in range(n):
            fn()
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / n

    def time_each(fn, n):
        """Per-call device times (one CUDA event pair per call): median and min over n calls (SURVEY.md 8(d) protocol)."""
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        torch.cuda.synchronize()
        for a, b in evs:
            a.record(stream)
            fn()
            b.record(stream)
        torch.cuda.synchronize()
        t = sorted(a.elapsed_time(b) for a, b in evs)
        return {"median": t[len(t) // 2], "min": t[0], "calls": n}

    ms_fwd = max_over_ranks(time_op(op_fwd, steps))
    ms_adj = max_over_ranks(time_op(op_adj, steps))
    n_each = (max(20, steps) if K == 1 else max(5, steps)) if headline else steps
    each_fwd, each_adj = time_each(op_fwd, n_each), time_each(op_adj, n_each)
    ms_normal = None
    if K == 1:  # F^T F m (one solver iteration, configs[4]); the intermediate d never leaves the device
        n_out = torch.empty_like(m)
        for _ in range(2):
            tt.tt_normal(h, m, n_out, stream)
        ms_normal = max_over_ranks(time_op(lambda: tt.tt_normal(h, m, n_out, stream), steps))
        del n_out

    # ---- end to end through the C ABI with HOST vectors -------------------------------------
    e2e = None
    if headline:
        m_h, d_h = m.cpu().pin_memory(), d.cpu().pin_memory()
        d_oh, m_oh = torch.empty_like(d_h).pin_memory(), torch.empty_like(m_h).pin_memory()
        if K == 1:
            def step_host():
                tt.tt_matvec_host(h, m_h, d_oh, stream)
                tt.tt_rmatvec_host(h, d_h, m_oh, stream)
            e2e_api = "tt_matvec_host + tt_rmatvec_host, pinned host vectors"
        else:
            def step_host():  # no *_host variant of the k-RHS calls: explicit copies on the same stream
                with torch.cuda.stream(stream):
                    m.copy_(m_h, non_blocking=True)
                    tt.tt_matvec_batched(h, K, m, d_out, stream)
                    d_oh.copy_(d_out, non_blocking=True)
                    d.copy_(d_h, non_blocking=True)
                    tt.tt_rmatvec_batched(h, K, d, m_out, stream)
                    m_oh.copy_(m_out, non_blocking=True)
            e2e_api = "pinned host -> device copies + tt_matvec_batched / tt_rmatvec_batched + device -> host copies"
        step_host()
        torch.cuda.synchronize()
        n_e2e = max(2, min(steps, 5 if K == 1 else 2))
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            step_host()
        stream.synchronize()
        ms_e2e = max_over_ranks((time.perf_counter() - t0) * 1e3 / n_e2e)
        e2e = {"value": ms_e2e if shard else ms_e2e / args.gpus, "unit": "ms",
               "h2d_bytes_per_step": (m_h.numel() + d_h.numel()) * es, "d2h_bytes_per_step": (d_oh.numel() + m_oh.numel()) * es,
               "steps": n_e2e, "api": e2e_api}
        del m_h, d_h, d_oh, m_oh

    # ---- roofline of the dominant kernel -----------------------------------
    peaks, peak_kind = measured_peaks()
    peak = float(peaks.get("hbm_gbs", FALLBACK_HBM_GBS))
    n_f, ldp = w.N_t + 1, (w.N_m + 15) // 16 * 16
    fhat_bytes = n_f * w.N_d * ldp * 2 * es
    vec_bytes = (w.N_t * w.N_m + (w.N_t // r_out) * w.N_d) * es * K
    bytes_op = fhat_bytes + vec_bytes                           # 8(d): |Fhat| + |m| + |d| per op; un-fused intermediates
    if K == 1:                                                  # (mhat, partials) count against the achieved figure
        xhat_bytes = n_f * ldp * 2 * es
        dhat_bytes = n_f * w.N_d * 2 * es
        chunk = 2048 if n_f * ((ldp + 4095) // 4096) < 148 * 2 * 8 else 4096      # the planner's choice (tt_api.cu)
        n_chunks = (ldp + chunk - 1) // chunk
        part_bytes = n_f * n_chunks * w.N_d * 2 * es
        bytes_fwd_kernel = fhat_bytes + xhat_bytes + part_bytes     # what A2 itself moves: Fhat + xhat read, partials written
        bytes_adj_kernel = fhat_bytes + dhat_bytes + xhat_bytes     # B2: Fhat + dhat read, xhat written
        ach_fwd = bytes_op / (fwd[1] * 1e-3) / 1e9 if fwd[1] > 0 else 0.0
        ach_adj = bytes_op / (adj[1] * 1e-3) / 1e9 if adj[1] > 0 else 0.0
        traffic, traffic_src = None, "no committed ncu capture of this config"
        rec = NCU_TRAFFIC.get(cfg_name)
        if rec is not None:
            if rec["kernel"] in describe and not shard:
                traffic, traffic_src = rec["bytes"], f"{rec['profile']} ({rec['kernel']})"
            else:
                traffic_src = f"{rec['profile']} was captured with '{rec['kernel']}', this run launches '{describe}'"
        roofline = {
            "bound": "hbm", "kernel": "gemv_fwd_kernel (A2, per-frequency matvec streaming Fhat)",
            "achieved": ach_fwd, "peak": peak, "unit": "GB/s", "frac": ach_fwd / peak,
            "traffic": traffic, "traffic_source": traffic_src,
            "peak_kind": f"{peak_kind} copy bandwidth (MEASURED_PEAKS.json hbm_gbs)" if peak_kind == "measured"
                         else "fallback 6.65 TB/s (B200_PROFILING.md)",
            "how": "achieved = algorithmic bytes per op (|Fhat| + |m| + |d|, SURVEY.md 8(d)) / mean duration of the dominant "
                   "kernel's launches in the timed region (CUDA events recorded by libtt on the launching stream)",
            "algorithmic_bytes_per_launch": bytes_op, "ms_per_launch": fwd[1], "launches_timed": fwd[3],
            "frac_of_nominal_8TBs": ach_fwd / NOMINAL_HBM_GBS,
            "kernel_bytes_per_launch": bytes_fwd_kernel,
            "achieved_kernel_bytes": bytes_fwd_kernel / (fwd[1] * 1e-3) / 1e9 if fwd[1] > 0 else 0.0,
            "whole_op": {"matvec_frac": bytes_op / (ms_fwd * 1e-3) / 1e9 / peak, "rmatvec_frac": bytes_op / (ms_adj * 1e-3) / 1e9 / peak,
                         "what": "the same bytes / the whole F.m and F^T.d (FFTs and un-fused intermediates included)"},
            "adjoint_kernel": {"kernel": "gemv_adj_kernel (B2)" + (", with the persistent B3 consumer CTAs running beside it" if "B3 consumer" in describe else ""),
                               "achieved": ach_adj, "frac": ach_adj / peak,
                               "algorithmic_bytes_per_launch": bytes_op, "kernel_bytes_per_launch": bytes_adj_kernel,
                               "ms_per_launch": adj[1], "frac_of_nominal_8TBs": ach_adj / NOMINAL_HBM_GBS},
            "kernels": describe,
        }
    elif w.dtype == torch.float32 and K % 16 == 0:
        # fp32 k-RHS, k a multiple of 16: per-frequency complex64 GEMMs on tcgen05 kind::tf32 with three MMAs per product
        # (3xTF32, tt_gemm32_umma.cu).  Tensor work = 3 x the algorithmic flops; the tf32 peak is the measured bf16 figure of
        # MEASURED_PEAKS.json x the guide's nominal tf32/bf16 ratio.  These GEMMs are short and fat (N_d x 2k outputs per
        # frequency): each also streams Fhat and the k spectra once, so both rooflines are computed and the nearer one named.
        peaks, _ = measured_peaks()
        bf16 = peaks.get("bf16_tflops_sustained") or peaks.get("bf16_tflops")
        peak_t = bf16 * (1.1 / 2.25) if bf16 else None
        flops = 8.0 * n_f * w.N_d * w.N_m * K
        hbm_bytes = fhat_bytes + n_f * w.N_m * K * 8
        ach_fwd = 3.0 * flops / (fwd[1] * 1e-3) / 1e12 if fwd[1] > 0 else 0.0
        ach_adj = 3.0 * flops / (adj[1] * 1e-3) / 1e12 if adj[1] > 0 else 0.0
        adj_umma = w.N_d <= 128
        hbm_fwd = hbm_bytes / (fwd[1] * 1e-3) / 1e9 if fwd[1] > 0 else 0.0
        hbm_adj = hbm_bytes / (adj[1] * 1e-3) / 1e9 if adj[1] > 0 else 0.0
        tensor = {"achieved": ach_fwd, "peak": peak_t, "unit": "TFLOP/s", "frac": ach_fwd / peak_t if peak_t else None,
                  "peak_kind": "MEASURED_PEAKS.json bf16_tflops(_sustained) x nominal tf32/bf16 ratio 1.1/2.25" if bf16 else "no measured peak",
                  "effective_fp32_TFLOPs": flops / (fwd[1] * 1e-3) / 1e12 if fwd[1] > 0 else 0.0,
                  "algorithmic_flops_per_launch": flops, "tensor_flops_per_launch": 3.0 * flops,
                  "adjoint": {"achieved": ach_adj if adj_umma else None, "frac": ach_adj / peak_t if (peak_t and adj_umma) else None,
                              "effective_fp32_TFLOPs": flops / (adj[1] * 1e-3) / 1e12 if adj[1] > 0 else 0.0}}
        hbm = {"achieved": hbm_fwd, "peak": peak, "unit": "GB/s", "frac": hbm_fwd / peak,
               "peak_kind": f"{peak_kind} copy bandwidth (MEASURED_PEAKS.json hbm_gbs)" if peak_kind == "measured"
                            else "fallback 6.65 TB/s (B200_PROFILING.md)",
               "algorithmic_bytes_per_launch": hbm_bytes, "adjoint": {"achieved": hbm_adj, "frac": hbm_adj / peak}}
        # the roofline that binds is the one the kernel sits closer to: at the paper's shapes (N_d 49 - 100, k 32) that is HBM
        # (every launch streams Fhat and the k spectra once), with the tensor pipe at about half of its 3xTF32 ceiling
        hbm_binds = tensor["frac"] is None or hbm["frac"] >= tensor["frac"]
        first, second = (hbm, tensor) if hbm_binds else (tensor, hbm)
        roofline = {
            "bound": "hbm" if hbm_binds else "tensor",
            "kernel": "gemm32_umma_fwd_kernel (k-RHS A2: per-frequency complex64 GEMM, tcgen05.mma kind::tf32, A from tensor "
                      "memory, 3 MMAs per fp32 product)",
            "achieved": first["achieved"], "peak": first["peak"], "unit": first["unit"], "frac": first["frac"], "traffic": None,
            "peak_kind": first["peak_kind"], "ms_per_launch": fwd[1], "launches_timed": fwd[3],
            "how": "both rooflines of the kernel are computed from the same event-timed launches (algorithmic bytes = |Fhat| + "
                   "k spectra; tensor work = 3 MMAs x 8 flop per complex multiply-add); `bound` names the one with the larger fraction",
            "hbm": hbm, "tensor": tensor, "other_bound": second["frac"],
            "adjoint_kernel": {"kernel": "gemm32_umma_adj_kernel (k-RHS B2, tcgen05, TMA-stored tiles)" if adj_umma
                                         else "gemm32_adj_kernel (k-RHS B2, FP32 FMA: N_d > 128)",
                               "achieved": (hbm if hbm_binds else tensor)["adjoint"]["achieved"],
                               "frac": (hbm if hbm_binds else tensor)["adjoint"]["frac"], "ms_per_launch": adj[1]},
        }
    elif w.dtype == torch.float32:
        # fp32 k-RHS, k not a multiple of 16: register-tiled complex64 FMA GEMMs (tt_gemm32.cu), bound by the FP32 FMA pipe.  Peak derived from the
        # unit counts of the guide: 148 SMs x 128 FP32 FMA lanes x 2 flop x the SM clock sampled during this run.
        clk = clocks.summary().get("sm_mhz") or 1965.0
        peak32 = 148 * 128 * 2 * clk * 1e6 / 1e12
        flops = 8.0 * n_f * w.N_d * w.N_m * K
        ach_fwd = flops / (fwd[1] * 1e-3) / 1e12 if fwd[1] > 0 else 0.0
        ach_adj = flops / (adj[1] * 1e-3) / 1e12 if adj[1] > 0 else 0.0
        roofline = {
            "bound": "alu", "kernel": "gemm32_fwd_kernel (k-RHS A2: per-frequency complex64 GEMM, FP32 FMA)",
            "achieved": ach_fwd, "peak": peak32, "unit": "TFLOP/s", "frac": ach_fwd / peak32, "traffic": None,
            "peak_kind": f"148 SMs x 128 FMA lanes x 2 flop x {clk:.0f} MHz (nominal FP32 FMA rate; three-register FFMA issues "
                         "every other cycle per sub-partition on this part, so ~half of it is the practical ceiling)",
            "algorithmic_flops_per_launch": flops, "ms_per_launch": fwd[1], "launches_timed": fwd[3],
            "hbm_bytes_per_launch": fhat_bytes + n_f * w.N_m * K * 8,
            "adjoint_kernel": {"kernel": "gemm32_adj_kernel (k-RHS B2)", "achieved": ach_adj, "frac": ach_adj / peak32,
                               "ms_per_launch": adj[1]},
        }
    else:
        # the k-RHS per-frequency GEMMs are a dense contraction on the FP64 tensor pipe (DMMA); its peak is
        # measured in this run by the library's DMMA probe (there is no FP64 figure in MEASURED_PEAKS.json)
        sink = torch.empty(148 * 8 * 256, dtype=torch.float64, device=dev)
        best = 0.0
        for _ in range(3):
            fl = [0.0]
            t = time_op(lambda: fl.__setitem__(0, tt.tt_probe_dmma(4000, sink, stream)), 3)
            best = max(best, fl[0] / (t * 1e-3) / 1e12)
        flops = 8.0 * n_f * w.N_d * w.N_m * K                  # 4 real MACs per complex MAC
        ach_fwd = flops / (fwd[1] * 1e-3) / 1e12 if fwd[1] > 0 else 0.0
        ach_adj = flops / (adj[1] * 1e-3) / 1e12 if adj[1] > 0 else 0.0
        roofline = {
            "bound": "tensor", "kernel": "gemm_fwd_kernel (k-RHS A2: per-frequency complex GEMM, mma.sync m8n8k4 f64)",
            "achieved": ach_fwd, "peak": best, "unit": "TFLOP/s", "frac": ach_fwd / best if best else None,
            "traffic": None, "peak_kind": "FP64 DMMA peak measured in this run by tt_probe_dmma "
                                          "(bf16 measured 1620 TF/s x nominal fp64/bf16 ratio 40/2250 = 28.8 TF/s for comparison)",
            "algorithmic_flops_per_launch": flops, "ms_per_launch": fwd[1], "launches_timed": fwd[3],
            "hbm_bytes_per_launch": fhat_bytes + n_f * w.N_m * K * 16,
            "whole_op": {"matvec_TFLOPs": flops / (ms_fwd * 1e-3) / 1e12, "rmatvec_TFLOPs": flops / (ms_adj * 1e-3) / 1e12,
                         "matvec_frac": flops / (ms_fwd * 1e-3) / 1e12 / best if best else None,
                         "rmatvec_frac": flops / (ms_adj * 1e-3) / 1e12 / best if best else None,
                         "what": "the same flops / the whole batched F.M and F^T.D (batched FFTs included)"},
            "adjoint_kernel": {"kernel": "gemm_adj_kernel (k-RHS B2)", "achieved": ach_adj,
                               "frac": ach_adj / best if best else None, "ms_per_launch": adj[1]},
        }

    # ---- bandwidth probes in the same run (copy and read-only stream) -------------------------
    probe = None
    if headline:
        probe = {}
        try:
            nb = 8 << 30
            a = torch.empty(nb, dtype=torch.uint8, device=dev); a.zero_()
            b = torch.empty(nb, dtype=torch.uint8, device=dev)
            sink = torch.empty(1 << 16, dtype=torch.uint8, device=dev)
            with torch.cuda.stream(stream):
                probe["read_only_gbs"] = nb / (min(time_op(lambda: tt.tt_probe_stream_read(a, nb, sink, stream), 5)
                                                   for _ in range(3)) * 1e-3) / 1e9
                probe["copy_gbs"] = 2 * nb / (min(time_op(lambda: b.copy_(a), 5) for _ in range(3)) * 1e-3) / 1e9
            del a, b
        except RuntimeError as e:  # pragma: no cover
            probe["error"] = str(e)

    # ---- comparison row: the same operation with library FFTs and batched library matmuls ------
    # (torch.fft = cuFFT, torch.bmm = cuBLAS; timed on the plan's own spectrum, never linked into libtt)
    libs = None
    if lib_baseline:
        try:
            Fv = tt.tt_debug_spectrum_view(h, w.N_t, w.N_d, w.dtype)[:, :, :w.N_m]
            L2 = 2 * w.N_t

            def lib_fwd():
                mh_ = torch.fft.rfft(m, n=L2, dim=0)                       # [n_f, N_m]
                dh_ = torch.bmm(Fv, mh_.unsqueeze(2)).squeeze(2)           # [n_f, N_d]
                return torch.fft.irfft(dh_, n=L2, dim=0)[:w.N_t]

            def lib_adj():
                dh_ = torch.fft.rfft(d, n=L2, dim=0)                       # [n_f, N_d]
                mh_ = torch.bmm(Fv.conj().transpose(1, 2), dh_.unsqueeze(2)).squeeze(2)
                return torch.fft.irfft(mh_, n=L2, dim=0)[:w.N_t]

            with torch.cuda.stream(stream):
                r1, r2 = lib_fwd(), lib_adj()
                e1 = float((r1 - d_out).norm() / d_out.norm()); e2 = float((r2 - m_out).norm() / m_out.norm())
                del r1, r2
                t_lf = time_op(lib_fwd, max(2, steps // 2))
                t_la = time_op(lib_adj, max(2, steps // 2))
            libs = {"what": "torch.fft.rfft/irfft (cuFFT) + torch.bmm over frequencies (cuBLAS) on the same spectrum",
                    "matvec_ms": t_lf, "rmatvec_ms": t_la, "rel_diff_vs_libtt": [e1, e2]}
            del Fv
        except Exception as e:  # e.g. out of memory for the library temporaries
            libs = {"error": str(e)[:200]}
            torch.cuda.empty_cache()

    launches_per_step = 7                      # A1, A2 (matvec or GEMM), partial reduce, A3, B1, B2, B3
    if K == 1 and "B3 consumer" in describe:   # F^T d in producer / consumer mode: B3 consumer beside B2, clean-up B3 behind it
        launches_per_step = 8
    out = {
        "metric": METRIC, "value": ms_step if shard else ms_step / args.gpus, "unit": "ms", "n_gpus": args.gpus,
        "steps": steps,
        "warmup": warmup, "ms_per_step": ms_step, "higher_is_better": False, "scaling": "strong" if shard else "weak",
        "vs_baseline": None, "dtype": "f32" if w.dtype == torch.float32 else "f64", "data": "synthetic",
        "config": config_dict(w_full, args, cfg_name),
        "e2e": e2e,
        "gpu_launches": launches_per_step * steps,
        "clocks": clocks.summary(),
        "roofline": roofline,
        "ops": {
            "matvec_ms": ms_fwd, "rmatvec_ms": ms_adj, "normal_ms": ms_normal, "k_rhs": K,
            "matvec_ms_per_call": each_fwd, "rmatvec_ms_per_call": each_adj,
            "normal_GBs": (2 * fhat_bytes + 2 * w.N_t * w.N_m * es) / (ms_normal * 1e-3) / 1e9 if ms_normal else None,
            "normal_frac_of_measured_copy": (2 * fhat_bytes + 2 * w.N_t * w.N_m * es) / (ms_normal * 1e-3) / 1e9 / peak if ms_normal else None,
            "matvec_GBs": bytes_op / (ms_fwd * 1e-3) / 1e9, "rmatvec_GBs": bytes_op / (ms_adj * 1e-3) / 1e9,
            "roofline_bytes_per_op": bytes_op,
            "matvec_frac_of_8TBs": bytes_op / (ms_fwd * 1e-3) / 1e9 / NOMINAL_HBM_GBS,
            "rmatvec_frac_of_8TBs": bytes_op / (ms_adj * 1e-3) / 1e9 / NOMINAL_HBM_GBS,
            "matvec_frac_of_measured_copy": bytes_op / (ms_fwd * 1e-3) / 1e9 / peak,
            "rmatvec_frac_of_measured_copy": bytes_op / (ms_adj * 1e-3) / 1e9 / peak,
            "stages_matvec_ms": {"A1_fft": fwd[0], "A2_gemv": fwd[1], "A3_reduce_ifft": fwd[2]},
            "stages_rmatvec_ms": {"B1_fft": adj[0], "B2_gemv": adj[1], "B3_ifft": adj[2]},
        },
        "probe": probe,
        "library_baseline": libs,
        "plan": {"create_s": t_plan, "device_bytes": plan.device_bytes, "input_generation_s": t_gen},
    }
    if shard:
        out["exchange"] = {"collective": "NCCL all-reduce (sum) of d, N_d*N_t reals, once per F.m" if dist is not None else "none (single process)",
                           "world_size": world, "bytes": d_out.numel() * es}
    plan.close()
    del m, d, d_out, m_out
    torch.cuda.empty_cache()

    # ---- CPU legs: the oracle (and the FFT algorithm restated with library calls) on this box's host cores -----
    if sample is not None:
        out["cpu_baseline"] = cpu_baseline(w, sample)
        if fft_sample is not None:
            try:
                out["cpu_fft_baseline"] = cpu_fft_baseline(w, *fft_sample, threads=out["cpu_baseline"]["cores"])
            except Exception as exc:
                out["cpu_fft_baseline"] = {"error": f"{type(exc).__name__}: {exc}"[:200]}
    return out


def summarise_leg(leg, name):
    """The short legs of the other BASELINE.json configs inside the default line: ms, GB/s or TFLOP/s, roofline, clocks."""
    ops, rf = leg["ops"], leg["roofline"]
    keep = {"workload": leg["config"]["workload"], "steps": leg["steps"], "warmup": leg["warmup"], "ms_per_step": leg["ms_per_step"],
            "dtype": leg["dtype"], "matvec_ms": ops["matvec_ms"], "rmatvec_ms": ops["rmatvec_ms"], "normal_ms": ops["normal_ms"],
            "k_rhs": ops["k_rhs"], "clocks": leg["clocks"], "gpu_launches": leg["gpu_launches"],
            "stages_matvec_ms": ops["stages_matvec_ms"], "stages_rmatvec_ms": ops["stages_rmatvec_ms"],
            "plan_device_bytes": leg["plan"]["device_bytes"]}
    if rf["bound"] == "hbm":
        keep.update({"matvec_GBs": ops["matvec_GBs"], "rmatvec_GBs": ops["rmatvec_GBs"], "normal_GBs": ops["normal_GBs"],
                     "roofline_bytes_per_op": ops["roofline_bytes_per_op"]})
    keep["roofline"] = {k: rf[k] for k in ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic", "peak_kind",
                                            "ms_per_launch", "launches_timed", "whole_op", "adjoint_kernel") if k in rf}
    if name == "C5":   # configs[4] is quoted on the normal operator: Fhat streamed twice
        keep["headline_op"] = {"op": "tt_normal (F^T F m)", "ms": ops["normal_ms"], "GBs": ops["normal_GBs"],
                               "frac_of_measured_copy": ops["normal_frac_of_measured_copy"]}
    return keep


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C3", choices=sorted(synth.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "shard"],
                    help="N>1: independent replicas (default, the north star's one-GPU path) or the parameter axis "
                         "sharded over the ranks with one all-reduce of d per F.m (paper_2501_14911_b200/sharded.py)")
    ap.add_argument("--online", action="store_true",
                    help="time the online phase (eq 4.13 MAP inference, K-solve, K assembly) instead of the matvec pair; "
                         "meant for --config P5, the paper's own shape")
    ap.add_argument("--f64", action="store_true",
                    help="--online: the gain form in fp64 (the paper's storage precision): complex128 spectrum of G* (103 GB at P5)")
    ap.add_argument("--phase3", action="store_true",
                    help="--online: also time the Phase 3 actions Gamma_post(q) v (eq 4.10) and Q d_obs (eq 4.11) with the p2q plans")
    ap.add_argument("--k-cols", type=int, default=64, help="--online: columns of K assembled and timed")
    ap.add_argument("--k-batch", type=int, default=1, help="--online: right-hand sides per batched call in tt_assemble_K")
    ap.add_argument("--k-rhs", type=int, default=0,
                    help="run the k-RHS batched calls with k right-hand sides on any config (default: the config's own, "
                         "32 for C4, else 1); fp32 configs then take the complex64 GEMM path (tcgen05 for k a multiple of 16)")
    ap.add_argument("--out-every", type=int, default=0,
                    help="data side on every r-th time step (tt_plan_create_coarse); default 10 for Q5 (the p2q map), else 1")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-library-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true",
                    help="default C3 run at N=1: skip the short C5 / C2 / C4 legs reported under `configs`")
    ap.add_argument("--scale-nm", type=float, default=1.0,
                    help="multiply the config's N_m by this factor: for profiler captures of long kernels only (ncu replays a "
                         "kernel ~40 times and saves / restores device memory around each pass); the line it prints names the "
                         "scaled workload and is not a bench line of the config")
    ap.add_argument("--two-launch-rmatvec", action="store_true",
                    help="for profiler captures: F^T d as B2 then B3 (tt_debug_set l2r_mb = 0).  The default form runs B3 as "
                         "persistent consumer CTAs BESIDE B2; a profiler that serialises kernels makes those CTAs give up "
                         "after 50 ms and shows the clean-up B3 doing all the work - correct, but not the timeline of a real run")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    w = synth.CONFIGS[args.config]
    if args.scale_nm != 1.0:
        w = w.scaled(N_m=max(1, int(w.N_m * args.scale_nm)), name=f"{w.name} with N_m x {args.scale_nm:g} (profiler capture, not a bench line)")
    if args.k_rhs > 0:
        w = w.scaled(k_rhs=args.k_rhs)
    if args.impl == "reference":
        return run_reference(args, w)
    if args.online:
        return run_online_f64(args, w) if args.f64 else run_online(args, w)

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libtt has no CPU path")
    torch.cuda.set_device(local_rank)
    dist = None
    # one process per GPU under torchrun; a single rank launched by torchrun (RANK set, WORLD_SIZE = 1) with --parallel shard
    # also brings NCCL up, so that the exchange step of the sharded path runs through the real collective on one GPU
    if world > 1 or (args.parallel == "shard" and "RANK" in os.environ and "MASTER_ADDR" in os.environ):
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    from paper_2501_14911_b200 import binding as tt
    tt.lib()
    if args.two_launch_rmatvec:
        tt.tt_debug_set("l2r_mb", 0)
    ctx = Ctx(tt=tt, dev=torch.device("cuda", local_rank), dist=dist, rank=rank, world=world, local_rank=local_rank)

    out = measure(ctx, args, w, args.config, steps=args.steps, warmup=args.warmup, headline=True)

    # ---- the other BASELINE.json configs, short legs in the same invocation (driver-timed; N = 1 only) ----
    if world == 1 and args.config == "C3" and not args.no_other_configs and args.k_rhs == 0 and args.scale_nm == 1.0 \
            and args.parallel == "replicas":
        others = {}
        for name in ("C5", "C2", "C4"):
            try:
                torch.cuda.empty_cache()
                wo = synth.CONFIGS[name]
                leg = measure(ctx, args, wo, name, steps=5 if wo.k_rhs > 1 else 10, warmup=3, headline=False)
                others[name] = summarise_leg(leg, name)
            except Exception as exc:   # a failed leg must not take the headline line with it
                others[name] = {"error": f"{type(exc).__name__}: {exc}"[:300]}
        out["configs"] = others

    if rank == 0:
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
