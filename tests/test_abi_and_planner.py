"""CPU-only checks of the boundary and the planner's host logic (no compute calls, no GPU):
libtt.so builds, loads and exports every symbol include/tt.h declares; the FFT plan tables
(radices, digit-reversal slots, twiddles) reproduce numpy's FFT when the kernel's in-place
decimation-in-frequency recurrence is replayed on the host."""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def tt():
    from paper_2501_14911_b200 import binding
    binding.lib()
    return binding


def declared_symbols(header="tt.h"):
    with open(os.path.join(ROOT, "include", header)) as f:
        src = re.sub(r"/\*.*?\*/", "", f.read(), flags=re.S)
    return sorted(set(re.findall(r"\b(tt_[A-Za-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(tt):
    names = declared_symbols()
    assert "tt_plan_create" in names and "tt_matvec" in names and "tt_rmatvec" in names
    assert "tt_normal" in names and "tt_matvec_batched" in names and len(names) >= 18
    assert not any(n.startswith(("tt_probe", "tt_debug")) for n in names)   # the product ABI carries no probes or tuning knobs
    L = tt.lib()
    for n in names:
        assert hasattr(L, n), f"libtt.so does not export {n}"
    assert sorted(tt.EXPORTS) == names        # the binding wraps exactly the declared calls
    for n in names:
        assert hasattr(tt, n)
    # developer hooks (include/tt_dev.h, same library) and bench.py's probes (include/tt_probe.h, libttprobe.so)
    dev = declared_symbols("tt_dev.h")
    assert sorted(tt.DEV_EXPORTS) == dev
    for n in dev:
        assert hasattr(L, n) and hasattr(tt, n)
    probes = declared_symbols("tt_probe.h")
    assert sorted(tt.PROBE_EXPORTS) == probes
    P = tt.probe_lib()
    for n in probes:
        assert hasattr(P, n) and hasattr(tt, n) and not hasattr(L, n)


def test_version_and_status_strings(tt):
    assert tt.tt_version() >= 100
    assert tt.tt_status_string(0) == "TT_OK"
    assert tt.tt_status_string(-5) == "TT_ERR_UNSUPPORTED_NT"
    assert tt.tt_status_string(-10) == "TT_ERR_NO_DEVICE"
    assert tt.tt_status_string(-999) == "TT_ERR_UNKNOWN"


def test_no_gpu_means_loud_failure_not_fallback(tt):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import ctypes
    out = ctypes.c_void_p()
    buf = (ctypes.c_double * 64)()
    st = tt.lib().tt_plan_create(ctypes.byref(out), 2, 4, 8, tt.TT_F64, 0, 1, ctypes.addressof(buf), None)
    assert tt.tt_status_string(st) == "TT_ERR_NO_DEVICE" and out.value is None


def replay_dif(z, radices, tw):
    """The kernel's in-place DIF stages (tt_fft.cu: fft_stage) on one series, in numpy."""
    x = np.array(z, dtype=np.complex128)
    N = len(x)
    Ns = N
    for r in radices:
        M = Ns // r
        for blk in range(N // Ns):
            for j in range(M):
                idx = blk * Ns + j + M * np.arange(r)
                a = x[idx]
                y = np.array([np.sum(a * np.exp(-2j * np.pi * np.arange(r) * q / r)) for q in range(r)])
                if M > 1:
                    y = y * tw[j * np.arange(r) * (N // Ns) * 2]
                x[idx] = y
        Ns = M
    return x


@pytest.mark.parametrize("max_radix", [25, 8], ids=["fp32plan", "fp64plan"])
@pytest.mark.parametrize("N_t", [1, 2, 3, 4, 5, 6, 7, 8, 12, 15, 21, 32, 35, 49, 50, 60, 64, 100, 210, 256, 400, 500, 512])
def test_fft_plan_tables_reproduce_numpy_fft(tt, N_t, max_radix):
    radices, pos, tw = tt.tt_debug_fft_tables(N_t, max_radix)
    assert int(np.prod(radices)) == N_t if radices else N_t == 1
    assert all(r in (2, 3, 4, 5, 7, 8, 16, 20, 25) and r <= max_radix for r in radices)
    assert sorted(pos.tolist()) == list(range(N_t))                     # a permutation
    L = 2 * N_t
    k = np.arange(L)
    assert np.abs(tw - np.exp(-2j * np.pi * k / L)).max() < 5e-15           # numpy rounds the argument
    assert tw[0] == 1.0 and tw[N_t] == -1.0                              # exact on the axes
    rng = np.random.default_rng(N_t)
    x = rng.standard_normal(N_t)                                        # one real series
    xp = np.concatenate([x, np.zeros(N_t + (N_t % 2))])                 # zero padding (room for odd N_t)
    z = xp[0:2 * N_t:2] + 1j * xp[1:2 * N_t:2]                          # z_n = x_2n + i x_2n+1
    Z = replay_dif(z, radices, tw)[pos]                                 # natural order via pos
    assert np.abs(Z - np.fft.fft(z)).max() < 1e-11 * max(1.0, np.abs(Z).max())
    # the real-FFT post-processing of fft_r2c_kernel: X_k, k = 0..N_t, of the length-2N_t padded series
    kk = np.arange(N_t + 1)
    Zk, Zn = Z[kk % N_t], np.conj(Z[(N_t - kk) % N_t])
    X = 0.5 * (Zk + Zn) + tw[kk] * (-0.5j) * (Zk - Zn)
    ref = np.fft.rfft(np.concatenate([x, np.zeros(N_t)]))
    assert np.abs(X - ref).max() < 1e-11 * max(1.0, np.abs(ref).max())


def test_compile_time_trig_matches_libm(tt):
    """cos/sin(2 pi k/n) used for the butterflies' internal twiddles: exact on the axes, <= 2 ulp elsewhere."""
    two_pi = 2 * np.longdouble("3.14159265358979323846264338327950288")    # 80-bit reference
    for n in (3, 5, 7, 8, 16, 20, 25):
        for k in range(-n, 2 * n + 1):
            c, s = tt.tt_debug_trig(k, n)
            a = two_pi * np.longdouble(k % n) / np.longdouble(n)
            assert abs(np.longdouble(c) - np.cos(a)) < 2.3e-16 and abs(np.longdouble(s) - np.sin(a)) < 2.3e-16
    assert tt.tt_debug_trig(0, 16) == (1.0, 0.0) and tt.tt_debug_trig(4, 16) == (0.0, 1.0)
    assert tt.tt_debug_trig(8, 16) == (-1.0, 0.0) and tt.tt_debug_trig(12, 16) == (0.0, -1.0)
    c, s = tt.tt_debug_trig(2, 16)
    assert c == s                                                       # (1 - i)/sqrt(2) symmetric


@pytest.mark.parametrize("N_t", [11, 13, 22, 65536 * 2])
def test_unsupported_nt(tt, N_t):
    with pytest.raises(tt.TTError) as e:
        tt.tt_debug_fft_tables(N_t)
    assert e.value.status == -5


def test_online_phase_argument_validation_without_a_gpu(tt):
    """Host logic of the second half of include/tt.h: shape / NULL checks come before any device work."""
    import ctypes
    L = tt.lib()
    out = ctypes.c_void_p()
    buf = (ctypes.c_double * 16)()
    assert tt.tt_status_string(L.tt_chol_create(ctypes.byref(out), 0, buf, 4, None)) == "TT_ERR_SHAPE"
    assert tt.tt_status_string(L.tt_chol_create(ctypes.byref(out), 4, buf, 3, None)) == "TT_ERR_SHAPE"     # ld < n
    assert tt.tt_status_string(L.tt_chol_create(ctypes.byref(out), 4, None, 4, None)) == "TT_ERR_NULL"
    assert tt.tt_status_string(L.tt_chol_create(None, 4, buf, 4, None)) == "TT_ERR_NULL"
    assert tt.tt_status_string(L.tt_chol_solve(None, buf, buf, None)) == "TT_ERR_NULL"
    assert tt.tt_status_string(L.tt_map_create(ctypes.byref(out), None, None, None, buf, None)) == "TT_ERR_NULL"
    assert tt.tt_status_string(L.tt_map_infer(None, 0, buf, buf, None)) == "TT_ERR_NULL"
    assert tt.tt_status_string(L.tt_assemble_K(None, None, buf, 0, 1, buf, 4, None)) == "TT_ERR_NULL"
    # coarse output grid: out_every must divide N_t (checked before the device is touched)
    for bad in (0, 3, 64):
        st = L.tt_plan_create_coarse(ctypes.byref(out), 2, 8, 32, bad, tt.TT_F64, tt.TT_TIME_MAJOR, 1, buf, None)
        assert tt.tt_status_string(st) == "TT_ERR_SHAPE"
    L.tt_chol_destroy(None); L.tt_map_destroy(None)        # NULL-safe
    assert L.tt_chol_device_bytes(None) == 0
    assert tt.tt_status_string(-11) == "TT_ERR_NOT_SPD" and tt.tt_status_string(-12) == "TT_ERR_MISMATCH"
