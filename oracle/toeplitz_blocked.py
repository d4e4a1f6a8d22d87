"""CPU ORACLE (test infrastructure) - ctypes front end of toeplitz_blocked.c.

Builds oracle/libtto.so with gcc (-O3 -march=native -fopenmp) on first use and
whenever the source or the host CPU changed (the repo snapshot travels from
the build container to the GPU box, whose CPU may differ), then exposes

    matvec(F, m)   -> d   fp64 [N_t, N_d]      eq (2.5)
    rmatvec(F, d)  -> m'  fp64 [N_t, N_m]      its transpose

for fp32 or fp64 inputs (converted exactly to fp64 inside).  F may be any
slice F[:, s0:s1, p0:p1] of the block column whose last axis is contiguous
(strides are passed through), which is how bench.py times a bounded sample.

Shares no code with the CUDA path; only tests/, smoke() and bench.py's
cpu_baseline / --impl reference leg may import it.
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "toeplitz_blocked.c")
_LIB = os.path.join(_HERE, "libtto.so")
_SIG = os.path.join(_HERE, "libtto.sig")
_lib = None


def _host_signature() -> str:
    h = hashlib.sha256()
    with open(_SRC, "rb") as f:
        h.update(f.read())
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith(("model name", "flags")):
                    h.update(line.encode())
                    if line.startswith("flags"):
                        break
    except OSError:
        pass
    return h.hexdigest()


def build(force: bool = False) -> str:
    """Compile the C oracle for this host if needed; returns the library path."""
    sig = _host_signature()
    if not force and os.path.exists(_LIB) and os.path.exists(_SIG):
        with open(_SIG) as f:
            if f.read().strip() == sig:
                return _LIB
    tmp = _LIB + f".tmp{os.getpid()}"
    cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-shared", "-fPIC", "-std=c11",
           "-o", tmp, _SRC]
    subprocess.run(cmd, check=True, capture_output=True)
    os.replace(tmp, _LIB)
    with open(_SIG, "w") as f:
        f.write(sig)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i64, vp = ctypes.c_int64, ctypes.c_void_p
        for name in ("tto_matvec_f64", "tto_matvec_f32", "tto_rmatvec_f64", "tto_rmatvec_f32"):
            fn = getattr(lib, name)
            fn.argtypes = [i64, i64, i64, vp, i64, i64, vp, i64, vp, i64]
            fn.restype = None
        lib.tto_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def num_threads() -> int:
    """OpenMP threads the C oracle will use (the `cores` of bench.py's cpu_baseline)."""
    return int(_load().tto_num_threads())


def _prep(F, v):
    F = np.asarray(F)
    if F.dtype not in (np.float32, np.float64):
        F = F.astype(np.float64)
    assert F.ndim == 3 and F.strides[2] == F.itemsize, "last axis of F must be contiguous"
    v = np.ascontiguousarray(np.asarray(v), dtype=F.dtype)
    assert v.ndim == 2 and v.shape[0] == F.shape[0]
    return F, v


def matvec(F, m) -> np.ndarray:
    F, m = _prep(F, m)
    N_t, N_d, N_m = F.shape
    assert m.shape[1] == N_m
    d = np.empty((N_t, N_d), dtype=np.float64)
    fn = _load().tto_matvec_f64 if F.dtype == np.float64 else _load().tto_matvec_f32
    it = F.itemsize
    fn(N_d, N_m, N_t, F.ctypes.data, F.strides[0] // it, F.strides[1] // it,
       m.ctypes.data, N_m, d.ctypes.data, N_d)
    return d


def rmatvec(F, d) -> np.ndarray:
    F, d = _prep(F, d)
    N_t, N_d, N_m = F.shape
    assert d.shape[1] == N_d
    out = np.empty((N_t, N_m), dtype=np.float64)
    fn = _load().tto_rmatvec_f64 if F.dtype == np.float64 else _load().tto_rmatvec_f32
    it = F.itemsize
    fn(N_d, N_m, N_t, F.ctypes.data, F.strides[0] // it, F.strides[1] // it,
       d.ctypes.data, N_d, out.ctypes.data, N_m)
    return out


def normal(F, m) -> np.ndarray:
    """F^T (F m) (eq 2.12 with identity noise covariance); the intermediate d stays fp64."""
    F = np.asarray(F)
    d = matvec(F, m)
    return rmatvec(np.asarray(F, dtype=np.float64) if F.dtype != np.float64 else F, d)
