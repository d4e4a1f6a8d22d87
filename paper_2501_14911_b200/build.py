"""Builds paper_2501_14911_b200/libtt.so (the C-ABI library of include/tt.h) with nvcc for sm_100a.

    python -m paper_2501_14911_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The library is built in-tree so that it travels with the
repo snapshot to the GPU box; object files go to paper_2501_14911_b200/build/ (git-ignored).
A source/flag hash next to the library skips the rebuild when nothing changed.
"""
from __future__ import annotations

import hashlib
import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
BUILD = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libtt.so")
PROBE_LIB = os.path.join(HERE, "libttprobe.so")     # include/tt_probe.h: bench.py's hardware probes, not part of libtt
STAMP = os.path.join(BUILD, "libtt.stamp")

SOURCES = ["tt_api.cu", "tt_fft.cu", "tt_gemv.cu", "tt_gemm.cu", "tt_gemm32.cu", "tt_gemm32_umma.cu", "tt_trsv.cu", "tt_online.cu", "tt_kdirect.cu", "tt_kdirect_umma.cu"]
PROBE_SOURCE = "tt_probe.cu"
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC",
    "-Xptxas", "-v",
    "--expt-relaxed-constexpr",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libtt cannot be built (there is no CPU fallback)")


def _hash() -> str:
    h = hashlib.sha256()
    h.update(" ".join(NVCC_FLAGS).encode())
    names = sorted(os.listdir(CSRC)) + ["../../include/tt.h", "../../include/tt_dev.h", "../../include/tt_probe.h"]
    for name in names:
        path = os.path.join(CSRC, name)
        if os.path.isfile(path):
            h.update(name.encode())
            with open(path, "rb") as f:
                h.update(f.read())
    return h.hexdigest()


def is_current() -> bool:
    """True if libtt.so exists and its stamp carries the hash of the sources and flags in this tree."""
    if not (os.path.exists(LIB) and os.path.exists(PROBE_LIB) and os.path.exists(STAMP)):
        return False
    with open(STAMP) as f:
        return f.read().strip() == _hash()


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile and link libtt.so if needed; returns its path."""
    sig = _hash()
    if not force and os.path.exists(LIB) and os.path.exists(PROBE_LIB) and os.path.exists(STAMP):
        with open(STAMP) as f:
            if f.read().strip() == sig:
                return LIB
    os.makedirs(BUILD, exist_ok=True)
    nvcc = _nvcc()

    def compile_one(src: str) -> str:
        obj = os.path.join(BUILD, src.replace(".cu", ".o"))
        cmd = [nvcc, *NVCC_FLAGS, "-I", INCLUDE, "-c", os.path.join(CSRC, src), "-o", obj]
        res = subprocess.run(cmd, capture_output=True, text=True)
        with open(obj + ".log", "w") as f:
            f.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{res.stdout}\n{res.stderr}")
        if verbose:
            sys.stderr.write(res.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES) + 1) as ex:
        objs = list(ex.map(compile_one, SOURCES + [PROBE_SOURCE]))
    for lib, lib_objs in ((LIB, objs[:-1]), (PROBE_LIB, objs[-1:])):
        tmp = lib + f".tmp{os.getpid()}"
        cmd = [nvcc, "-shared", "-o", tmp, *lib_objs, "-cudart", "shared"]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode != 0:
            raise RuntimeError(f"link failed:\n{res.stdout}\n{res.stderr}")
        os.replace(tmp, lib)
    with open(STAMP, "w") as f:
        f.write(sig)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
