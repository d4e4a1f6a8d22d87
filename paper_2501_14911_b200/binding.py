"""Thin Python binding of libtt (include/tt.h): argument marshalling only.

Every function has the name and the argument order of the C call it wraps; tensors are
passed as raw pointers (`tensor.data_ptr()`), streams as `torch.cuda.Stream.cuda_stream`.
PyTorch is used for device memory and streams only; every step of the path runs in the
library's own CUDA kernels.  If libtt.so cannot be built or loaded this module raises:
there is no CPU or PyTorch fallback.
"""
from __future__ import annotations

import ctypes
import os

import torch

from . import build as _build

TT_F32, TT_F64 = 0, 1
TT_TIME_MAJOR, TT_SPACE_MAJOR = 0, 1
TT_OK = 0
TT_OP_MATVEC, TT_OP_RMATVEC, TT_OP_NORMAL, TT_OP_MATVEC_BATCHED, TT_OP_RMATVEC_BATCHED = range(5)
TT_MAP_PAPER, TT_MAP_GAIN = 0, 1

_lib = None


class TTError(RuntimeError):
    def __init__(self, call: str, status: int, cuda_error: int = 0):
        self.status = status
        self.cuda_error = cuda_error
        name = lib().tt_status_string(status).decode()
        extra = f" (cudaError {cuda_error})" if cuda_error else ""
        super().__init__(f"{call} failed: {name} [{status}]{extra}")


def lib() -> ctypes.CDLL:
    """Loads (building first if needed) paper_2501_14911_b200/libtt.so."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if not os.path.exists(path) or os.environ.get("TT_REBUILD") == "1":
        path = _build.build()
    else:
        try:
            path = _build.build()  # no-op when the source hash matches
        except RuntimeError as exc:
            # no nvcc on this box: the library that travelled with the repo is only good if it was built from these sources
            if not _build.is_current():
                raise RuntimeError(f"{path} was built from other sources than paper_2501_14911_b200/csrc (hash mismatch) and "
                                   f"cannot be rebuilt here: {exc}") from exc
    L = ctypes.CDLL(path)
    vp, i64, ci, sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_size_t
    pp = ctypes.POINTER(vp)
    sigs = {
        "tt_version": (ci, []),
        "tt_status_string": (ctypes.c_char_p, [ci]),
        "tt_plan_create": (ci, [pp, i64, i64, i64, ci, ci, ci, vp, vp]),
        "tt_plan_create_coarse": (ci, [pp, i64, i64, i64, i64, ci, ci, ci, vp, vp]),
        "tt_plan_destroy": (None, [vp]),
        "tt_plan_device_bytes": (sz, [vp]),
        "tt_plan_last_cuda_error": (ci, [vp]),
        "tt_plan_get_spectrum": (ci, [vp, vp, vp]),
        "tt_plan_describe": (ci, [vp, ctypes.c_char_p, sz]),
        "tt_matvec": (ci, [vp, vp, vp, vp]),
        "tt_rmatvec": (ci, [vp, vp, vp, vp]),
        "tt_normal": (ci, [vp, vp, vp, vp]),
        "tt_matvec_batched": (ci, [vp, ci, vp, vp, vp]),
        "tt_rmatvec_batched": (ci, [vp, ci, vp, vp, vp]),
        "tt_normal_batched": (ci, [vp, ci, vp, vp, vp]),
        "tt_matvec_host": (ci, [vp, vp, vp, vp]),
        "tt_rmatvec_host": (ci, [vp, vp, vp, vp]),
        "tt_normal_host": (ci, [vp, vp, vp, vp]),
        "tt_plan_set_profiling": (ci, [vp, ci]),
        "tt_plan_stage_ms": (ci, [vp, ci, ctypes.POINTER(ctypes.c_float), ci]),
        "tt_debug_fft_tables": (ci, [i64, ci, ctypes.POINTER(ci), ctypes.POINTER(ci),
                                     ctypes.POINTER(ctypes.c_ushort), ctypes.POINTER(ctypes.c_double)]),
        "tt_debug_spectrum_view": (ci, [vp, pp, ctypes.POINTER(i64)]),
        "tt_debug_trig": (ci, [i64, i64, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]),
        "tt_debug_set": (ci, [ctypes.c_char_p, ci]),
        "tt_chol_create": (ci, [pp, i64, vp, i64, vp]),
        "tt_chol_destroy": (None, [vp]),
        "tt_chol_device_bytes": (sz, [vp]),
        "tt_chol_last_cuda_error": (ci, [vp]),
        "tt_chol_solve": (ci, [vp, vp, vp, vp]),
        "tt_chol_trsv": (ci, [vp, ci, vp, vp, vp]),
        "tt_assemble_K": (ci, [vp, vp, vp, i64, i64, vp, i64, vp]),
        "tt_assemble_K_direct": (ci, [vp, vp, vp, i64, i64, i64, ci, vp, i64, vp]),
        "tt_assemble_K_direct_static": (ci, [vp, vp, vp, i64, i64, i64, ci, vp, i64, vp]),
        "tt_K_add_noise": (ci, [vp, i64, ci, vp, i64, vp]),
        "tt_qoi_direct": (ci, [vp, vp, vp, i64, i64, i64, i64, i64, ci, vp, vp, i64, vp, i64, vp]),
        "tt_map_create": (ci, [pp, vp, vp, vp, vp, vp]),
        "tt_map_destroy": (None, [vp]),
        "tt_map_infer": (ci, [vp, ci, vp, vp, vp]),
        "tt_map_infer_host": (ci, [vp, ci, vp, vp, vp]),
        "tt_smw_apply": (ci, [vp, vp, vp, vp]),
        "tt_postcov_q_apply": (ci, [vp, vp, vp, vp, vp, vp, vp]),
        "tt_d2q_apply": (ci, [vp, vp, ci, vp, vp, vp, vp]),
        "tt_map_infer_partial": (ci, [vp, vp, vp, vp, vp]),
        "tt_map_infer_finish": (ci, [vp, vp, vp, vp]),
    }
    for name, (res, args) in sigs.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    _lib = L
    return L


EXPORTS = ["tt_version", "tt_status_string", "tt_plan_create", "tt_plan_create_coarse", "tt_plan_destroy", "tt_plan_device_bytes",
           "tt_plan_last_cuda_error", "tt_plan_get_spectrum", "tt_plan_describe", "tt_matvec", "tt_rmatvec", "tt_normal",
           "tt_matvec_batched", "tt_rmatvec_batched", "tt_normal_batched", "tt_matvec_host", "tt_rmatvec_host", "tt_normal_host",
           "tt_plan_set_profiling", "tt_plan_stage_ms",
           "tt_chol_create", "tt_chol_destroy", "tt_chol_device_bytes", "tt_chol_last_cuda_error", "tt_chol_solve",
           "tt_chol_trsv", "tt_assemble_K", "tt_assemble_K_direct", "tt_assemble_K_direct_static", "tt_K_add_noise", "tt_qoi_direct", "tt_map_create", "tt_map_destroy", "tt_map_infer", "tt_map_infer_host",
           "tt_map_infer_partial", "tt_map_infer_finish", "tt_smw_apply",
           "tt_postcov_q_apply", "tt_d2q_apply"]


# developer hooks (include/tt_dev.h: exported by libtt.so, not part of the product ABI) and the probe library (include/tt_probe.h)
DEV_EXPORTS = ["tt_debug_spectrum_view", "tt_debug_fft_tables", "tt_debug_trig", "tt_debug_set"]
PROBE_EXPORTS = ["tt_probe_stream_read", "tt_probe_dmma"]
_probe = None


def probe_lib() -> ctypes.CDLL:
    """Loads paper_2501_14911_b200/libttprobe.so (built together with libtt.so)."""
    global _probe
    if _probe is None:
        lib()
        P = ctypes.CDLL(_build.PROBE_LIB)
        vp, ci, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t
        P.tt_probe_stream_read.restype, P.tt_probe_stream_read.argtypes = ci, [vp, sz, vp, vp]
        P.tt_probe_dmma.restype, P.tt_probe_dmma.argtypes = ci, [ci, vp, ctypes.POINTER(ctypes.c_double), vp]
        _probe = P
    return _probe


def _stream(stream) -> int:
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def _check(call: str, status: int, plan: int | None = None):
    if status != TT_OK:
        ce = lib().tt_plan_last_cuda_error(plan) if plan else 0
        raise TTError(call, status, ce)


def tt_version() -> int:
    return lib().tt_version()


def tt_status_string(status: int) -> str:
    return lib().tt_status_string(status).decode()


def tt_plan_create(N_d: int, N_m: int, N_t: int, dtype: int, layout: int, k_max: int,
                   first_block_column, stream=None) -> int:
    """Returns the plan handle (an integer address).  first_block_column: tensor (cpu or cuda) or raw pointer."""
    ptr = first_block_column if isinstance(first_block_column, int) else first_block_column.data_ptr()
    out = ctypes.c_void_p()
    st = lib().tt_plan_create(ctypes.byref(out), N_d, N_m, N_t, dtype, layout, k_max, ptr, _stream(stream))
    _check("tt_plan_create", st)
    return out.value


def tt_plan_create_coarse(N_d: int, N_m: int, N_t: int, out_every: int, dtype: int, layout: int, k_max: int,
                          first_block_column, stream=None) -> int:
    """tt_plan_create with the data side on every out_every-th time step (the p2q map, reading R19)."""
    ptr = first_block_column if isinstance(first_block_column, int) else first_block_column.data_ptr()
    out = ctypes.c_void_p()
    st = lib().tt_plan_create_coarse(ctypes.byref(out), N_d, N_m, N_t, out_every, dtype, layout, k_max, ptr,
                                     _stream(stream))
    _check("tt_plan_create_coarse", st)
    return out.value


def tt_plan_destroy(plan: int) -> None:
    lib().tt_plan_destroy(plan)


def tt_plan_device_bytes(plan: int) -> int:
    return lib().tt_plan_device_bytes(plan)


def tt_plan_last_cuda_error(plan: int) -> int:
    return lib().tt_plan_last_cuda_error(plan)


def tt_plan_get_spectrum(plan: int, dst: torch.Tensor, stream=None) -> None:
    _check("tt_plan_get_spectrum", lib().tt_plan_get_spectrum(plan, dst.data_ptr(), _stream(stream)), plan)


def tt_plan_describe(plan: int) -> str:
    buf = ctypes.create_string_buffer(1024)
    _check("tt_plan_describe", lib().tt_plan_describe(plan, buf, 1024), plan)
    return buf.value.decode()


def _ptr(x) -> int:
    return x if isinstance(x, int) else x.data_ptr()


def tt_matvec(plan: int, m, d, stream=None) -> None:
    _check("tt_matvec", lib().tt_matvec(plan, _ptr(m), _ptr(d), _stream(stream)), plan)


def tt_rmatvec(plan: int, d, m, stream=None) -> None:
    _check("tt_rmatvec", lib().tt_rmatvec(plan, _ptr(d), _ptr(m), _stream(stream)), plan)


def tt_normal(plan: int, m, out, stream=None) -> None:
    _check("tt_normal", lib().tt_normal(plan, _ptr(m), _ptr(out), _stream(stream)), plan)


def tt_matvec_batched(plan: int, k: int, M, D, stream=None) -> None:
    _check("tt_matvec_batched", lib().tt_matvec_batched(plan, k, _ptr(M), _ptr(D), _stream(stream)), plan)


def tt_rmatvec_batched(plan: int, k: int, D, M, stream=None) -> None:
    _check("tt_rmatvec_batched", lib().tt_rmatvec_batched(plan, k, _ptr(D), _ptr(M), _stream(stream)), plan)


def tt_normal_batched(plan: int, k: int, M, Out, stream=None) -> None:
    _check("tt_normal_batched", lib().tt_normal_batched(plan, k, _ptr(M), _ptr(Out), _stream(stream)), plan)


def tt_matvec_host(plan: int, m_host, d_host, stream=None) -> None:
    _check("tt_matvec_host", lib().tt_matvec_host(plan, _ptr(m_host), _ptr(d_host), _stream(stream)), plan)


def tt_rmatvec_host(plan: int, d_host, m_host, stream=None) -> None:
    _check("tt_rmatvec_host", lib().tt_rmatvec_host(plan, _ptr(d_host), _ptr(m_host), _stream(stream)), plan)


def tt_normal_host(plan: int, m_host, out_host, stream=None) -> None:
    _check("tt_normal_host", lib().tt_normal_host(plan, _ptr(m_host), _ptr(out_host), _stream(stream)), plan)


def tt_plan_set_profiling(plan: int, enabled: bool) -> None:
    _check("tt_plan_set_profiling", lib().tt_plan_set_profiling(plan, int(bool(enabled))), plan)


def tt_plan_stage_ms(plan: int, op: int) -> tuple[float, float, float, int]:
    """(fft_ms, stream_kernel_ms, ifft_ms, n_calls) averaged over the recorded calls of kind `op`."""
    buf = (ctypes.c_float * 4)()
    _check("tt_plan_stage_ms", lib().tt_plan_stage_ms(plan, op, buf, 4), plan)
    return float(buf[0]), float(buf[1]), float(buf[2]), int(buf[3])


def tt_probe_stream_read(src, nbytes: int, sink, stream=None) -> None:
    st = probe_lib().tt_probe_stream_read(_ptr(src), nbytes, _ptr(sink), _stream(stream))
    if st != 0:
        raise RuntimeError(f"tt_probe_stream_read failed: {st}")


class _CudaView:
    """Minimal __cuda_array_interface__ carrier so that torch can wrap plan-owned device memory."""

    def __init__(self, ptr, shape, typestr):
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": typestr, "data": (ptr, False),
                                         "version": 3, "strides": None}


def tt_debug_spectrum_view(plan: int, N_t: int, N_d: int, dtype) -> torch.Tensor:
    """Read-only torch view [N_t+1, N_d, row_pitch] (complex) of the plan's spectrum, no copy."""
    ptr, pitch = ctypes.c_void_p(), ctypes.c_int64()
    _check("tt_debug_spectrum_view", lib().tt_debug_spectrum_view(plan, ctypes.byref(ptr), ctypes.byref(pitch)), plan)
    ts = "<c8" if dtype == torch.float32 else "<c16"
    return torch.as_tensor(_CudaView(ptr.value, (N_t + 1, N_d, pitch.value), ts), device="cuda")


def tt_probe_dmma(iters: int, sink, stream=None) -> float:
    """Enqueues the DMMA probe; returns the flop count of the launch."""
    fl = ctypes.c_double()
    st = probe_lib().tt_probe_dmma(iters, _ptr(sink), ctypes.byref(fl), _stream(stream))
    if st != 0:
        raise RuntimeError(f"tt_probe_dmma failed: {st}")
    return fl.value


def tt_debug_fft_tables(N_t: int, max_radix: int = 25):
    """(radices, pos, tw) of the planner's FFT plan for an N_t-point series; runs without a GPU."""
    import numpy as np
    n = ctypes.c_int()
    radix = (ctypes.c_int * 16)()
    pos = (ctypes.c_ushort * max(1, N_t))()
    tw = (ctypes.c_double * (4 * max(1, N_t)))()
    st = lib().tt_debug_fft_tables(N_t, max_radix, ctypes.byref(n), radix, pos, tw)
    _check("tt_debug_fft_tables", st)
    return (list(radix[: n.value]), np.array(pos[:N_t], dtype=np.int64),
            np.array(tw[: 4 * N_t]).reshape(2 * N_t, 2) @ np.array([1.0, 1.0j]))


def tt_debug_trig(k: int, n: int) -> tuple[float, float]:
    c, s = ctypes.c_double(), ctypes.c_double()
    _check("tt_debug_trig", lib().tt_debug_trig(k, n, ctypes.byref(c), ctypes.byref(s)))
    return c.value, s.value


def tt_debug_set(key: str, value: int) -> None:
    _check("tt_debug_set", lib().tt_debug_set(key.encode(), value))


def tt_chol_create(n: int, L, ld: int | None = None, stream=None) -> int:
    """Handle of the prepared factor.  L: [n, n] float64 tensor (cpu or cuda, row-major) or raw pointer."""
    out = ctypes.c_void_p()
    st = lib().tt_chol_create(ctypes.byref(out), n, _ptr(L), n if ld is None else ld, _stream(stream))
    _check("tt_chol_create", st)
    return out.value


def tt_chol_destroy(chol: int) -> None:
    lib().tt_chol_destroy(chol)


def tt_chol_device_bytes(chol: int) -> int:
    return lib().tt_chol_device_bytes(chol)


def tt_chol_last_cuda_error(chol: int) -> int:
    return lib().tt_chol_last_cuda_error(chol)


def _check_chol(call: str, status: int, chol: int):
    if status != TT_OK:
        raise TTError(call, status, lib().tt_chol_last_cuda_error(chol))


def tt_chol_solve(chol: int, b, x, stream=None) -> None:
    _check_chol("tt_chol_solve", lib().tt_chol_solve(chol, _ptr(b), _ptr(x), _stream(stream)), chol)


def tt_chol_trsv(chol: int, transposed: bool, b, x, stream=None) -> None:
    _check_chol("tt_chol_trsv", lib().tt_chol_trsv(chol, int(bool(transposed)), _ptr(b), _ptr(x), _stream(stream)), chol)


def tt_assemble_K(F: int, G: int, noise_var, col0: int, ncols: int, K, ldk: int, stream=None) -> None:
    _check("tt_assemble_K", lib().tt_assemble_K(F, G, _ptr(noise_var), col0, ncols, _ptr(K), ldk, _stream(stream)), F)


def tt_assemble_K_direct(Fcol, Gcol, noise_var, N_d: int, N_m: int, N_t: int, dtype: int, K, ldk: int, stream=None) -> None:
    """noise_var None: K = F G* alone (a rank's partial of the sharded assembly, see tt_K_add_noise)."""
    nv = None if noise_var is None else _ptr(noise_var)
    _check("tt_assemble_K_direct", lib().tt_assemble_K_direct(_ptr(Fcol), _ptr(Gcol), nv, N_d, N_m, N_t, dtype,
                                                                _ptr(K), ldk, _stream(stream)))


def tt_K_add_noise(noise_var, n: int, dtype: int, K, ldk: int, stream=None) -> None:
    _check("tt_K_add_noise", lib().tt_K_add_noise(_ptr(noise_var), n, dtype, _ptr(K), ldk, _stream(stream)))


def tt_qoi_direct(Fqcol, Gqcol, Gcol, N_q: int, N_d: int, N_m: int, N_t: int, out_every: int, dtype: int, chol: int,
                  Q, ldq: int, post_cov_q, ldc: int, stream=None) -> None:
    _check_chol("tt_qoi_direct", lib().tt_qoi_direct(_ptr(Fqcol), _ptr(Gqcol), _ptr(Gcol), N_q, N_d, N_m, N_t, out_every, dtype,
                                                      chol, _ptr(Q), ldq, _ptr(post_cov_q), ldc, _stream(stream)), chol)


def tt_map_create(F: int | None, G: int, chol: int, noise_var, stream=None) -> int:
    out = ctypes.c_void_p()
    _check("tt_map_create", lib().tt_map_create(ctypes.byref(out), F, G, chol, _ptr(noise_var), _stream(stream)))
    return out.value


def tt_map_destroy(m: int) -> None:
    lib().tt_map_destroy(m)


def tt_map_infer(m: int, form: int, d_obs, m_map, stream=None) -> None:
    _check("tt_map_infer", lib().tt_map_infer(m, form, _ptr(d_obs), _ptr(m_map), _stream(stream)))


def tt_smw_apply(m: int, u, out, stream=None) -> None:
    _check("tt_smw_apply", lib().tt_smw_apply(m, _ptr(u), _ptr(out), _stream(stream)))


def tt_postcov_q_apply(m: int, Fq: int, Gq: int, v, work, out, stream=None) -> None:
    _check("tt_postcov_q_apply", lib().tt_postcov_q_apply(m, Fq, Gq, _ptr(v), _ptr(work), _ptr(out), _stream(stream)))


def tt_d2q_apply(m: int, Fq: int, form: int, d_obs, work, q, stream=None) -> None:
    _check("tt_d2q_apply", lib().tt_d2q_apply(m, Fq, form, _ptr(d_obs), _ptr(work), _ptr(q), _stream(stream)))


def tt_map_infer_partial(m: int, d_obs, a_scratch, b, stream=None) -> None:
    _check("tt_map_infer_partial", lib().tt_map_infer_partial(m, _ptr(d_obs), _ptr(a_scratch), _ptr(b), _stream(stream)))


def tt_map_infer_finish(m: int, b, m_map, stream=None) -> None:
    _check("tt_map_infer_finish", lib().tt_map_infer_finish(m, _ptr(b), _ptr(m_map), _stream(stream)))


def tt_map_infer_host(m: int, form: int, d_obs_host, m_map_host, stream=None) -> None:
    _check("tt_map_infer_host", lib().tt_map_infer_host(m, form, _ptr(d_obs_host), _ptr(m_map_host), _stream(stream)))


_DT = {torch.float32: TT_F32, torch.float64: TT_F64}


def _sync_quietly() -> None:
    """Device synchronisation before a handle is destroyed; tolerant of interpreter shutdown (module globals gone)."""
    try:
        torch.cuda.synchronize()
    except Exception:
        pass


class Plan:
    """RAII convenience over the calls above (tests and bench.py use it).

    Vectors are torch CUDA tensors in the plan's dtype and layout (time-major [N_t, N_m] /
    [N_t, N_d], or [N_t, N_*, k] for the k-RHS calls); outputs are allocated with torch.
    """

    def __init__(self, first_block_column: torch.Tensor, layout: int = TT_TIME_MAJOR, k_max: int = 1,
                 stream=None, out_every: int = 1):
        assert first_block_column.dim() == 3 and first_block_column.is_contiguous()
        self.N_t, self.N_d, self.N_m = first_block_column.shape
        self.dtype = first_block_column.dtype
        self.layout, self.k_max, self.out_every = layout, k_max, out_every
        self.handle = tt_plan_create_coarse(self.N_d, self.N_m, self.N_t, out_every, _DT[self.dtype], layout, k_max,
                                            first_block_column, stream)

    def close(self):
        if getattr(self, "handle", None):
            _sync_quietly()
            tt_plan_destroy(self.handle)
            self.handle = None

    __del__ = close

    def _shape(self, n_space: int, k: int | None, data: bool = False):
        n_time = self.N_t // self.out_every if data else self.N_t
        base = (n_time, n_space) if self.layout == TT_TIME_MAJOR else (n_space, n_time)
        if k is None:
            return base
        return base + (k,) if self.layout == TT_TIME_MAJOR else (k,) + base

    def _out(self, n_space: int, k: int | None = None, data: bool = False, stream=None):
        """Output allocated on the stream the kernels will run on (the caching allocator must not hand the block to
        another stream's tensor before they finish)."""
        if isinstance(stream, torch.cuda.Stream):
            with torch.cuda.stream(stream):
                return torch.empty(self._shape(n_space, k, data), dtype=self.dtype, device="cuda")
        return torch.empty(self._shape(n_space, k, data), dtype=self.dtype, device="cuda")

    def _vec(self, t: torch.Tensor, n_space: int, k: int | None = None, data: bool = False, what: str = "vector"):
        """The raw-pointer calls trust their arguments; the convenience class does not."""
        n = 1
        for x in self._shape(n_space, k, data):
            n *= x
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == self.dtype and t.is_contiguous() and t.numel() == n):
            raise ValueError(f"{what}: expected a contiguous CUDA tensor of {n} x {self.dtype}, got "
                             f"{tuple(t.shape)} {t.dtype} on {t.device}{'' if t.is_contiguous() else ' (not contiguous)'}")
        return t

    def matvec(self, m, out=None, stream=None):
        self._vec(m, self.N_m, what="m")
        out = self._out(self.N_d, data=True, stream=stream) if out is None else self._vec(out, self.N_d, data=True, what="out")
        tt_matvec(self.handle, m, out, stream)
        return out

    def rmatvec(self, d, out=None, stream=None):
        self._vec(d, self.N_d, data=True, what="d")
        out = self._out(self.N_m, stream=stream) if out is None else self._vec(out, self.N_m, what="out")
        tt_rmatvec(self.handle, d, out, stream)
        return out

    def normal(self, m, out=None, stream=None):
        self._vec(m, self.N_m, what="m")
        out = self._out(self.N_m, stream=stream) if out is None else self._vec(out, self.N_m, what="out")
        tt_normal(self.handle, m, out, stream)
        return out

    def matvec_batched(self, M, out=None, stream=None):
        k = M.shape[-1] if self.layout == TT_TIME_MAJOR else M.shape[0]
        self._vec(M, self.N_m, k, what="M")
        out = self._out(self.N_d, k, data=True, stream=stream) if out is None else self._vec(out, self.N_d, k, data=True, what="out")
        tt_matvec_batched(self.handle, k, M, out, stream)
        return out

    def rmatvec_batched(self, D, out=None, stream=None):
        k = D.shape[-1] if self.layout == TT_TIME_MAJOR else D.shape[0]
        self._vec(D, self.N_d, k, data=True, what="D")
        out = self._out(self.N_m, k, stream=stream) if out is None else self._vec(out, self.N_m, k, what="out")
        tt_rmatvec_batched(self.handle, k, D, out, stream)
        return out

    def spectrum(self):
        cdt = torch.complex64 if self.dtype == torch.float32 else torch.complex128
        out = torch.empty((self.N_t + 1, self.N_d, self.N_m), dtype=cdt, device="cuda")
        tt_plan_get_spectrum(self.handle, out)
        return out

    @property
    def device_bytes(self) -> int:
        return tt_plan_device_bytes(self.handle)


class Chol:
    """RAII convenience over tt_chol_*: the two triangular solves with the Cholesky factor of K."""

    def __init__(self, L: torch.Tensor, stream=None):
        assert L.dim() == 2 and L.shape[0] == L.shape[1] and L.dtype == torch.float64 and L.stride(1) == 1
        self.n = L.shape[0]
        self.handle = tt_chol_create(self.n, L, L.stride(0), stream)

    def close(self):
        if getattr(self, "handle", None):
            _sync_quietly()
            tt_chol_destroy(self.handle)
            self.handle = None

    __del__ = close

    def _vec(self, t, what):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == self.n):
            raise ValueError(f"{what}: expected a contiguous CUDA tensor of {self.n} x float64, got {tuple(t.shape)} {t.dtype} on {t.device}")
        return t

    def _out(self, stream):
        if isinstance(stream, torch.cuda.Stream):
            with torch.cuda.stream(stream):
                return torch.empty(self.n, dtype=torch.float64, device="cuda")
        return torch.empty(self.n, dtype=torch.float64, device="cuda")

    def solve(self, b, out=None, stream=None):
        self._vec(b, "b")
        out = self._out(stream) if out is None else self._vec(out, "out")
        tt_chol_solve(self.handle, b, out, stream)
        return out

    def trsv(self, b, transposed=False, out=None, stream=None):
        self._vec(b, "b")
        out = self._out(stream) if out is None else self._vec(out, "out")
        tt_chol_trsv(self.handle, transposed, b, out, stream)
        return out

    @property
    def device_bytes(self) -> int:
        return tt_chol_device_bytes(self.handle)


def assemble_K(F: Plan, G: Plan, noise_var: torch.Tensor, cols: tuple[int, int] | None = None,
               out: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """K = Gamma_noise + F G* as an [n, n] float64 CUDA tensor (columns `cols` = (col0, ncols) only, if given)."""
    n = F.N_d * F.N_t
    K = torch.zeros((n, n), dtype=torch.float64, device="cuda") if out is None else out
    col0, ncols = cols if cols is not None else (0, n)
    tt_assemble_K(F.handle, G.handle, noise_var, col0, ncols, K, K.stride(0), stream)
    return K


def tt_assemble_K_direct_static(Fcol, Gcol, noise_var, N_d: int, N_m: int, N_t: int, dtype: int, K, ldk: int, stream=None) -> None:
    """tt_assemble_K_direct without any allocation (TT_F32; scratch in a 64 MiB static device array; TT_ERR_STATIC_LIMIT = -13
    when the problem does not fit)."""
    nv = None if noise_var is None else _ptr(noise_var)
    _check("tt_assemble_K_direct_static", lib().tt_assemble_K_direct_static(_ptr(Fcol), _ptr(Gcol), nv, N_d, N_m, N_t, dtype,
                                                                              _ptr(K), ldk, _stream(stream)))


def assemble_K_direct(Fcol: torch.Tensor, Gcol: torch.Tensor, noise_var: torch.Tensor | None, out: torch.Tensor | None = None,
                      stream=None) -> torch.Tensor:
    """K = Gamma_noise + F G* from the [N_t, N_d, N_m] block columns F_k and G_k = F_k Gamma_prior (no plans, no matvecs)."""
    N_t, N_d, N_m = Fcol.shape
    assert Gcol.shape == Fcol.shape and Gcol.dtype == Fcol.dtype and Fcol.is_contiguous() and Gcol.is_contiguous()
    n = N_t * N_d
    K = torch.empty((n, n), dtype=torch.float64, device="cuda") if out is None else out
    tt_assemble_K_direct(Fcol, Gcol, noise_var, N_d, N_m, N_t, TT_F32 if Fcol.dtype == torch.float32 else TT_F64,
                         K, K.stride(0), stream)
    return K


def qoi_direct(Fqcol: torch.Tensor, Gqcol: torch.Tensor, Gcol: torch.Tensor, out_every: int, chol: "Chol", stream=None):
    """(Q, Gamma_post(q)) as dense float64 CUDA tensors [n_q, n] and [n_q, n_q] from the block columns (tt_qoi_direct)."""
    N_t, N_q, N_m = Fqcol.shape
    N_d = Gcol.shape[1]
    assert Gqcol.shape == Fqcol.shape and Gcol.shape == (N_t, N_d, N_m) and Fqcol.dtype == Gqcol.dtype == Gcol.dtype
    assert Fqcol.is_contiguous() and Gqcol.is_contiguous() and Gcol.is_contiguous()
    nq, n = (N_t // out_every) * N_q, N_t * N_d
    Q = torch.empty((nq, n), dtype=torch.float64, device="cuda")
    C = torch.empty((nq, nq), dtype=torch.float64, device="cuda")
    tt_qoi_direct(Fqcol, Gqcol, Gcol, N_q, N_d, N_m, N_t, out_every, TT_F32 if Fqcol.dtype == torch.float32 else TT_F64,
                  chol.handle, Q, n, C, nq, stream)
    return Q, C


class MapInference:
    """RAII convenience over tt_map_*: the online MAP point of eq (4.13)."""

    def __init__(self, F: Plan | None, G: Plan, chol: Chol, noise_var: torch.Tensor, stream=None):
        self.F, self.G, self.chol = F, G, chol          # keep the borrowed objects alive
        self.handle = tt_map_create(F.handle if F is not None else None, G.handle, chol.handle, noise_var, stream)

    def close(self):
        if getattr(self, "handle", None):
            _sync_quietly()
            tt_map_destroy(self.handle)
            self.handle = None

    __del__ = close

    def infer(self, d_obs, form: int = TT_MAP_PAPER, out=None, stream=None):
        self.G._vec(d_obs, self.G.N_d, data=True, what="d_obs")
        out = self.G._out(self.G.N_m, stream=stream) if out is None else self.G._vec(out, self.G.N_m, what="out")
        tt_map_infer(self.handle, form, d_obs, out, stream)
        return out

    def smw_apply(self, u, out=None, stream=None):
        """(I - G* K^-1 F) u: Gamma_post(m) v for u = Gamma_prior v (eq 4.7), m_map^prior for u = m_prior (eq 4.8)."""
        out = torch.empty_like(u) if out is None else out
        tt_smw_apply(self.handle, u, out, stream)
        return out

    def infer_partial(self, d_obs, stream=None):
        """First half of eq (4.13): returns (a_scratch, b); b is this rank's partial F G* y."""
        a, b = self.G._out(self.G.N_m), self.G._out(self.G.N_d, data=True)
        tt_map_infer_partial(self.handle, d_obs, a, b, stream)
        return a, b

    def infer_finish(self, b, out, stream=None):
        tt_map_infer_finish(self.handle, b, out, stream)
        return out
