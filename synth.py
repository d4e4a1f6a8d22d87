"""Seeded synthetic inputs for the block-Toeplitz p2o matvec (harness code).

This module holds NONE of the method's arithmetic: it only draws the block
column F_k (k = 0..N_t-1, each N_d x N_m), the parameter vector m and the data
vector d of the five workloads named in BASELINE.json, with the recipe frozen
in DESIGN.md ("Input recipe").  Both the CPU oracle's tests and the CUDA
path's tests/bench take their inputs from here (a module of its own at the repo root, outside the product
package), so the two sides always see
the same bytes.

Every element is a pure function of (seed, tensor_id, linear_index): a
splitmix64-style hash gives two 32-bit uniforms, Box-Muller (fp64) gives a
standard normal, the deterministic envelope is applied in fp64 and the result
is rounded once to the config dtype.  Being counter-based, any slice can be
drawn on its own (one sensor row of a 40 GB block column, say) and on any
device; full-size tensors are drawn directly on the GPU in bounded chunks.

The paper's own F comes from 49 adjoint PDE solves and is
not available; these stand-ins keep its shape regime N_d << N_m, N_t >> 1
(eq 4.3) and sizes (~1e8 parameters, ~100 sensors,
PAPER.md:234, 381).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace

import torch

TENSOR_F, TENSOR_M, TENSOR_D, TENSOR_SCALE, TENSOR_CENTRE, TENSOR_L = 0, 1, 2, 3, 4, 5

_MASK64 = (1 << 64) - 1


def _i64(x: int) -> int:
    """Two's-complement int64 view of an unsigned 64-bit constant."""
    x &= _MASK64
    return x - (1 << 64) if x >= (1 << 63) else x


_GOLDEN = _i64(0x9E3779B97F4A7C15)
_MIX1 = _i64(0xBF58476D1CE4E5B9)
_MIX2 = _i64(0x94D049BB133111EB)


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    """Logical shift right on int64 (torch's >> is arithmetic)."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def hash64(seed: int, tensor_id: int, index: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser of (index, tensor_id, seed); int64 in, int64 out (wrapping)."""
    key = _i64((tensor_id + 1) * 0x9E3779B97F4A7C15 + (seed + 1) * 0xD1B54A32D192ED03)
    x = index * _GOLDEN + key
    x = (x ^ _lsr(x, 30)) * _MIX1
    x = (x ^ _lsr(x, 27)) * _MIX2
    return x ^ _lsr(x, 31)


def uniform01(seed: int, tensor_id: int, index: torch.Tensor) -> torch.Tensor:
    """One uniform in (0,1) per index, fp64, from the high 32 bits."""
    h = hash64(seed, tensor_id, index)
    return (_lsr(h, 32).to(torch.float64) + 0.5) * (1.0 / 4294967296.0)


def normal01(seed: int, tensor_id: int, index: torch.Tensor) -> torch.Tensor:
    """One N(0,1) per index (Box-Muller on the two 32-bit halves), fp64."""
    h = hash64(seed, tensor_id, index)
    u1 = (_lsr(h, 32).to(torch.float64) + 0.5) * (1.0 / 4294967296.0)
    u2 = ((h & 0xFFFFFFFF).to(torch.float64) + 0.5) * (1.0 / 4294967296.0)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config.  dtype is the dtype of the stored inputs."""
    name: str
    N_d: int
    N_m: int
    N_t: int
    dtype: torch.dtype
    seed: int
    tau: float               # F_k decays like exp(-k/tau)
    sensor_scale: bool = False   # per-sensor factor c_s ~ U[0.5, 2]
    bump: bool = False           # per-sensor Gaussian bump in p, sigma = 5% of N_m
    k_rhs: int = 1

    @property
    def n_params(self) -> int:
        return self.N_m * self.N_t

    def scaled(self, **kw) -> "Workload":
        """Same recipe at other sizes (parity tests on shrunken copies)."""
        return replace(self, **kw)


CONFIGS = {
    # BASELINE.json configs[0..4]
    "C1": Workload("C1-tiny-fp64", 4, 64, 32, torch.float64, 0, 8.0),
    "C2": Workload("C2-medium-fp64", 64, 16384, 256, torch.float64, 1, 32.0, sensor_scale=True),
    "C3": Workload("C3-paper-scale-c64", 100, 250000, 400, torch.float32, 2, 100.0, bump=True),
    "C4": Workload("C4-krhs-fp64", 64, 65536, 512, torch.float64, 3, 64.0, k_rhs=32),
    "C5": Workload("C5-normal-c64", 200, 100000, 400, torch.float32, 4, 100.0),
    # the paper's own test configuration: 7x7 sensors, 513x513 parameters, 500 steps,
    # 131 584 500 parameters, 24 500 data - the workload of the online phase (eq 4.13)
    "P5": Workload("P5-paper-sec5-online-c64", 49, 263169, 500, torch.float32, 5, 100.0, sensor_scale=True),
    # the paper's p2q map: 4x4 QoI locations, the same parameter grid and fine time grid,
    # QoIs sampled at 1 Hz (every 10th step): 800 QoIs; 17 GB block column in fp64, 8.4 GB here in fp32
    "Q5": Workload("Q5-paper-sec5-p2q-c64", 16, 263169, 500, torch.float32, 6, 100.0, sensor_scale=True),
}

NOISE_LEVEL = 0.05   # relative noise of the online workload (the paper uses 2-6 %)


def _sensor_scale(w: Workload, s: torch.Tensor) -> torch.Tensor:
    return 0.5 + 1.5 * uniform01(w.seed, TENSOR_SCALE, s)


def _sensor_centre(w: Workload, s: torch.Tensor) -> torch.Tensor:
    mu = torch.floor(uniform01(w.seed, TENSOR_CENTRE, s) * w.N_m)
    return torch.clamp(mu, max=w.N_m - 1)


def block_column(w: Workload, device="cpu", k_range=None, s_range=None, p_range=None,
                 out: torch.Tensor | None = None, chunk_elems: int = 1 << 25) -> torch.Tensor:
    """First block column F_k[s,p], layout [k][s][p] (p fastest), dtype w.dtype.

    Ranges select a sub-box; each element depends only on its global (k,s,p),
    so a slice equals the same slice of the full tensor bit for bit (on one
    device type).  Drawn in chunks of whole k-planes to bound scratch memory.
    """
    k0, k1 = k_range or (0, w.N_t)
    s0, s1 = s_range or (0, w.N_d)
    p0, p1 = p_range or (0, w.N_m)
    nk, ns, np_ = k1 - k0, s1 - s0, p1 - p0
    if out is None:
        out = torch.empty((nk, ns, np_), dtype=w.dtype, device=device)
    assert out.shape == (nk, ns, np_)
    dev = out.device
    s_idx = torch.arange(s0, s1, device=dev, dtype=torch.int64)
    p_idx = torch.arange(p0, p1, device=dev, dtype=torch.int64)
    env_sp = torch.ones((ns, 1), dtype=torch.float64, device=dev)
    if w.sensor_scale:
        env_sp = env_sp * _sensor_scale(w, s_idx)[:, None]
    # rows of s processed per chunk so that scratch stays ~chunk_elems fp64
    rows = max(1, min(ns, chunk_elems // max(1, np_)))
    sigma = 0.05 * w.N_m
    for k in range(k0, k1):
        decay = math.exp(-k / w.tau)
        for r0 in range(0, ns, rows):
            r1 = min(ns, r0 + rows)
            lin = ((k * w.N_d + s_idx[r0:r1, None]) * w.N_m + p_idx[None, :])
            z = normal01(w.seed, TENSOR_F, lin)
            z = z * (decay * env_sp[r0:r1])
            if w.bump:
                mu = _sensor_centre(w, s_idx[r0:r1])[:, None]
                z = z * torch.exp(-((p_idx[None, :].to(torch.float64) - mu) ** 2) / (2.0 * sigma * sigma))
            out[k - k0, r0:r1] = z.to(w.dtype)
    return out


def _vector(w: Workload, tensor_id: int, n_time: int, n_space: int, device, k_rhs: int,
            chunk_elems: int = 1 << 25) -> torch.Tensor:
    shape = (n_time, n_space) if k_rhs == 1 else (n_time, n_space, k_rhs)
    total = n_time * n_space * k_rhs
    out = torch.empty(total, dtype=w.dtype, device=device)
    for a in range(0, total, chunk_elems):
        b = min(total, a + chunk_elems)
        idx = torch.arange(a, b, device=out.device, dtype=torch.int64)
        out[a:b] = normal01(w.seed, tensor_id, idx).to(w.dtype)
    return out.view(shape)


def vector_m(w: Workload, device="cpu", k_rhs: int | None = None) -> torch.Tensor:
    """Parameter vector, time-major [j][p] (paper's stacking), or [j][p][r] for k RHS."""
    return _vector(w, TENSOR_M, w.N_t, w.N_m, device, w.k_rhs if k_rhs is None else k_rhs)


def vector_d(w: Workload, device="cpu", k_rhs: int | None = None) -> torch.Tensor:
    """Data vector, time-major [i][s], or [i][s][r] for k RHS."""
    return _vector(w, TENSOR_D, w.N_t, w.N_d, device, w.k_rhs if k_rhs is None else k_rhs)


# ---------------------------------------------------------------------------------------------
# Inputs of the online phase (eq 4.13): stand-ins for what Phases 1-2 of the paper would deliver.
# ---------------------------------------------------------------------------------------------
def prior_gamma(w: Workload, device="cpu") -> torch.Tensor:
    """Diagonal of a time-invariant spatial prior covariance Gamma_s (fp64, [N_m]), smooth and positive:
    gamma_p = 0.5 + exp(-((p - N_m/2) / (N_m/4))^2).  Stands in for the paper's elliptic-operator prior
    (eq 5.1), which needs a sparse solver; only 'time-invariant, block diagonal in time' matters here
    (PAPER.md:368), because that is what makes G* block Toeplitz."""
    p = torch.arange(w.N_m, device=device, dtype=torch.float64)
    return 0.5 + torch.exp(-((p - 0.5 * w.N_m) / (0.25 * w.N_m)) ** 2)


def scaled_block_column(w: Workload, F: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
    """The SECOND input block column of the online phase at sizes where it has to be drawn on the device: column p of
    every block of F scaled by the prior weight prior_gamma(w)[p], in fp64, rounded once to w.dtype.  In the paper this
    array is the output of N_d prior solves (Phase 2) and an INPUT of the online phase; the formula
    G_k = F_k Gamma_s belongs to oracle/online_plain.gstar_block_column, which the small parity tests use directly and
    which tests/test_synth.py holds this generator to, bit for bit.  Works plane by plane to bound scratch memory."""
    g = prior_gamma(w, F.device)
    out = torch.empty_like(F) if out is None else out
    for k in range(F.shape[0]):
        out[k] = (F[k].to(torch.float64) * g[None, : F.shape[2]]).to(w.dtype)
    return out


def noise_var(w: Workload, device="cpu") -> torch.Tensor:
    """Diagonal of Gamma_noise, [N_t, N_d] in w.dtype: per sensor, constant in time (the paper adds noise
    per sensor relative to that sensor's signal):  (NOISE_LEVEL)^2 * v_s  with
    v_s = c_s^2 N_m tau / 2, the scale of Var(d_i[s]) for m ~ N(0, I) under the F recipe."""
    s = torch.arange(w.N_d, device=device, dtype=torch.int64)
    c = _sensor_scale(w, s) if w.sensor_scale else torch.ones(w.N_d, dtype=torch.float64, device=device)
    v = (NOISE_LEVEL ** 2) * c * c * (w.N_m * w.tau * 0.5)
    return v[None, :].expand(w.N_t, w.N_d).contiguous().to(w.dtype)


def factor_standin(n: int, seed: int, device="cpu", rows_per_chunk: int = 1024) -> torch.Tensor:
    """A lower-triangular [n, n] fp64 matrix with the profile of a Cholesky factor (diagonal in (1, 2), strictly
    lower entries N(0, 1/n), zeros above): stands in for the factor of K = Gamma_noise + F G* where assembling
    the true K (N_d N_t matvec pairs) is not affordable - the cost of the triangular solves does
    not depend on the values.  Counter-based like everything else here: entry (r, c) depends on (seed, r*n + c)."""
    L = torch.zeros((n, n), dtype=torch.float64, device=device)
    col = torch.arange(n, device=L.device, dtype=torch.int64)
    for r0 in range(0, n, rows_per_chunk):
        r1 = min(n, r0 + rows_per_chunk)
        row = torch.arange(r0, r1, device=L.device, dtype=torch.int64)
        lin = row[:, None] * n + col[None, :]
        blk = normal01(seed, TENSOR_L, lin) * (1.0 / math.sqrt(n))
        blk = torch.where(col[None, :] < row[:, None], blk, torch.zeros_like(blk))
        L[r0:r1] = blk
        L[row, row] = 1.0 + uniform01(seed, TENSOR_L, row * n + row)
    return L
