"""CPU ORACLE (test infrastructure, NOT the product path) - plain definition.

The p2o map F of a discrete LTI system is block lower-triangular Toeplitz
(eq 2.4-2.6): with zero-based time steps,

    d_i = sum_{j=0..i} F_{i-j} m_j ,      F_k := B A^k C  (N_d x N_m),
                                          i = 0..N_t-1               (eq 2.5)

(the paper's d_{i+1} is our d_i: output step i sees m_0..m_i, F_0 = B A^0 C on
the block diagonal; reading R1), and its transpose,
the discretise-then-optimise adjoint ("realized by simply
transposing these maps"; reading R2), is

    m'_j = sum_{i=j..N_t-1} F_{i-j}^T d_i ,   j = 0..N_t-1.

The FFT method of PAPER.md:265 reaches exactly these sums ("exact up to
rounding error"), so the oracle is the definition written
out as a direct time-domain block convolution, O(N_t^2 N_d N_m), with no FFT
anywhere.  All arithmetic is fp64: inputs of any dtype are converted exactly
to fp64 first; the inner sum over space (one N_d x N_m block times a vector,
numpy matmul as the library step) is formed first and then added, j (or i)
ascending, into the per-output accumulator.

Array layout (paper's stacking): everything time-major,
    F : [N_t, N_d, N_m]      block column, F[k] = F_k
    m : [N_t, N_m]  or [N_t, N_m, k]   (k right-hand sides, column-independent)
    d : [N_t, N_d]  or [N_t, N_d, k]

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference leg may import this module.  It shares no code with the CUDA path.
Pins: tests/test_oracle_pins.py (dense brute force, the paper's recurrence
eq 2.2-2.3, impulse, causality, shift, linearity, adjoint identity, closed
forms, exact-integer case).  No function here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a), dtype=np.float64)


def matvec(F, m) -> np.ndarray:
    """d = F m, eq (2.5).  Returns fp64 [N_t, N_d(, k)]."""
    F, m = _f64(F), _f64(m)
    N_t, N_d, N_m = F.shape
    assert m.shape[0] == N_t and m.shape[1] == N_m
    d = np.zeros((N_t, N_d) + m.shape[2:], dtype=np.float64)
    for i in range(N_t):
        acc = np.zeros((N_d,) + m.shape[2:], dtype=np.float64)
        for j in range(i + 1):
            acc += F[i - j] @ m[j]          # block F_{i-j} (N_d x N_m) times m_j
        d[i] = acc
    return d


def rmatvec(F, d) -> np.ndarray:
    """m' = F^T d: transpose of eq (2.5).  Returns fp64 [N_t, N_m(, k)]."""
    F, d = _f64(F), _f64(d)
    N_t, N_d, N_m = F.shape
    assert d.shape[0] == N_t and d.shape[1] == N_d
    out = np.zeros((N_t, N_m) + d.shape[2:], dtype=np.float64)
    for j in range(N_t):
        acc = np.zeros((N_m,) + d.shape[2:], dtype=np.float64)
        for i in range(j, N_t):
            acc += F[i - j].T @ d[i]        # block F_{i-j}^T (N_m x N_d) times d_i
        out[j] = acc
    return out


def normal(F, m) -> np.ndarray:
    """F^T (F m): the data-misfit Hessian of eq (2.12) with Gamma_noise = I."""
    return rmatvec(F, matvec(F, m))


def matvec_entry(F, m, i: int, s: int) -> float:
    """One output d_i[s] of eq (2.5), for sampled parity at sizes where matvec() is too slow.

    F is the full [N_t, N_d, N_m] block column or a sensor slice [N_t, 1, N_m] with s=0.
    """
    acc = 0.0
    for j in range(i + 1):
        acc += float(np.dot(np.asarray(F[i - j][s], dtype=np.float64),
                            np.asarray(m[j], dtype=np.float64)))
    return acc


def rmatvec_entry(F, d, j: int, p: int) -> float:
    """One output m'_j[p] of the transpose of eq (2.5).  F may be a [N_t, N_d, 1] slice with p=0."""
    N_t = F.shape[0]
    acc = 0.0
    for i in range(j, N_t):
        acc += float(np.dot(np.asarray(F[i - j][:, p], dtype=np.float64),
                            np.asarray(d[i], dtype=np.float64)))
    return acc


# ---------------------------------------------------------------------------------------------
# Output on a coarser time grid: the p2q map of the paper's example (N_t^q = 50 << N_t = 500,
# PAPER.md:162, 381).  The paper says only that "the block structure ... changes correspondingly";
# DESIGN.md reading R19: the QoI is the fine-grid output sampled at the end of every r-th step,
#     q_I = (F_q m)_{r(I+1)-1} = sum_{j=0..r(I+1)-1} F_{r(I+1)-1-j} m_j ,   I = 0..N_t/r - 1,
# (the paper's 1-based q_I at time I*r*dt), the stored block column staying the fine-grid one
# (N_t blocks of N_q x N_m: the 16 x 1.05 GB = 17 GB of PAPER.md:393).  Its transpose is
#     m'_j = sum_{I : r(I+1)-1 >= j} F_{r(I+1)-1-j}^T q_I .
# ---------------------------------------------------------------------------------------------
def matvec_decimated(F, m, r: int) -> np.ndarray:
    """q = S F m with S = 'keep fine steps r-1, 2r-1, ...'.  Returns fp64 [N_t // r, N_q(, k)]."""
    F, m = _f64(F), _f64(m)
    N_t, N_q, N_m = F.shape
    assert N_t % r == 0 and m.shape[0] == N_t and m.shape[1] == N_m
    q = np.zeros((N_t // r, N_q) + m.shape[2:], dtype=np.float64)
    for I in range(N_t // r):
        i = r * (I + 1) - 1
        acc = np.zeros((N_q,) + m.shape[2:], dtype=np.float64)
        for j in range(i + 1):
            acc += F[i - j] @ m[j]
        q[I] = acc
    return q


def rmatvec_decimated(F, q, r: int) -> np.ndarray:
    """m' = F^T S^T q.  q: [N_t // r, N_q(, k)].  Returns fp64 [N_t, N_m(, k)]."""
    F, q = _f64(F), _f64(q)
    N_t, N_q, N_m = F.shape
    assert N_t % r == 0 and q.shape[0] == N_t // r and q.shape[1] == N_q
    out = np.zeros((N_t, N_m) + q.shape[2:], dtype=np.float64)
    for j in range(N_t):
        acc = np.zeros((N_m,) + q.shape[2:], dtype=np.float64)
        for I in range(N_t // r):
            i = r * (I + 1) - 1
            if i >= j:
                acc += F[i - j].T @ q[I]
        out[j] = acc
    return out
