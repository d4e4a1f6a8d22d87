"""Pins for the CPU oracle (CPU only): the oracle is checked against what the
paper and the mathematics fix, never against itself.

Each test names the passage it pins.  A plausible mistake anywhere in the
oracle (dropped term, wrong sign/index, transposed block, off-by-one delay,
wrong half kept in the adjoint) fails at least one of them.
"""
import itertools
from fractions import Fraction

import numpy as np
import pytest

from oracle import toeplitz_blocked as ob
from oracle import toeplitz_plain as op

RNG = np.random.default_rng(20250114)

SHAPES = [(3, 5, 7), (1, 4, 6), (4, 1, 5), (2, 3, 1), (1, 1, 1), (4, 64, 32)]  # (N_d, N_m, N_t)


def dense_from_block_column(F):
    """Explicit (N_d N_t) x (N_m N_t) matrix of eq (2.5): block (i,j) = F_{i-j} for i >= j else 0."""
    N_t, N_d, N_m = F.shape
    A = np.zeros((N_t * N_d, N_t * N_m))
    for i in range(N_t):
        for j in range(N_t):
            if i >= j:
                for s in range(N_d):
                    for p in range(N_m):
                        A[i * N_d + s, j * N_m + p] = F[i - j, s, p]
    return A


def naive_matmul(A, x):
    y = [0.0] * A.shape[0]
    for r in range(A.shape[0]):
        acc = 0.0
        for c in range(A.shape[1]):
            acc += A[r, c] * x[c]
        y[r] = acc
    return np.array(y)


def rel(a, b):
    nb = np.linalg.norm(np.ravel(b))
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / (nb if nb > 0 else 1.0)


@pytest.fixture(params=[op, ob], ids=["plain", "blocked"])
def orc(request):
    return request.param


# ---------------------------------------------------------------- brute force (eq 2.5)
@pytest.mark.parametrize("N_d,N_m,N_t", SHAPES)
def test_dense_brute_force(orc, N_d, N_m, N_t):
    F = RNG.standard_normal((N_t, N_d, N_m))
    m = RNG.standard_normal((N_t, N_m))
    d = RNG.standard_normal((N_t, N_d))
    A = dense_from_block_column(F)
    if A.size <= 200_000:
        Am, ATd = naive_matmul(A, m.ravel()), naive_matmul(A.T, d.ravel())
    else:
        Am, ATd = A @ m.ravel(), A.T @ d.ravel()
    assert rel(orc.matvec(F, m), Am) <= 1e-14
    assert rel(orc.rmatvec(F, d), ATd) <= 1e-14
    assert rel(orc.normal(F, m), A.T @ (A @ m.ravel())) <= 1e-13


# ---------------------------------------------------------------- eq (2.2)-(2.3): the paper's recurrence
def test_state_space_recurrence_pins_index_convention(orc):
    """F_k = B A^k C and w_{k+1} = A w_k + C m_k, d_{k+1} = B w_{k+1}, w_0 = 0.
    Zero-based output step i is the paper's d_{i+1} and must equal (F m)_i: no extra delay."""
    N_w, N_m, N_d, N_t = 5, 3, 2, 9
    A = RNG.standard_normal((N_w, N_w))
    A *= 0.9 / max(abs(np.linalg.eigvals(A)))
    B = RNG.standard_normal((N_d, N_w))
    C = RNG.standard_normal((N_w, N_m))
    F = np.stack([B @ np.linalg.matrix_power(A, k) @ C for k in range(N_t)])
    m = RNG.standard_normal((N_t, N_m))
    w = np.zeros(N_w)
    d_rec = np.zeros((N_t, N_d))
    for k in range(N_t):
        w = A @ w + C @ m[k]
        d_rec[k] = B @ w           # paper's d_{k+1}
    assert rel(orc.matvec(F, m), d_rec) <= 1e-13


# ---------------------------------------------------------------- impulses return the block column
def test_impulse_returns_block_column_bit_exact(orc):
    N_d, N_m, N_t = 3, 6, 8
    F = RNG.standard_normal((N_t, N_d, N_m))
    for j0, p0 in [(0, 0), (2, 4), (N_t - 1, N_m - 1)]:
        m = np.zeros((N_t, N_m)); m[j0, p0] = 1.0
        d = orc.matvec(F, m)
        for i in range(N_t):
            want = F[i - j0, :, p0] if i >= j0 else np.zeros(N_d)
            assert np.array_equal(d[i], want)          # exact: every other product is 0
    # transpose; i0 = N_t-1 catches "wrong half kept" in an FFT adjoint (R5)
    for i0, s0 in [(N_t - 1, 1), (0, 0), (3, 2)]:
        dd = np.zeros((N_t, N_d)); dd[i0, s0] = 1.0
        mm = orc.rmatvec(F, dd)
        for j in range(N_t):
            want = F[i0 - j, s0, :] if j <= i0 else np.zeros(N_m)
            assert np.array_equal(mm[j], want)


def test_causality_and_shift_equivariance(orc):
    """Block lower-triangular (causal) and block Toeplitz (shift-invariant)."""
    N_d, N_m, N_t = 2, 5, 10
    F = RNG.standard_normal((N_t, N_d, N_m))
    m = RNG.standard_normal((N_t, N_m))
    d = orc.matvec(F, m)
    i0 = 4
    m2 = m.copy(); m2[i0 + 1:] = RNG.standard_normal((N_t - i0 - 1, N_m))
    assert np.array_equal(orc.matvec(F, m2)[: i0 + 1], d[: i0 + 1])
    for tau in (1, 3, N_t - 1):
        ms = np.zeros_like(m); ms[tau:] = m[: N_t - tau]
        ds = orc.matvec(F, ms)
        assert np.all(ds[:tau] == 0.0)
        assert rel(ds[tau:], d[: N_t - tau]) <= 1e-15


def test_linearity_and_adjoint_identity(orc):
    N_d, N_m, N_t = 3, 17, 12
    F = RNG.standard_normal((N_t, N_d, N_m))
    a, b = RNG.standard_normal((2, N_t, N_m))
    d = RNG.standard_normal((N_t, N_d))
    al, be = 0.7, -1.9
    assert rel(orc.matvec(F, al * a + be * b), al * orc.matvec(F, a) + be * orc.matvec(F, b)) <= 1e-14
    lhs = np.vdot(orc.matvec(F, a), d)          # <F m, d>
    rhs = np.vdot(a, orc.rmatvec(F, d))         # <m, F^T d>
    assert abs(lhs - rhs) <= 1e-13 * max(abs(lhs), 1.0)


# ---------------------------------------------------------------- closed forms
def test_scalar_geometric_closed_form(orc):
    """N_d = N_m = 1, F_k = a^k, m_j = b^j  =>  d_i = (a^{i+1} - b^{i+1}) / (a - b); exact rationals."""
    N_t = 12
    a, b = Fraction(1, 2), Fraction(1, 4)
    F = np.array([float(a ** k) for k in range(N_t)]).reshape(N_t, 1, 1)
    m = np.array([float(b ** j) for j in range(N_t)]).reshape(N_t, 1)
    want = np.array([float((a ** (i + 1) - b ** (i + 1)) / (a - b)) for i in range(N_t)])
    got = orc.matvec(F, m).ravel()
    assert got[0] == 1.0 and got[1] == 0.75
    assert rel(got, want) <= 1e-15
    # a == b: d_i = (i+1) a^i
    got = orc.matvec(F, F.reshape(N_t, 1)).ravel()
    assert rel(got, [(i + 1) * float(a ** i) for i in range(N_t)]) <= 1e-15
    # transpose with d_i = b^i:  m'_j = b^j (1 - (ab)^{N_t-j}) / (1 - ab)
    want = [float(b ** j * (1 - (a * b) ** (N_t - j)) / (1 - a * b)) for j in range(N_t)]
    assert rel(orc.rmatvec(F, m).ravel(), want) <= 1e-15


def test_textbook_reductions(orc):
    N_d, N_m, N_t = 3, 4, 6
    F0 = RNG.standard_normal((N_d, N_m))
    m = RNG.standard_normal((N_t, N_m))
    # F_k = delta_{k0} F_0  =>  block diagonal
    F = np.zeros((N_t, N_d, N_m)); F[0] = F0
    assert rel(orc.matvec(F, m), m @ F0.T) <= 1e-15
    # N_d = N_m, F_k = delta_{k1} I  =>  pure one-step delay
    F = np.zeros((N_t, N_m, N_m)); F[1] = np.eye(N_m)
    d = orc.matvec(F, m)
    assert np.all(d[0] == 0) and np.array_equal(d[1:], m[:-1])
    # N_d = N_m = 1  =>  truncated linear convolution (library routine, test only)
    f, x = RNG.standard_normal(N_t * 3), RNG.standard_normal(N_t * 3)
    n = f.size
    assert rel(orc.matvec(f.reshape(n, 1, 1), x.reshape(n, 1)).ravel(), np.convolve(f, x)[:n]) <= 1e-14
    # transpose = truncated correlation
    want = np.array([sum(f[i - j] * x[i] for i in range(j, n)) for j in range(n)])
    assert rel(orc.rmatvec(f.reshape(n, 1, 1), x.reshape(n, 1)).ravel(), want) <= 1e-14


def test_exact_integer_case(orc):
    N_d, N_m, N_t = 3, 9, 7
    F = RNG.integers(-4, 5, (N_t, N_d, N_m)).astype(np.float64)
    m = RNG.integers(-4, 5, (N_t, N_m)).astype(np.float64)
    d = RNG.integers(-4, 5, (N_t, N_d)).astype(np.float64)
    A = dense_from_block_column(F)
    assert np.array_equal(orc.matvec(F, m).ravel(), A @ m.ravel())
    assert np.array_equal(orc.rmatvec(F, d).ravel(), A.T @ d.ravel())


def test_normal_operator_symmetric_psd(orc):
    """F^T F is the data-misfit Hessian with identity noise covariance (eq 2.12)."""
    N_d, N_m, N_t = 2, 6, 5
    F = RNG.standard_normal((N_t, N_d, N_m))
    a, b = RNG.standard_normal((2, N_t, N_m))
    Ha, Hb = orc.normal(F, a), orc.normal(F, b)
    assert abs(np.vdot(a, Hb) - np.vdot(Ha, b)) <= 1e-12 * abs(np.vdot(a, Hb))
    assert abs(np.vdot(a, Ha) - np.linalg.norm(orc.matvec(F, a)) ** 2) <= 1e-12 * np.vdot(a, Ha)


# ---------------------------------------------------------------- the two builds and the helpers
@pytest.mark.parametrize("N_d,N_m,N_t", [(4, 64, 32), (3, 1031, 9), (5, 2500, 6)])
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_blocked_equals_plain(N_d, N_m, N_t, dtype):
    F = RNG.standard_normal((N_t, N_d, N_m)).astype(dtype)
    m = RNG.standard_normal((N_t, N_m)).astype(dtype)
    d = RNG.standard_normal((N_t, N_d)).astype(dtype)
    assert rel(ob.matvec(F, m), op.matvec(F, m)) <= 1e-14
    assert rel(ob.rmatvec(F, d), op.rmatvec(F, d)) <= 1e-14


def test_blocked_accepts_slices():
    N_d, N_m, N_t = 6, 300, 8
    F = RNG.standard_normal((N_t, N_d, N_m)).astype(np.float32)
    m = RNG.standard_normal((N_t, N_m)).astype(np.float32)
    d = RNG.standard_normal((N_t, N_d)).astype(np.float32)
    full_d, full_m = op.matvec(F, m), op.rmatvec(F, d)
    assert rel(ob.matvec(F[:, 2:5, :], m), full_d[:, 2:5]) <= 1e-14        # sensor slice -> rows of d
    assert rel(ob.rmatvec(F[:, :, 100:228], d), full_m[:, 100:228]) <= 1e-14  # parameter slice -> cols of m'


def test_entry_helpers_and_multi_rhs():
    N_d, N_m, N_t, k = 3, 11, 7, 4
    F = RNG.standard_normal((N_t, N_d, N_m))
    M = RNG.standard_normal((N_t, N_m, k))
    D = RNG.standard_normal((N_t, N_d, k))
    dk, mk = op.matvec(F, M), op.rmatvec(F, D)
    for r in range(k):           # each column independently (K is built column by column)
        assert rel(dk[..., r], op.matvec(F, M[..., r])) <= 1e-15
        assert rel(mk[..., r], op.rmatvec(F, D[..., r])) <= 1e-15
    A = dense_from_block_column(F)
    d, mm = A @ M[..., 0].ravel(), A.T @ D[..., 0].ravel()
    for i, s in itertools.product((0, 3, N_t - 1), (0, N_d - 1)):
        assert abs(op.matvec_entry(F, M[..., 0], i, s) - d[i * N_d + s]) <= 1e-13
    for j, p in itertools.product((0, 2, N_t - 1), (0, N_m - 1)):
        assert abs(op.rmatvec_entry(F, D[..., 0], j, p) - mm[j * N_m + p]) <= 1e-13


# ---------------------------------------------------------------- coarser output grid (p2q, reading R19)
@pytest.mark.parametrize("N_q,N_m,N_t,r", [(2, 3, 6, 2), (1, 4, 9, 3), (3, 2, 8, 8), (2, 5, 10, 5), (2, 3, 7, 1)])
def test_decimated_output_dense_and_adjoint(N_q, N_m, N_t, r):
    F = RNG.standard_normal((N_t, N_q, N_m))
    m = RNG.standard_normal((N_t, N_m))
    q = RNG.standard_normal((N_t // r, N_q))
    A = dense_from_block_column(F)
    keep = np.concatenate([np.arange(N_q) + (r * (I + 1) - 1) * N_q for I in range(N_t // r)])
    Aq = A[keep]                                             # S A: the rows of the fine steps r-1, 2r-1, ...
    assert rel(op.matvec_decimated(F, m, r), Aq @ m.ravel()) <= 1e-14
    assert rel(op.rmatvec_decimated(F, q, r), Aq.T @ q.ravel()) <= 1e-14
    lhs = np.vdot(op.matvec_decimated(F, m, r), q)
    assert abs(lhs - np.vdot(m, op.rmatvec_decimated(F, q, r))) <= 1e-13 * max(1.0, abs(lhs))
    assert np.array_equal(op.matvec_decimated(F, m, r), op.matvec(F, m)[r - 1::r])       # S (F m): the same sums
    up = np.zeros((N_t, N_q)); up[r - 1::r] = q
    assert rel(op.rmatvec_decimated(F, q, r), op.rmatvec(F, up)) <= 1e-15                  # F^T (S^T q)
    if r == 1:
        assert np.array_equal(op.matvec_decimated(F, m, 1), op.matvec(F, m))
        assert np.array_equal(op.rmatvec_decimated(F, q, 1), op.rmatvec(F, q))


def test_decimated_output_is_the_sampled_recurrence():
    # eq (2.2)-(2.3) with a QoI observation operator B_q (eq 2.14-2.16), sampled every r steps:
    # q_I = B_q w_{r(I+1)} in the paper's 1-based state index, i.e. after r(I+1) steps of the recurrence
    n_w, N_q, N_m, N_t, r = 5, 2, 3, 12, 4
    A = RNG.standard_normal((n_w, n_w)); A *= 0.9 / np.abs(np.linalg.eigvals(A)).max()
    Bq, C = RNG.standard_normal((N_q, n_w)), RNG.standard_normal((n_w, N_m))
    F = np.stack([Bq @ np.linalg.matrix_power(A, k) @ C for k in range(N_t)])
    m = RNG.standard_normal((N_t, N_m))
    w, out = np.zeros(n_w), []
    for k in range(N_t):
        w = A @ w + C @ m[k]
        if (k + 1) % r == 0:
            out.append(Bq @ w)
    assert rel(op.matvec_decimated(F, m, r), np.array(out)) <= 1e-13
