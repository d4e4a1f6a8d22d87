"""Pins for oracle/online_plain.py (CPU only): the data-space machinery (K, its triangular
solves) and the online MAP point of eq (4.13) are checked against what the paper and the
mathematics fix - dense linear algebra on explicitly assembled matrices at tiny sizes,
library routines and closed forms - never against the oracle itself.

Dense reference objects (assembled entry by entry from the definitions):
    A    = the p2o matrix of eq (2.5)
    Gp   = Gamma_prior(m) = I_{N_t} (x) Gamma_s
    Gn   = Gamma_noise, diagonal
    H    = A^T Gn^{-1} A + Gp^{-1}                                     (eq 2.12)
"""
import numpy as np
import pytest
import scipy.linalg

from oracle import online_plain as oo
from oracle import toeplitz_plain as op

RNG = np.random.default_rng(4130)
SHAPES = [(3, 5, 7), (2, 6, 4), (1, 3, 5), (4, 2, 3), (2, 1, 6)]   # (N_d, N_m, N_t)


def dense_from_block_column(F):
    N_t, N_d, N_m = F.shape
    A = np.zeros((N_t * N_d, N_t * N_m))
    for i in range(N_t):
        for j in range(i + 1):
            A[i * N_d:(i + 1) * N_d, j * N_m:(j + 1) * N_m] = F[i - j]
    return A


def spd(n, rng, cond=20.0):
    Q, _ = np.linalg.qr(rng.standard_normal((n, n)))
    return (Q * np.linspace(1.0, cond, n)) @ Q.T


def setup(N_d, N_m, N_t, diag_prior=False):
    F = RNG.standard_normal((N_t, N_d, N_m)) * np.exp(-np.arange(N_t) / 3.0)[:, None, None]
    Gs = RNG.uniform(0.5, 2.0, N_m) if diag_prior else spd(N_m, RNG)
    nv = RNG.uniform(0.05, 0.2, (N_t, N_d))
    A = dense_from_block_column(F)
    Gs_full = np.diag(Gs) if diag_prior else Gs
    Gp = np.kron(np.eye(N_t), Gs_full)
    return F, Gs, nv, A, Gp


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / max(np.linalg.norm(np.ravel(b)), 1e-300)


# ------------------------------------------------------------------ G* = Gamma_prior F^*
@pytest.mark.parametrize("N_d,N_m,N_t", SHAPES)
@pytest.mark.parametrize("diag_prior", [False, True])
def test_gstar_is_prior_times_adjoint(N_d, N_m, N_t, diag_prior):
    F, Gs, nv, A, Gp = setup(N_d, N_m, N_t, diag_prior)
    G = oo.gstar_block_column(F, Gs)
    d = RNG.standard_normal((N_t, N_d))
    assert rel(oo.apply_gstar(G, d), Gp @ (A.T @ d.ravel())) <= 1e-13
    # G* is block Toeplitz with the structure of F*: dense(G)^T = Gp A^T
    assert rel(dense_from_block_column(G).T, Gp @ A.T) <= 1e-13


# ------------------------------------------------------------------ K = Gamma_noise + F G*  (eq 4.6/4.7)
@pytest.mark.parametrize("N_d,N_m,N_t", SHAPES)
def test_K_dense(N_d, N_m, N_t):
    F, Gs, nv, A, Gp = setup(N_d, N_m, N_t)
    K = oo.assemble_K(F, oo.gstar_block_column(F, Gs), nv)
    K_ref = np.diag(nv.ravel()) + A @ Gp @ A.T             # eq (4.6): Gamma_noise + F Gamma_prior F*
    assert rel(K, K_ref) <= 1e-13
    assert rel(K, K.T) <= 1e-13
    assert np.linalg.eigvalsh(0.5 * (K + K.T)).min() >= nv.min() * (1 - 1e-9)   # K - Gamma_noise is PSD


def test_K_entry_equals_assembled_K():
    N_d, N_m, N_t = 3, 5, 7
    F, Gs, nv, A, Gp = setup(N_d, N_m, N_t)
    G = oo.gstar_block_column(F, Gs)
    K_ref = np.diag(nv.ravel()) + A @ Gp @ A.T
    for i in range(N_t):
        for s in range(N_d):
            for i2 in (0, 3, N_t - 1):
                for s2 in range(N_d):
                    noise = nv[i, s] if (i, s) == (i2, s2) else 0.0
                    got = oo.K_entry(F[:, s, :], G[:, s2, :], i, i2, noise)
                    assert abs(got - K_ref[i * N_d + s, i2 * N_d + s2]) <= 1e-12 * np.abs(K_ref).max()


# ------------------------------------------------------------------ triangular solves
@pytest.mark.parametrize("n", [1, 2, 7, 64, 130])
def test_substitution_against_lapack(n):
    L = np.tril(RNG.standard_normal((n, n))) + np.eye(n) * (2.0 + np.sqrt(n))
    b = RNG.standard_normal(n)
    y = oo.forward_substitution(L, b)
    x = oo.back_substitution_T(L, b)
    assert rel(y, scipy.linalg.solve_triangular(L, b, lower=True)) <= 1e-13
    assert rel(x, scipy.linalg.solve_triangular(L, b, lower=True, trans="T")) <= 1e-13
    assert rel(L @ y, b) <= 1e-13 and rel(L.T @ x, b) <= 1e-13
    K = L @ L.T
    assert rel(oo.chol_solve(L, b), np.linalg.solve(K, b)) <= 1e-10


def test_substitution_closed_forms():
    # L = lower triangle of ones: L y = b  <=>  y = first differences of b;  L^T x = b  <=>  x_i = b_i - b_{i+1}
    n = 9
    L = np.tril(np.ones((n, n)))
    b = np.arange(1.0, n + 1) ** 2
    assert np.array_equal(oo.forward_substitution(L, b), np.diff(b, prepend=0.0))
    assert np.array_equal(oo.back_substitution_T(L, b), b - np.append(b[1:], 0.0))
    # bidiagonal L (1 on the diagonal, -a below): y_i = sum_j a^{i-j} b_j, exactly representable for a = 1/2
    a = 0.5
    Lb = np.eye(n) - a * np.eye(n, k=-1)
    e0 = np.zeros(n); e0[0] = 1.0
    assert np.array_equal(oo.forward_substitution(Lb, e0), a ** np.arange(n))
    en = np.zeros(n); en[-1] = 1.0
    assert np.array_equal(oo.back_substitution_T(Lb, en), a ** np.arange(n)[::-1])


def test_cholesky_reconstructs():
    K = spd(40, RNG, cond=100.0)
    L = oo.cholesky(K)
    assert np.array_equal(L, np.tril(L)) and (np.diag(L) > 0).all()
    assert rel(L @ L.T, K) <= 1e-14


# ------------------------------------------------------------------ eq (4.13) against eq (2.12)
@pytest.mark.parametrize("N_d,N_m,N_t", SHAPES)
@pytest.mark.parametrize("diag_prior", [False, True])
def test_map_point_solves_normal_equations(N_d, N_m, N_t, diag_prior):
    F, Gs, nv, A, Gp = setup(N_d, N_m, N_t, diag_prior)
    G = oo.gstar_block_column(F, Gs)
    L = oo.cholesky(oo.assemble_K(F, G, nv))
    d_obs = RNG.standard_normal((N_t, N_d))
    m_map = oo.map_point(F, G, nv, L, d_obs)
    Gn_inv = np.diag(1.0 / nv.ravel())
    H = A.T @ Gn_inv @ A + np.linalg.inv(Gp)                         # Hessian of eq (2.12)
    m_ref = np.linalg.solve(H, A.T @ Gn_inv @ d_obs.ravel())         # eq (2.12) with m_prior = 0
    assert rel(m_map, m_ref) <= 1e-10
    # it minimises the negative log posterior of eq (2.11): the gradient vanishes
    grad = A.T @ Gn_inv @ (A @ m_map.ravel() - d_obs.ravel()) + np.linalg.solve(Gp, m_map.ravel())
    assert np.linalg.norm(grad) <= 1e-9 * np.linalg.norm(A.T @ Gn_inv @ d_obs.ravel())
    # the algebraically equal gain form  Gamma_prior F* K^{-1} d_obs  (K = Gamma_noise + F G*)
    K_ref = np.diag(nv.ravel()) + A @ Gp @ A.T
    assert rel(m_map, Gp @ A.T @ np.linalg.solve(K_ref, d_obs.ravel())) <= 1e-10


@pytest.mark.parametrize("N_d,N_m,N_t", SHAPES[:3])
def test_post_cov_is_inverse_hessian(N_d, N_m, N_t):
    # eq (4.7) (I - G* K^{-1} F) Gamma_prior  ==  H^{-1} of eq (2.13)/(4.5), column by column
    F, Gs, nv, A, Gp = setup(N_d, N_m, N_t)
    G = oo.gstar_block_column(F, Gs)
    L = oo.cholesky(oo.assemble_K(F, G, nv))
    H = A.T @ np.diag(1.0 / nv.ravel()) @ A + np.linalg.inv(Gp)
    Hinv = np.linalg.inv(H)
    n = N_t * N_m
    for c in RNG.choice(n, size=min(n, 6), replace=False):
        e = np.zeros(n); e[c] = 1.0
        col = oo.post_cov_apply(F, G, L, Gs, e.reshape(N_t, N_m))
        assert rel(col, Hinv[:, c]) <= 1e-9


@pytest.mark.parametrize("N_d,N_m,N_t", SHAPES[:3])
def test_smw_operator(N_d, N_m, N_t):
    # (I - G* K^{-1} F) u:  with u = Gamma_prior v it is H^{-1} v (eq 4.7 vs 2.13); with u = m_prior it is the prior-mean
    # term of eq (4.8), Gamma_post Gamma_prior^{-1} m_prior, and together with eq (4.13) it solves eq (2.12) with m_prior != 0
    F, Gs, nv, A, Gp = setup(N_d, N_m, N_t)
    G = oo.gstar_block_column(F, Gs)
    L = oo.cholesky(oo.assemble_K(F, G, nv))
    Gn_inv = np.diag(1.0 / nv.ravel())
    H = A.T @ Gn_inv @ A + np.linalg.inv(Gp)
    v = RNG.standard_normal((N_t, N_m))
    u = (Gp @ v.ravel()).reshape(N_t, N_m)
    assert rel(oo.smw_apply(F, G, L, u), np.linalg.solve(H, v.ravel())) <= 1e-9
    assert rel(oo.smw_apply(F, G, L, u), oo.post_cov_apply(F, G, L, Gs, v)) <= 1e-13
    m_prior = RNG.standard_normal((N_t, N_m))
    d_obs = RNG.standard_normal((N_t, N_d))
    m_full = np.linalg.solve(H, A.T @ Gn_inv @ d_obs.ravel() + np.linalg.solve(Gp, m_prior.ravel()))   # eq (2.12)
    got = oo.map_point(F, G, nv, L, d_obs) + oo.smw_apply(F, G, L, m_prior)                              # eq (4.13) + (4.8)
    assert rel(got, m_full) <= 1e-9


@pytest.mark.parametrize("N_d,N_m,N_t,N_q,r", [(3, 5, 6, 2, 2), (2, 4, 9, 1, 3), (1, 3, 4, 2, 1)])
def test_phase3_against_dense(N_d, N_m, N_t, N_q, r):
    # eq (4.9)/(2.18): Gamma_post(q) = F_q H^{-1} F_q^*;  eq (4.11): Q = F_q H^{-1} F^* Gamma_noise^{-1}, with F_q = S A_q
    F, Gs, nv, A, Gp = setup(N_d, N_m, N_t)
    Fq = RNG.standard_normal((N_t, N_q, N_m)) * np.exp(-np.arange(N_t) / 3.0)[:, None, None]
    G, Gq = oo.gstar_block_column(F, Gs), oo.gstar_block_column(Fq, Gs)
    L = oo.cholesky(oo.assemble_K(F, G, nv))
    Aq_fine = dense_from_block_column(Fq)
    keep = np.concatenate([np.arange(N_q) + (r * (I + 1) - 1) * N_q for I in range(N_t // r)])
    Aq = Aq_fine[keep]
    Gn_inv = np.diag(1.0 / nv.ravel())
    Hinv = np.linalg.inv(A.T @ Gn_inv @ A + np.linalg.inv(Gp))
    v = RNG.standard_normal((N_t // r, N_q))
    d_obs = RNG.standard_normal((N_t, N_d))
    assert rel(oo.post_cov_q_apply(F, G, L, Fq, Gq, r, v), Aq @ Hinv @ Aq.T @ v.ravel()) <= 1e-9
    assert rel(oo.d2q_apply(F, G, nv, L, Fq, r, d_obs), Aq @ Hinv @ A.T @ Gn_inv @ d_obs.ravel()) <= 1e-9


def test_zero_noise_limit_fits_the_data():
    # Gamma_noise -> 0: K -> F G*, so F m_map = F G* K^{-1} d_obs -> d_obs (N_m N_t >= N_d N_t, F full row rank)
    N_d, N_m, N_t = 2, 6, 5
    F, Gs, _, A, Gp = setup(N_d, N_m, N_t)
    # exactly: F m_map - d_obs = -Gamma_noise K^{-1} d_obs, so the misfit is bounded by noise * ||K^{-1}||
    nv = np.full((N_t, N_d), 1e-6)
    G = oo.gstar_block_column(F, Gs)
    K = oo.assemble_K(F, G, nv)
    L = oo.cholesky(K)
    d_obs = RNG.standard_normal((N_t, N_d))
    m_map = oo.map_point(F, G, nv, L, d_obs)
    bound = 1e-6 * np.linalg.norm(np.linalg.inv(A @ Gp @ A.T), 2)
    assert bound < 1e-3
    assert rel(op.matvec(F, m_map), d_obs) <= 1.01 * bound + 1e-7


def test_infinite_noise_limit_returns_prior_mean():
    N_d, N_m, N_t = 2, 4, 5
    F, Gs, _, A, Gp = setup(N_d, N_m, N_t)
    nv = np.full((N_t, N_d), 1e12)
    G = oo.gstar_block_column(F, Gs)
    L = oo.cholesky(oo.assemble_K(F, G, nv))
    d_obs = RNG.standard_normal((N_t, N_d))
    m_map = oo.map_point(F, G, nv, L, d_obs)
    # first order in 1/noise: m_map -> Gamma_prior F* Gamma_noise^{-1} d_obs
    assert rel(m_map, Gp @ A.T @ (d_obs.ravel() / nv.ravel())) <= 1e-8


# ------------------------------------------------------------------ reading R20: the algebra behind tt_assemble_K_direct / tt_qoi_direct
def _toeplitz_product(Acol, Bcol):
    """[(i,q),(t,s)] -> sum_{j <= min(i,t)} A_{i-j}[q,:] . B_{t-j}[s,:], written as the GPU path forms it: one product of the
    block columns seen as matrices, then running sums down the block diagonals.  Plain numpy, no oracle code."""
    N_t, Na, N_m = Acol.shape
    Nb = Bcol.shape[1]
    W = Acol.reshape(N_t * Na, N_m) @ Bcol.reshape(N_t * Nb, N_m).T
    P = W.copy()
    for i in range(1, N_t):
        for t in range(1, N_t):
            P[i * Na:(i + 1) * Na, t * Nb:(t + 1) * Nb] += P[(i - 1) * Na:i * Na, (t - 1) * Nb:t * Nb]
    return P


@pytest.mark.parametrize("N_d,N_m,N_t", SHAPES)
def test_K_is_one_product_of_the_block_columns_plus_running_sums(N_d, N_m, N_t):
    F, Gs, nv, A, Gp = setup(N_d, N_m, N_t)
    G = oo.gstar_block_column(F, Gs)
    K_direct = _toeplitz_product(F, G) + np.diag(nv.ravel())
    assert rel(K_direct, oo.assemble_K(F, G, nv)) <= 1e-13
    assert rel(K_direct, np.diag(nv.ravel()) + A @ Gp @ A.T) <= 1e-13


@pytest.mark.parametrize("r", [1, 2, 3])
def test_dense_Q_and_post_cov_q_from_toeplitz_products(r):
    """Q = B K^{-1} and Gamma_post(q) = A - Q B^T with B = F_q G*, A = F_q G_q* on the coarse rows (R19), against the operator
    forms of eq (4.11) and eq (4.10) applied to every unit vector."""
    N_d, N_q, N_m, N_t = 2, 3, 7, 6
    F, Gs, nv, _, _ = setup(N_d, N_m, N_t)
    Fq = RNG.standard_normal((N_t, N_q, N_m)) * np.exp(-np.arange(N_t) / 2.0)[:, None, None]
    G, Gq = oo.gstar_block_column(F, Gs), oo.gstar_block_column(Fq, Gs)
    K = oo.assemble_K(F, G, nv)
    L = oo.cholesky(K)
    rows = np.array([(r * (I + 1) - 1) * N_q + q for I in range(N_t // r) for q in range(N_q)])
    B = _toeplitz_product(Fq, G)[rows]
    Amat = _toeplitz_product(Fq, Gq)[np.ix_(rows, rows)]
    Q = np.linalg.solve(K, B.T).T
    C = Amat - Q @ B.T
    n, nq = N_t * N_d, len(rows)
    Q_ref = np.stack([oo.d2q_apply(F, G, nv, L, Fq, r, e.reshape(N_t, N_d)).ravel() for e in np.eye(n)], axis=1)
    C_ref = np.stack([oo.post_cov_q_apply(F, G, L, Fq, Gq, r, e.reshape(N_t // r, N_q)).ravel() for e in np.eye(nq)], axis=1)
    assert rel(Q, Q_ref) <= 1e-11
    assert rel(C, C_ref) <= 1e-11
