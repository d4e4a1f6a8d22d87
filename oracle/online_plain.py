"""CPU ORACLE (test infrastructure, NOT the product path) - the data-space machinery of
Phase 2 and the online inference of Phase 4, written out from the paper.

What the paper defines (PAPER.md = /root/reference/PAPER.md):

  * time-invariant prior covariance, block diagonal in time ("spatial correlation only,
    leading to a shift-invariant prior covariance matrix with block-diagonal structure",
    PAPER.md:368):  Gamma_prior(m) = I_{N_t} (x) Gamma_s,  Gamma_s (N_m x N_m) SPD;
  * G* := Gamma_prior(m) F*  (PAPER.md:302), which is then block Toeplitz with the structure
    of F*: its blocks are Gamma_s F_k^T, so G* is the transpose-structured operator of the
    block column  G_k := F_k Gamma_s  (N_d x N_m), and  G* d = rmatvec(G, d);
  * K := Gamma_noise + F G*  (eq 4.7), computed "column-by-column"
    (PAPER.md:296, 407), Gamma_noise diagonal;
  * K = L L^T Cholesky-factorised offline, "triangular solves are done in the online phase"
    (PAPER.md:294, 407);
  * Gamma_post(m) = (I - G* K^{-1} F) Gamma_prior(m)                       (eq 4.7)
  * m_map = (I - G* K^{-1} F) G* Gamma_noise^{-1} d_obs   (+ 0: m_prior = 0)
                                                                           (eq 4.13)

Every function follows the cited passage step by step in the paper's order, in fp64, with
the plain block convolution of oracle/toeplitz_plain.py for F and G* (no FFT anywhere) and
textbook substitution loops for the triangular solves; numpy.linalg.cholesky (LAPACK) is the
library step for the factorisation, which the paper also leaves to a library.

Layouts: block columns [N_t, N_d, N_m]; parameter vectors [N_t, N_m]; data vectors
[N_t, N_d]; the data-space index of K and L is  row = i*N_d + s  (the paper's stacking of
d); noise_var holds the diagonal of Gamma_noise as [N_t, N_d].

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this module.  It shares no code with the CUDA path.
Pins: tests/test_oracle_online_pins.py - dense normal equations (eq 2.12), the dense inverse
Hessian (eq 2.13 / 4.5) against eq (4.6)/(4.7), dense assembly of K, library triangular
solves, first-difference closed form, data fit in the zero-noise limit.  No function here is
"parity unpinned".
"""
from __future__ import annotations

import numpy as np

from . import toeplitz_plain as tp


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a), dtype=np.float64)


def gstar_block_column(F, Gamma_s) -> np.ndarray:
    """Block column G_k = F_k Gamma_s of G* = Gamma_prior F* (PAPER.md:302).

    Gamma_s: [N_m, N_m] symmetric positive definite, or [N_m] = its diagonal.
    """
    F, Gs = _f64(F), _f64(Gamma_s)
    if Gs.ndim == 1:
        return F * Gs[None, None, :]
    return np.stack([F[k] @ Gs for k in range(F.shape[0])])


def apply_gstar(G, d) -> np.ndarray:
    """G* d: block (j, i) of G* is G_{i-j}^T for i >= j - the structure of F*."""
    return tp.rmatvec(G, d)


def assemble_K(F, G, noise_var) -> np.ndarray:
    """K = Gamma_noise + F G*, column by column.

    Column (i', s') is F (G* e_{(i',s')}) + Gamma_noise e_{(i',s')}.  Returns [n, n], n = N_t N_d,
    index i*N_d + s.  All n unit vectors go through the column-independent k-RHS form of the
    block convolution at once.
    """
    F, G, nv = _f64(F), _f64(G), _f64(noise_var)
    N_t, N_d, _ = F.shape
    n = N_t * N_d
    E = np.eye(n, dtype=np.float64).reshape(N_t, N_d, n)   # E[:, :, c] = unit data vector c
    cols = tp.matvec(F, apply_gstar(G, E))                  # [N_t, N_d, n]
    K = cols.reshape(n, n)
    K[np.arange(n), np.arange(n)] += nv.reshape(n)
    return K


def cholesky(K) -> np.ndarray:
    """Lower Cholesky factor, K = L L^T.  Library step (LAPACK potrf)."""
    return np.linalg.cholesky(_f64(K))


def forward_substitution(L, b) -> np.ndarray:
    """Solves L y = b for lower-triangular L, row by row: y_i = (b_i - sum_{j<i} L_ij y_j) / L_ii."""
    L, b = _f64(L), _f64(b)
    n = L.shape[0]
    y = np.zeros_like(b)
    for i in range(n):
        y[i] = (b[i] - L[i, :i] @ y[:i]) / L[i, i]
    return y


def back_substitution_T(L, y) -> np.ndarray:
    """Solves L^T x = y for lower-triangular L, last row first: x_i = (y_i - sum_{j>i} L_ji x_j) / L_ii."""
    L, y = _f64(L), _f64(y)
    n = L.shape[0]
    x = np.zeros_like(y)
    for i in range(n - 1, -1, -1):
        x[i] = (y[i] - L[i + 1:, i] @ x[i + 1:]) / L[i, i]
    return x


def chol_solve(L, b) -> np.ndarray:
    """K^{-1} b with K = L L^T: the two triangular solves of the online phase."""
    return back_substitution_T(L, forward_substitution(L, b))


def map_point(F, G, noise_var, L, d_obs, conv=tp) -> np.ndarray:
    """m_map of eq (4.13) with m_prior = 0, in the paper's order of operations
    (footnote 14: G*, F, solve with the prefactorised K, G*):

        y = Gamma_noise^{-1} d_obs ;  a = G* y ;  b = F a ;  c = K^{-1} b ;  m_map = a - G* c.

    conv: the oracle module that supplies the block convolution (toeplitz_plain, or toeplitz_blocked - the same
    sums in C/OpenMP - for sizes where the numpy loops are too slow).
    """
    nv, d = _f64(noise_var), _f64(d_obs)
    N_t, N_d = F.shape[0], F.shape[1]
    y = d / nv
    a = conv.rmatvec(G, y)                                   # G* y
    b = conv.matvec(F, a)
    c = chol_solve(L, b.reshape(N_t * N_d)).reshape(N_t, N_d)
    return a - conv.rmatvec(G, c)


def smw_apply(F, G, L, u, conv=tp) -> np.ndarray:
    """(I - G* K^{-1} F) u: the operator of eq (4.7) and eq (4.8), in the paper's order
    F, K-solve, G*, subtract.  u: [N_t, N_m].  With u = Gamma_prior v it is Gamma_post(m) v; with u = m_prior it is
    the prior-mean contribution m_map^prior of eq (4.8)."""
    u = _f64(u)
    N_t, N_d = F.shape[0], F.shape[1]
    c = chol_solve(L, conv.matvec(F, u).reshape(N_t * N_d)).reshape(N_t, N_d)
    return u - conv.rmatvec(G, c)


def post_cov_apply(F, G, L, Gamma_s, v) -> np.ndarray:
    """Gamma_post(m) v = (I - G* K^{-1} F) Gamma_prior(m) v, eq (4.7).

    Gamma_s as in gstar_block_column; v: [N_t, N_m].
    """
    F, G, Gs, v = _f64(F), _f64(G), _f64(Gamma_s), _f64(v)
    N_t, N_d, _ = F.shape
    u = v * Gs[None, :] if Gs.ndim == 1 else v @ Gs          # Gamma_prior v (Gamma_s symmetric)
    c = chol_solve(L, tp.matvec(F, u).reshape(N_t * N_d)).reshape(N_t, N_d)
    return u - apply_gstar(G, c)


def K_entry(F_s, G_s2, i: int, i2: int, noise: float = 0.0) -> float:
    """One entry K[(i, s), (i2, s2)] of K = Gamma_noise + F G* (PAPER.md:306), for sampled parity at sizes where
    assemble_K is out of reach: row (i, s) of F times column (i2, s2) of G*,

        sum_{j=0..min(i, i2)} F_{i-j}[s, :] . G_{i2-j}[s2, :]     (+ noise if (i, s) == (i2, s2), passed by the caller).

    F_s: [N_t, N_m] = F[:, s, :];  G_s2: [N_t, N_m] = G[:, s2, :].
    """
    acc = 0.0
    for j in range(min(i, i2) + 1):
        acc += float(np.dot(np.asarray(F_s[i - j], dtype=np.float64), np.asarray(G_s2[i2 - j], dtype=np.float64)))
    return acc + noise


# ---------------------------------------------------------------------------------------------
# Phase 3: QoI posterior covariance and the data-to-QoI map, through the p2q map F_q on its
# coarser output grid (oracle/toeplitz_plain.matvec_decimated, reading R19) and G_q* = Gamma_prior F_q*.
# ---------------------------------------------------------------------------------------------
def post_cov_q_apply(F, G, L, Fq, Gq, r: int, v) -> np.ndarray:
    """Gamma_post(q) v = F_q (I - G* K^{-1} F) G_q* v, eq (4.10).  v: [N_t/r, N_q]."""
    a = tp.rmatvec_decimated(Gq, v, r)                     # G_q* v
    return tp.matvec_decimated(Fq, smw_apply(F, G, L, a), r)


def d2q_apply(F, G, noise_var, L, Fq, r: int, d_obs) -> np.ndarray:
    """q_map = Q d_obs with Q = F_q (I - G* K^{-1} F) G* Gamma_noise^{-1}, eq (4.11)/(4.14), m_prior = 0."""
    return tp.matvec_decimated(Fq, map_point(F, G, noise_var, L, d_obs), r)
