"""ORACLE (TEST INFRASTRUCTURE ONLY): the Lanczos algorithm exactly as
Algorithm 1 of the paper states it, fp64, three explicit
vectors f_{j-1}, f_j, q_j, no fusion, no in-place trick, no lazy
normalisation.  `matvec` is any callable y = H x (dense matrix product for the
small cases, the tier-1 matrix-free product for the large ones).

Output indexing (reading Q9): alpha[j-1] = a_j, beta[j-1] = b_{j+1}
for j = 1..m, so T_m of PAPER.md:150 has diagonal alpha[0:m] and off-diagonal
beta[0:m-1].

Breakdown (Algorithm 1 lines 8-10, reading Q11): stop after the
iteration in which b_{j+1} <= tau * max(1, max_k |a_k|) or b_{j+1} is not
finite; tau = 0 is the paper's literal test.

Pins: the Krylov identities checked in tests/test_oracle_pins.py (T_m equals
F^T H F for the explicitly stored Lanczos basis on a small dense H; lambda_min
of T_dim equals dense eigvalsh), and the closed-form energies.
"""
from __future__ import annotations

import numpy as np


def lanczos(matvec, f1: np.ndarray, m: int, tau: float = 1e-10, keep_basis: bool = False):
    f1 = np.asarray(f1, dtype=np.float64)
    f = f1 / np.sqrt(np.dot(f1, f1))          # "a random initial vector f_1 of norm 1"
    f_prev = np.zeros_like(f)                 # line 2: f_0 <- 0
    b = 0.0                                   # line 1: b_1 <- 0
    alpha, beta = [], []
    basis = [f.copy()] if keep_basis else None
    for _ in range(m):                        # line 3
        q = matvec(f) - b * f_prev            # line 4
        a = float(np.dot(q, f))               # line 5
        q = q - a * f                         # line 6
        b_next = float(np.sqrt(np.dot(q, q)))  # line 7
        alpha.append(a)
        beta.append(b_next)
        scale = max(1.0, max(abs(x) for x in alpha))
        if not np.isfinite(b_next) or b_next <= tau * scale:   # lines 8-10
            break
        f_prev = f
        f = q / b_next                        # line 11
        b = b_next
        if keep_basis:
            basis.append(f.copy())
    alpha = np.array(alpha)
    beta = np.array(beta)
    if keep_basis:
        return alpha, beta, np.array(basis)
    return alpha, beta


def tridiagonal_matrix(alpha: np.ndarray, beta: np.ndarray, m: int | None = None) -> np.ndarray:
    """T_m of PAPER.md:150."""
    m = len(alpha) if m is None else m
    T = np.diag(np.asarray(alpha[:m], dtype=np.float64))
    for k in range(m - 1):
        T[k, k + 1] = T[k + 1, k] = beta[k]
    return T


def ground_energy(alpha: np.ndarray, beta: np.ndarray, m: int | None = None) -> float:
    """E_0^(m) = lambda_min(T_m), "with standard methods":
    LAPACK's dense symmetric eigensolver on the explicit T_m."""
    return float(np.linalg.eigvalsh(tridiagonal_matrix(alpha, beta, m))[0])
