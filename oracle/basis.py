"""ORACLE (test infrastructure, not product code) -- LGL basis and 1-D DG operators.

Plain NumPy, fp64, written from /root/reference/PAPER.md (arXiv 2202.13532) Section 5.2.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this package; it shares no code with paper_2202_13532_b200/ (the CUDA path).

Every function cites the equation it restates.  Index convention (reading C11):
(Upsilon F)_j = sum_k Upsilon[j, k] F_k, i.e. the paper's upper index is the row.
Parity pins: tests/test_oracle_basis.py (closed-form nodes/weights n=2..7, quadrature
exactness, brute-force mass matrix, Eq.53==Eq.57, Eq.55==Eq.58, invariants).
"""
from __future__ import annotations

import numpy as np
from numpy.polynomial import legendre as npleg


def legendre_table(n: int, xi: np.ndarray):
    """P_s(xi) and P'_s(xi) for s = 0..n-1 by the three-term (Bonnet) recurrence.
    Returns (P, dP) each of shape [n, len(xi)].  (Used by Eq. 45-58.)"""
    xi = np.asarray(xi, dtype=np.float64)
    P = np.zeros((n, xi.size))
    dP = np.zeros((n, xi.size))
    P[0] = 1.0
    if n > 1:
        P[1] = xi
        dP[1] = 1.0
    for s in range(1, n - 1):
        P[s + 1] = ((2 * s + 1) * xi * P[s] - s * P[s - 1]) / (s + 1)
        dP[s + 1] = dP[s - 1] + (2 * s + 1) * P[s]
    return P, dP


def lgl_nodes_weights(n: int):
    """Eq. 45: nodes are the roots of (1 - xi^2) P'_{n-1}(xi); weights
    w_j = 2 / (n (n-1) P_{n-1}(xi_j)^2).  Roots of P'_{n-1} via the Legendre-series
    derivative (library root finder), polished by two Newton steps on P'_{n-1}."""
    if n < 2:
        raise ValueError("LGL needs n >= 2")
    c = np.zeros(n)
    c[n - 1] = 1.0                                  # P_{n-1} as a Legendre series
    interior = np.sort(npleg.legroots(npleg.legder(c))) if n > 2 else np.zeros(0)
    d1 = npleg.legder(c)
    d2 = npleg.legder(c, 2)
    for _ in range(2):
        interior = interior - npleg.legval(interior, d1) / npleg.legval(interior, d2)
    xi = np.concatenate(([-1.0], interior, [1.0]))
    xi = 0.5 * (xi - xi[::-1])                      # enforce exact antisymmetry
    Pn1 = npleg.legval(xi, c)
    w = 2.0 / (n * (n - 1) * Pn1 ** 2)
    return xi, w


def gamma_lgl(n: int) -> np.ndarray:
    """Eq. 46: gamma_k = 2/(2k+1) for k < n-1, gamma_{n-1} = 2/(n-1)."""
    g = 2.0 / (2.0 * np.arange(n) + 1.0)
    g[n - 1] = 2.0 / (n - 1)
    return g


def vandermonde(n: int):
    """Eq. 39 / text after Eq. 46: V[j,k] = P_k(xi_j),
    Vinv[k,j] = w_j gamma_k^{-1} P_k(xi_j)."""
    xi, w = lgl_nodes_weights(n)
    P, _ = legendre_table(n, xi)
    V = P.T.copy()
    Vinv = (P / gamma_lgl(n)[:, None]) * w[None, :]
    return V, Vinv


def mass_matrix(n: int) -> np.ndarray:
    """Eq. 50: M_ij = w_i (delta_ij - alpha w_j P_{n-1}(xi_i) P_{n-1}(xi_j)),
    alpha = n(n-1)/(2(2n-1))."""
    xi, w = lgl_nodes_weights(n)
    P, _ = legendre_table(n, xi)
    alpha = n * (n - 1) / (2.0 * (2 * n - 1))
    p = P[n - 1]
    return w[:, None] * (np.eye(n) - alpha * w[None, :] * p[:, None] * p[None, :])


def inverse_mass_matrix(n: int) -> np.ndarray:
    """Eq. 51: Minv_ij = delta_ij / w_i + (n/2) P_{n-1}(xi_i) P_{n-1}(xi_j)."""
    xi, w = lgl_nodes_weights(n)
    P, _ = legendre_table(n, xi)
    p = P[n - 1]
    return np.diag(1.0 / w) + 0.5 * n * p[:, None] * p[None, :]


def lagrange_derivative_matrix(n: int) -> np.ndarray:
    """Eq. 55: D[j,k] = l'_k(xi_j), by differentiating Eq. 4 directly
    (sum over m != k of prod over r != k,m)."""
    xi, _ = lgl_nodes_weights(n)
    D = np.zeros((n, n))
    for j in range(n):
        for k in range(n):
            acc = 0.0
            for m in range(n):
                if m == k:
                    continue
                term = 1.0 / (xi[k] - xi[m])
                for r in range(n):
                    if r == k or r == m:
                        continue
                    term *= (xi[j] - xi[r]) / (xi[k] - xi[r])
                acc += term
            D[j, k] = acc
    return D


def derivative_matrix_eq58(n: int) -> np.ndarray:
    """Eq. 58: D[j,k] = w_k sum_s gamma_s^{-1} P'_s(xi_j) P_s(xi_k)."""
    xi, w = lgl_nodes_weights(n)
    P, dP = legendre_table(n, xi)
    g = gamma_lgl(n)
    return np.einsum("s,sj,sk->jk", 1.0 / g, dP, P) * w[None, :]


def upsilon_eq57(n: int) -> np.ndarray:
    """Eq. 57: Upsilon[j,k] = w_k sum_{s<n} (s + 1/2) P_s(xi_j) P'_s(xi_k).
    This is the oracle's definition of the weak-form internal-flux operator."""
    xi, w = lgl_nodes_weights(n)
    P, dP = legendre_table(n, xi)
    s = np.arange(n) + 0.5
    return np.einsum("s,sj,sk->jk", s, P, dP) * w[None, :]


def upsilon_eq53(n: int) -> np.ndarray:
    """Eq. 53: Upsilon[j,k] = (w_k/w_j) l'_j(xi_k) + (n/2) w_k P_{n-1}(xi_j) P'_{n-1}(xi_k).
    Cross-check only (tests)."""
    xi, w = lgl_nodes_weights(n)
    P, dP = legendre_table(n, xi)
    D = lagrange_derivative_matrix(n)               # D[k, j] = l'_j(xi_k)
    return (w[None, :] / w[:, None]) * D.T + 0.5 * n * w[None, :] * P[n - 1][:, None] * dP[n - 1][None, :]


def xi_lift_eq54(n: int) -> np.ndarray:
    """Eq. 54 (reading C8: 1/w_j): Xi[j, 0] / Xi[j, 1] = first / last column of
    M^{-1}: delta_{j,face}/w_j + (n/2) P_{n-1}(xi_j) P_{n-1}(xi_face)."""
    xi, w = lgl_nodes_weights(n)
    P, _ = legendre_table(n, xi)
    p = P[n - 1]
    Xi = np.zeros((n, 2))
    for col, face in enumerate((0, n - 1)):
        Xi[:, col] = 0.5 * n * p * p[face]
        Xi[face, col] += 1.0 / w[face]
    return Xi


def operators(n: int, mass_mode: int = 0):
    """Return (xi, w, Upsilon[n,n], Xi[n,2]) on the reference element [-1,1].
    mass_mode 0: the paper's exact LGL mass matrix (Eq. 57 + Eq. 54).
    mass_mode 1: lumped (diagonal) mass, reading C1: Upsilon[j,k] = (w_k/w_j) l'_j(xi_k)
    (the first term of Eq. 53) and Xi = delta/w (the first term of Eq. 54)."""
    xi, w = lgl_nodes_weights(n)
    if mass_mode == 0:
        return xi, w, upsilon_eq57(n), xi_lift_eq54(n)
    if mass_mode == 1:
        D = lagrange_derivative_matrix(n)
        ups = (w[None, :] / w[:, None]) * D.T
        Xi = np.zeros((n, 2))
        Xi[0, 0] = 1.0 / w[0]
        Xi[n - 1, 1] = 1.0 / w[n - 1]
        return xi, w, ups, Xi
    raise ValueError("mass_mode must be 0 or 1")
