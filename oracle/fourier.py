"""ORACLE (test infrastructure, not product code) -- DG -> Fourier transform and spectral Poisson.

Plain NumPy/SciPy, fp64, written from PAPER.md Section 5.3 (Eq. 59-71).  Shares no code with
the CUDA path.  Pins: tests/test_oracle_fourier.py (brute-force Gauss-Legendre quadrature of
the Fourier integral of l_j, c_0[1] = 1, single-cosine closed forms for c_p and E, the
O(dx^{n+1/2}) convergence of Fig. 4, C^0 continuity of E; broken_l2: Gauss quadrature of the squared
interpolant and the closed forms ||1||, ||x||).
"""
from __future__ import annotations

import numpy as np
from scipy.special import spherical_jn

from .basis import lgl_nodes_weights, legendre_table, gamma_lgl, mass_matrix


def node_coordinates(lo: float, hi: float, nelem: int, n: int) -> np.ndarray:
    """x_{mj} = xbar_m + xi_j dx/2 (inverse of Eq. 61), flattened [m*n + j]."""
    xi, _ = lgl_nodes_weights(n)
    dx = (hi - lo) / nelem
    xbar = lo + (np.arange(nelem) + 0.5) * dx
    return (xbar[:, None] + 0.5 * dx * xi[None, :]).reshape(-1)


def transform_tensor(lo: float, hi: float, nelem: int, n: int, pmax: int, p_first: int = 0) -> np.ndarray:
    """Eq. 63: T[p, m*n+j] = (dx/L) exp(-i k_p xbar_m) w_j
    sum_{s<n} gamma_s^{-1} (-i)^s P_s(xi_j) j_s(k_p dx/2), p = 0..pmax, k_p = 2 pi p / L.
    (Eq. 64 as printed is wrong, reading C7; Eq. 63 is the definition.)  xbar_m and x_mj are
    absolute coordinates; exp(i k_p x) is L-periodic so any interval [lo, lo+L) serves Eq. 60.
    p_first > 0 returns only the rows p = p_first..pmax (same arithmetic; for tests that walk a large pmax in slices)."""
    xi, w = lgl_nodes_weights(n)
    P, _ = legendre_table(n, xi)
    g = gamma_lgl(n)
    L = hi - lo
    dx = L / nelem
    xbar = lo + (np.arange(nelem) + 0.5) * dx
    T = np.zeros((pmax + 1 - p_first, nelem, n), dtype=np.complex128)
    for p in range(p_first, pmax + 1):
        kp = 2.0 * np.pi * p / L
        z = kp * dx / 2.0
        node = np.zeros(n, dtype=np.complex128)
        for s in range(n):
            node += (1.0 / g[s]) * (-1j) ** s * P[s] * spherical_jn(s, z)
        T[p - p_first] = (dx / L) * np.exp(-1j * kp * xbar)[:, None] * (w * node)[None, :]
    return T.reshape(pmax + 1 - p_first, nelem * n)


def node_coordinates_edges(edges: np.ndarray, n: int) -> np.ndarray:
    """x_{mj} = xbar_m + xi_j (dx)_m / 2 for explicitly given element edges (non-uniform widths), flattened [m*n + j]."""
    xi, _ = lgl_nodes_weights(n)
    e = np.asarray(edges, dtype=np.float64)
    xbar, dx = 0.5 * (e[:-1] + e[1:]), e[1:] - e[:-1]
    return (xbar[:, None] + 0.5 * dx[:, None] * xi[None, :]).reshape(-1)


def transform_tensor_edges(edges: np.ndarray, n: int, pmax: int) -> np.ndarray:
    """Eq. 63 with its per-element width: T[p, m*n+j] = ((dx)_m/L) exp(-i k_p xbar_m) w_j
    sum_{s<n} gamma_s^{-1} (-i)^s P_s(xi_j) j_s(k_p (dx)_m/2), L = edges[-1] - edges[0]."""
    xi, w = lgl_nodes_weights(n)
    P, _ = legendre_table(n, xi)
    g = gamma_lgl(n)
    e = np.asarray(edges, dtype=np.float64)
    nelem = e.size - 1
    L = e[-1] - e[0]
    T = np.zeros((pmax + 1, nelem, n), dtype=np.complex128)
    for p in range(pmax + 1):
        kp = 2.0 * np.pi * p / L
        for m in range(nelem):
            dx, xbar = e[m + 1] - e[m], 0.5 * (e[m] + e[m + 1])
            node = np.zeros(n, dtype=np.complex128)
            for s in range(n):
                node += (1.0 / g[s]) * (-1j) ** s * P[s] * spherical_jn(s, kp * dx / 2.0)
            T[p, m] = (dx / L) * np.exp(-1j * kp * xbar) * w * node
    return T.reshape(pmax + 1, nelem * n)


def fourier_project(T: np.ndarray, rho: np.ndarray) -> np.ndarray:
    """c_p = T_p^{mj} f_mj (text after Eq. 64). rho: [..., G] -> c: [..., pmax+1]."""
    return np.einsum("pg,...g->...p", T, rho)


def poisson_E(lo: float, hi: float, x: np.ndarray, c: np.ndarray) -> np.ndarray:
    """Eq. 71: E_mj = sum_{|p|<=pmax, p != 0} -(c_p/(i k_p)) exp(i k_p x_mj).
    c holds p = 0..pmax; c_{-p} = conj(c_p) because the density is real, so the two-sided sum is
    2 Re of the one-sided one.  p = 0 is dropped (reading C5: the neutralising background)."""
    L = hi - lo
    pmax = c.shape[-1] - 1
    E = np.zeros(c.shape[:-1] + x.shape)
    for p in range(1, pmax + 1):
        kp = 2.0 * np.pi * p / L
        Ep = -c[..., p] / (1j * kp)
        E += 2.0 * np.real(Ep[..., None] * np.exp(1j * kp * x))
    return E


def poisson_phi(lo: float, hi: float, x: np.ndarray, c: np.ndarray) -> np.ndarray:
    """Eq. 70: Phi_mj = sum_{p != 0} -(c_p / k_p^2) exp(i k_p x_mj)."""
    L = hi - lo
    pmax = c.shape[-1] - 1
    Phi = np.zeros(c.shape[:-1] + x.shape)
    for p in range(1, pmax + 1):
        kp = 2.0 * np.pi * p / L
        Phi += 2.0 * np.real((-c[..., p] / kp ** 2)[..., None] * np.exp(1j * kp * x))
    return Phi


def broken_l2(lo: float, hi: float, nelem: int, n: int, u: np.ndarray, v=None, edges=None) -> np.ndarray:
    """Eq. 72: eps = (1/N) sum_m sqrt(int_m (u - v)^2 dx) for nodal vectors u, v [..., N*n]; the
    integrand is the element's degree-(n-1) interpolant (Eq. 69), integrated exactly: d^T M d dx/2 with the LGL mass
    matrix M of Eq. 50.  edges: explicit element edges [nelem+1] for non-uniform widths."""
    d = np.asarray(u, dtype=np.float64) - (0.0 if v is None else np.asarray(v, dtype=np.float64))
    d = d.reshape(d.shape[:-1] + (nelem, n))
    M = mass_matrix(n)
    half = 0.5 * (hi - lo) / nelem if edges is None else 0.5 * np.diff(np.asarray(edges, dtype=np.float64))
    q = np.einsum("...mi,ij,...mj->...m", d, M, d) * half
    return np.sqrt(np.maximum(q, 0.0)).sum(axis=-1) / nelem


def field_energy(lo: float, hi: float, nelem: int, n: int, E: np.ndarray, edges=None) -> np.ndarray:
    """Domain-integrated electric field energy of Fig. 10: W = (1/2) int E(x)^2 dx for nodal vectors
    E [..., N*n], the integrand being each element's degree-(n-1) interpolant (Eq. 69), integrated exactly:
    (1/2) sum_m E_m^T M E_m (dx)_m / 2 with the LGL mass matrix M of Eq. 50."""
    e = np.asarray(E, dtype=np.float64)
    e = e.reshape(e.shape[:-1] + (nelem, n))
    M = mass_matrix(n)
    half = 0.5 * (hi - lo) / nelem if edges is None else 0.5 * np.diff(np.asarray(edges, dtype=np.float64))
    return 0.5 * (np.einsum("...mi,ij,...mj->...m", e, M, e) * half).sum(axis=-1)
