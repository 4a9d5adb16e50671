"""Pins for oracle/basis.py against what PAPER.md Section 5.2 and the mathematics fix."""
import math

import numpy as np
import pytest
from numpy.polynomial import legendre as npleg

from oracle import basis

ORDERS = [2, 3, 4, 5, 6, 7, 8, 10]


def closed_form_lgl(n):
    """Textbook closed forms of the LGL rule (roots of (1-x^2)P'_{n-1}, Eq. 45), n = 2..7."""
    s = math.sqrt
    if n == 2:
        return [-1, 1], [1, 1]
    if n == 3:
        return [-1, 0, 1], [1 / 3, 4 / 3, 1 / 3]
    if n == 4:
        a = 1 / s(5)
        return [-1, -a, a, 1], [1 / 6, 5 / 6, 5 / 6, 1 / 6]
    if n == 5:
        a = s(3 / 7)
        return [-1, -a, 0, a, 1], [1 / 10, 49 / 90, 32 / 45, 49 / 90, 1 / 10]
    if n == 6:
        a = s(1 / 3 - 2 * s(7) / 21)
        b = s(1 / 3 + 2 * s(7) / 21)
        wa, wb = (14 + s(7)) / 30, (14 - s(7)) / 30
        return [-1, -b, -a, a, b, 1], [1 / 15, wb, wa, wa, wb, 1 / 15]
    if n == 7:
        a = s(5 / 11 - 2 / 11 * s(5 / 3))
        b = s(5 / 11 + 2 / 11 * s(5 / 3))
        wa, wb = (124 + 7 * s(15)) / 350, (124 - 7 * s(15)) / 350
        return [-1, -b, -a, 0, a, b, 1], [1 / 21, wb, wa, 256 / 525, wa, wb, 1 / 21]
    raise ValueError


@pytest.mark.parametrize("n", [2, 3, 4, 5, 6, 7])
def test_lgl_closed_forms(n):
    xi, w = basis.lgl_nodes_weights(n)
    x0, w0 = closed_form_lgl(n)
    assert np.allclose(xi, x0, rtol=0, atol=2e-15)
    assert np.allclose(w, w0, rtol=0, atol=2e-15)


@pytest.mark.parametrize("n", ORDERS)
def test_lgl_defining_equation_and_exactness(n):
    """Eq. 45: (1-xi^2) P'_{n-1}(xi) = 0; the rule integrates degree <= 2n-3 exactly."""
    xi, w = basis.lgl_nodes_weights(n)
    c = np.zeros(n); c[n - 1] = 1
    resid = (1 - xi ** 2) * npleg.legval(xi, npleg.legder(c))
    assert np.max(np.abs(resid)) < 1e-12
    assert abs(w.sum() - 2) < 1e-14
    assert np.allclose(xi, -xi[::-1]) and np.allclose(w, w[::-1])
    for m in range(0, 2 * n - 2):
        exact = 0.0 if m % 2 else 2.0 / (m + 1)
        assert abs(np.dot(w, xi ** m) - exact) < 1e-13, m
    # and NOT exact at degree 2n-2 (so the rule is Lobatto, not Gauss)
    m = 2 * n - 2
    assert abs(np.dot(w, xi ** m) - 2.0 / (m + 1)) > 1e-6 or n > 8


@pytest.mark.parametrize("n", ORDERS)
def test_discrete_orthogonality_eq46(n):
    xi, w = basis.lgl_nodes_weights(n)
    P, _ = basis.legendre_table(n, xi)
    G = np.einsum("s,ks,ls->kl", w, P, P)
    assert np.allclose(G, np.diag(basis.gamma_lgl(n)), atol=1e-14)
    V, Vinv = basis.vandermonde(n)
    assert np.allclose(Vinv @ V, np.eye(n), atol=1e-13)


def _lagrange_values(xi, x):
    n = len(xi)
    L = np.ones((n, len(x)))
    for j in range(n):
        for k in range(n):
            if k != j:
                L[j] *= (x - xi[k]) / (xi[j] - xi[k])
    return L


@pytest.mark.parametrize("n", ORDERS)
def test_mass_matrix_brute_force(n):
    """Eq. 50 / 51 against M_ij = int l_i l_j by (n+2)-point Gauss-Legendre quadrature."""
    xi, w = basis.lgl_nodes_weights(n)
    xg, wg = npleg.leggauss(n + 2)
    L = _lagrange_values(xi, xg)
    M = np.einsum("q,iq,jq->ij", wg, L, L)
    assert np.allclose(basis.mass_matrix(n), M, atol=1e-14)
    assert np.allclose(basis.inverse_mass_matrix(n), np.linalg.inv(M), rtol=1e-11, atol=1e-11)


@pytest.mark.parametrize("n", ORDERS)
def test_upsilon_three_ways(n):
    """Eq. 57 == Eq. 53 == M^{-1} A^T with A_ij = <l_i | l_j'> by quadrature (Eq. 13, 52)."""
    xi, w = basis.lgl_nodes_weights(n)
    xg, wg = npleg.leggauss(n + 2)
    L = _lagrange_values(xi, xg)
    # derivative of Lagrange polynomials at Gauss points via the Legendre-series route
    dL = np.zeros_like(L)
    for j in range(n):
        e = np.zeros(n); e[j] = 1
        coef = npleg.legfit(xi, e, n - 1)
        dL[j] = npleg.legval(xg, npleg.legder(coef))
    M = np.einsum("q,iq,jq->ij", wg, L, L)
    # weak form: du_b/dt M_{b g} = F_b <l_b | d l_g>  =>  Ups[g, b] = sum_e Minv[g, e] <l_b | d l_e>
    Adv = np.einsum("q,bq,eq->be", wg, L, dL)           # <l_b | l_e'>
    ups_bf = np.linalg.solve(M, Adv.T)
    u57, u53 = basis.upsilon_eq57(n), basis.upsilon_eq53(n)
    assert np.allclose(u57, u53, atol=2e-12)
    assert np.allclose(u57, ups_bf, atol=2e-11)


@pytest.mark.parametrize("n", ORDERS)
def test_derivative_matrix(n):
    """Eq. 55 == Eq. 58; exact on monomials of degree <= n-1 (north_star pin)."""
    xi, _ = basis.lgl_nodes_weights(n)
    D = basis.lagrange_derivative_matrix(n)
    assert np.allclose(D, basis.derivative_matrix_eq58(n), atol=2e-12)
    for m in range(n):
        d_exact = m * xi ** (m - 1) if m > 0 else np.zeros(n)
        assert np.allclose(D @ xi ** m, d_exact, atol=1e-12)
    # identity Eq. 56: sum_s P_{n-1}(xi_s) l_s'(xi_j) = P'_{n-1}(xi_j)
    P, dP = basis.legendre_table(n, xi)
    assert np.allclose(D @ P[n - 1], dP[n - 1], atol=1e-11)


@pytest.mark.parametrize("n", ORDERS)
@pytest.mark.parametrize("mode", [0, 1])
def test_operator_invariants(n, mode):
    """Orientation pins (reading C11): w^T Ups = 0, Ups 1 = Xi_R - Xi_L, w^T Xi = (1,1),
    Ups + D = Xi_R e_R^T - Xi_L e_L^T (weak == strong form), centro-antisymmetry."""
    xi, w, ups, lift = basis.operators(n, mode)
    D = basis.lagrange_derivative_matrix(n)
    assert np.max(np.abs(w @ ups)) < 1e-12
    assert np.allclose(ups @ np.ones(n), lift[:, 1] - lift[:, 0], atol=1e-12)
    assert np.allclose(w @ lift, [1, 1], atol=1e-13)
    B = np.zeros((n, n)); B[:, n - 1] = lift[:, 1]; B[:, 0] = -lift[:, 0]
    assert np.allclose(ups + D, B, atol=1e-11)
    assert np.allclose(ups[::-1, ::-1], -ups, atol=1e-12)
    assert np.allclose(lift[::-1, ::-1], lift, atol=1e-13)


def test_xi_is_columns_of_inverse_mass():
    for n in ORDERS:
        Minv = basis.inverse_mass_matrix(n)
        assert np.allclose(basis.xi_lift_eq54(n), Minv[:, [0, n - 1]], atol=1e-13)


def test_worked_example_n4():
    """tests/golden/operators_n4.txt: n = 4 entries in closed form (derived by hand from Eq. 54/57
    with xi = +-1/sqrt5, w = 5/6, 1/6): Ups row 0 = (-5, -(5+5sqrt5)/4... ) -- see the fixture."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "operators_n4.txt")
    rows = [list(map(float, l.split())) for l in open(path) if l.strip() and not l.startswith("#")]
    ups_g, lift_g = np.array(rows[:4]), np.array(rows[4:8])
    assert np.allclose(basis.upsilon_eq57(4), ups_g, atol=1e-13)
    assert np.allclose(basis.xi_lift_eq54(4), lift_g, atol=1e-13)
