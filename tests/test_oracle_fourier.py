"""Pins for oracle/fourier.py against what PAPER.md Section 5.3 and the mathematics fix."""
import numpy as np
import pytest
from numpy.polynomial import legendre as npleg

from oracle import basis, fourier


def _lagrange_values(xi, x):
    n = len(xi)
    L = np.ones((n, len(x)))
    for j in range(n):
        for k in range(n):
            if k != j:
                L[j] *= (x - xi[k]) / (xi[j] - xi[k])
    return L


@pytest.mark.parametrize("n,N,pmax,lo,hi", [(4, 16, 16, 0.0, 4 * np.pi), (8, 8, 24, 0.0, 20 * np.pi),
                                            (6, 5, 12, -1.0, 2.5), (10, 4, 10, 0.0, 1.0)])
def test_transform_tensor_brute_force(n, N, pmax, lo, hi):
    """Eq. 63 against c_p = (1/L) int f e^{-ikx} dx (Eq. 60) with f = l_j on element m, the
    integral done by 80-point Gauss-Legendre quadrature."""
    T = fourier.transform_tensor(lo, hi, N, n, pmax).reshape(pmax + 1, N, n)
    xi, _ = basis.lgl_nodes_weights(n)
    xg, wg = npleg.leggauss(80)
    Lg = _lagrange_values(xi, xg)
    L = hi - lo
    dx = L / N
    for p in range(pmax + 1):
        kp = 2 * np.pi * p / L
        for m in (0, N // 2, N - 1):
            xbar = lo + (m + 0.5) * dx
            integ = (Lg * (wg * np.exp(-1j * kp * (xbar + 0.5 * dx * xg)))[None, :]).sum(axis=1) * (0.5 * dx / L)
            assert np.allclose(T[p, m], integ, atol=5e-16, rtol=1e-13), (p, m)


def test_spherical_bessel_identity_eq62():
    """Eq. 62: int P_s(xi) e^{-i z xi} dxi = 2 (-i)^s j_s(z), by quadrature."""
    from scipy.special import spherical_jn
    xg, wg = npleg.leggauss(60)
    for z in (0.0, 1e-3, 0.7, 3.0, 12.5):
        for s in range(10):
            c = np.zeros(s + 1); c[s] = 1
            lhs = np.sum(wg * npleg.legval(xg, c) * np.exp(-1j * z * xg))
            assert abs(lhs - 2 * (-1j) ** s * spherical_jn(s, z)) < 5e-14


def test_mean_mode_and_single_cosine():
    """c_0 of f == 1 is 1 (reading C7); rho = 1 + A cos(kx + phi) gives c_m = (A/2) e^{i phi}
    and E = -(A/k) sin(kx + phi)  (Eq. 68-71 with E = -Phi')."""
    lo, hi, N, n = 0.0, 20 * np.pi, 32, 8
    x = fourier.node_coordinates(lo, hi, N, n)
    T = fourier.transform_tensor(lo, hi, N, n, 16)
    c = fourier.fourier_project(T, np.ones_like(x))
    assert abs(c[0] - 1) < 1e-14 and np.max(np.abs(c[1:])) < 1e-14
    A, phi = 0.01, 0.3
    for m in (1, 3, 5):
        k = 2 * np.pi * m / (hi - lo)
        rho = 1 + A * np.cos(k * x + phi)
        c = fourier.fourier_project(T, rho)
        assert abs(c[m] - 0.5 * A * np.exp(1j * phi)) < 1e-13 * 1 + 2e-15
        E = fourier.poisson_E(lo, hi, x, c)
        Eex = -(A / k) * np.sin(k * x + phi)
        assert np.max(np.abs(E - Eex)) / np.max(np.abs(Eex)) < 1e-11, m


def test_config1_grid_accuracy():
    """n = 4, N = 16 (config 1): closed-form E only to ~1e-6 (discretisation)."""
    lo, hi, N, n = 0.0, 4 * np.pi, 16, 4
    x = fourier.node_coordinates(lo, hi, N, n)
    T = fourier.transform_tensor(lo, hi, N, n, 16)
    rho = 1 + 0.01 * np.cos(0.5 * x)
    E = fourier.poisson_E(lo, hi, x, fourier.fourier_project(T, rho))
    Eex = -0.02 * np.sin(0.5 * x)
    err = np.max(np.abs(E - Eex)) / 0.02
    assert 1e-10 < err < 2e-6


def test_E_is_continuous_and_derivative_matches_source():
    """The Fourier series is single valued: E agrees at duplicated interface nodes."""
    lo, hi, N, n = 0.0, 2 * np.pi, 10, 8
    rng = np.random.default_rng(5)
    x = fourier.node_coordinates(lo, hi, N, n)
    rho = np.sin(x) + rng.standard_normal(x.size)
    T = fourier.transform_tensor(lo, hi, N, n, 10)
    E = fourier.poisson_E(lo, hi, x, fourier.fourier_project(T, rho)).reshape(N, n)
    assert np.allclose(E[:-1, -1], E[1:, 0], atol=1e-13)
    assert abs(E[-1, -1] - E[0, 0]) < 1e-13


def _broken_l2(err_fn, lo, hi, N):
    """Eq. 72: (1/N) sum_m sqrt(int_m err^2) by 20-point Gauss quadrature per element."""
    xg, wg = npleg.leggauss(20)
    dx = (hi - lo) / N
    tot = 0.0
    for m in range(N):
        xm = lo + (m + 0.5) * dx + 0.5 * dx * xg
        tot += np.sqrt(np.sum(wg * err_fn(xm, m) ** 2) * 0.5 * dx)
    return tot / N


@pytest.mark.parametrize("n", [3, 4, 5, 6])
def test_poisson_convergence_fig4(n):
    """Fig. 4: Phi'' = sin(2 pi x) on [0,1], N = 10..25: error O(dx^{n+1/2}) in the
    broken l2 norm of Eq. 72 (Phi interpolated on the element basis, Eq. 69)."""
    lo, hi = 0.0, 1.0
    errs, Ns = [], [10, 15, 20, 25]
    xi, _ = basis.lgl_nodes_weights(n)
    for N in Ns:
        x = fourier.node_coordinates(lo, hi, N, n)
        T = fourier.transform_tensor(lo, hi, N, n, N)
        c = fourier.fourier_project(T, np.sin(2 * np.pi * x))
        Phi = fourier.poisson_phi(lo, hi, x, c).reshape(N, n)
        dx = 1.0 / N

        def err(xm, m):
            loc = (xm - (lo + (m + 0.5) * dx)) / (0.5 * dx)
            return _lagrange_values(xi, loc).T @ Phi[m] + np.sin(2 * np.pi * xm) / (4 * np.pi ** 2)
        errs.append(_broken_l2(err, lo, hi, N))
    slope = np.polyfit(np.log(1.0 / np.array(Ns)), np.log(errs), 1)[0]
    assert n - 0.2 < slope < n + 1.6, (slope, errs)


@pytest.mark.parametrize("n,N", [(2, 3), (3, 7), (4, 10), (7, 5), (8, 16), (10, 4)])
def test_broken_l2_against_gauss_quadrature_and_closed_forms(n, N):
    """fourier.broken_l2 (Eq. 72 with the exact LGL mass matrix, Eq. 50) against 20-point Gauss quadrature of the squared
    interpolant per element (exact: degree 2n-2 <= 18), and closed forms: ||1|| = sqrt(dx); ||x|| on [0, L]."""
    lo, hi = -0.5, 2.0
    dx = (hi - lo) / N
    xi, _ = basis.lgl_nodes_weights(n)
    rng = np.random.default_rng(100 * n + N)
    u, v = rng.standard_normal((3, N * n)), rng.standard_normal((3, N * n))
    xg, wg = npleg.leggauss(20)
    Lg = _lagrange_values(xi, xg)                                   # [n][20]
    d = (u - v).reshape(3, N, n)
    ref = np.sqrt(np.einsum("g,bmg->bm", wg, np.einsum("bmj,jg->bmg", d, Lg) ** 2) * 0.5 * dx).sum(axis=1) / N
    assert np.allclose(fourier.broken_l2(lo, hi, N, n, u, v), ref, rtol=1e-13, atol=0)
    assert np.allclose(fourier.broken_l2(lo, hi, N, n, u), fourier.broken_l2(lo, hi, N, n, u, np.zeros_like(u)), rtol=0, atol=0)
    assert abs(fourier.broken_l2(lo, hi, N, n, np.ones(N * n)) - np.sqrt(dx)) < 1e-14
    x = fourier.node_coordinates(lo, hi, N, n)
    edges = lo + dx * np.arange(N + 1)
    exact = np.sqrt((edges[1:] ** 3 - edges[:-1] ** 3) / 3.0).sum() / N      # int x^2 over each element
    assert abs(fourier.broken_l2(lo, hi, N, n, x) - exact) < 1e-13


def test_nonuniform_transform_brute_force_and_reduction_to_uniform():
    """transform_tensor_edges (Eq. 63 with (dx)_m) against 80-point Gauss quadrature of the Fourier integral of l_j on each
    element, c_0[1] = 1, and equality with transform_tensor when the edges are equally spaced."""
    n, pmax = 6, 14
    edges = np.array([-1.0, -0.4, -0.25, 0.3, 0.35, 1.1, 1.5])
    N = edges.size - 1
    T = fourier.transform_tensor_edges(edges, n, pmax).reshape(pmax + 1, N, n)
    xi, _ = basis.lgl_nodes_weights(n)
    xg, wg = npleg.leggauss(80)
    Lg = _lagrange_values(xi, xg)
    L = edges[-1] - edges[0]
    for p in range(pmax + 1):
        kp = 2 * np.pi * p / L
        for m in range(N):
            dx, xbar = edges[m + 1] - edges[m], 0.5 * (edges[m] + edges[m + 1])
            integ = (Lg * (wg * np.exp(-1j * kp * (xbar + 0.5 * dx * xg)))[None, :]).sum(axis=1) * (0.5 * dx / L)
            assert np.allclose(T[p, m], integ, atol=5e-16, rtol=1e-13), (p, m)
    assert abs(fourier.fourier_project(T.reshape(pmax + 1, -1), np.ones(N * n))[0] - 1.0) < 1e-14
    eq = np.linspace(0.5, 3.0, 9)
    assert np.allclose(fourier.transform_tensor_edges(eq, 5, 9), fourier.transform_tensor(0.5, 3.0, 8, 5, 9), atol=1e-16, rtol=1e-13)
    assert np.allclose(fourier.node_coordinates_edges(eq, 5), fourier.node_coordinates(0.5, 3.0, 8, 5), atol=1e-15)


def test_nonuniform_poisson_single_cosine_closed_form():
    """E = -(A/k) sin(kx + ph), Phi = -(A/k^2) cos(kx + ph) on a graded grid (widths varying 4x), n = 8."""
    n, N = 8, 24
    w = 1.0 + 0.6 * np.sin(np.arange(N) * 0.7)
    edges = np.concatenate([[0.0], np.cumsum(w)]) * (2 * np.pi / w.sum())
    x = fourier.node_coordinates_edges(edges, n)
    A, m, ph = 0.03, 3, 0.8
    c = fourier.fourier_project(fourier.transform_tensor_edges(edges, n, 12), 1 + A * np.cos(m * x + ph))
    assert abs(c[m] - 0.5 * A * np.exp(1j * ph)) < 1e-12 and abs(c[0] - 1) < 1e-13
    E = fourier.poisson_E(edges[0], edges[-1], x, c)
    assert np.max(np.abs(E + (A / m) * np.sin(m * x + ph))) < 1e-10 * A / m
    assert abs(fourier.broken_l2(0, 0, N, n, np.ones(N * n), edges=edges) - np.sqrt(np.diff(edges)).sum() / N) < 1e-14


@pytest.mark.parametrize("n,N", [(2, 5), (4, 3), (8, 4), (10, 2)])
def test_field_energy_against_exact_polynomial_integrals(n, N):
    """fourier.field_energy (Fig. 10; mass matrix of Eq. 50) against integrals that need no mass matrix: E = x on
    [0, 1] gives 1/6 for every order; a random polynomial of degree n - 1 per element, integrated by numpy's polynomial
    antiderivative of E^2, on equal and on unequal elements; E = P_{n-1} per element (closed form; a lumped quadrature
    sum_j w_j E_j^2 fails it)."""
    x01 = fourier.node_coordinates(0.0, 1.0, N, n)
    assert abs(fourier.field_energy(0.0, 1.0, N, n, x01) - 1.0 / 6.0) < 1e-14
    rng = np.random.default_rng(n * 100 + N)
    for edges in (None, np.concatenate(([-1.0], -1.0 + np.cumsum(rng.uniform(0.3, 1.2, N))))):
        lo, hi = (-1.0, 2.5) if edges is None else (edges[0], edges[-1])
        ed = np.linspace(lo, hi, N + 1) if edges is None else edges
        x = fourier.node_coordinates(lo, hi, N, n) if edges is None else fourier.node_coordinates_edges(edges, n)
        E = np.empty(N * n); exact = 0.0
        for m in range(N):
            poly = np.polynomial.Polynomial(rng.uniform(-1, 1, n))
            E[m * n:(m + 1) * n] = poly(x[m * n:(m + 1) * n])
            F = (poly * poly).integ()
            exact += 0.5 * (F(ed[m + 1]) - F(ed[m]))
        assert abs(fourier.field_energy(lo, hi, N, n, E, edges=edges) - exact) < 1e-13 * abs(exact)
        # E = P_{n-1}(xi) in every element: int P_{n-1}^2 dxi = 2/(2n-1), so W = L / (2 (2n-1)); the lumped LGL rule gives
        # 2/(n-1) instead -- the term the exact mass matrix of Eq. 50 corrects
        xi = basis.lgl_nodes_weights(n)[0]
        Pn1 = np.tile(npleg.legval(xi, [0.0] * (n - 1) + [1.0]), N)
        assert abs(fourier.field_energy(lo, hi, N, n, Pn1, edges=edges) - (hi - lo) / (2.0 * (2 * n - 1))) < 1e-13 * (hi - lo)
