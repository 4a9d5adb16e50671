"""Pins for oracle/vlasov2d2v.py (2D2V): invariants, reductions to the pinned 1D2V oracle, closed forms."""
import numpy as np
import pytest

from oracle import vlasov, vlasov2d2v as v4


def grid4(bc=(0, 0, 0, 0), N=(3, 2, 3, 4), n=(3, 4, 4, 3), omega_c=0.7, mass_mode=0, pmax=(2, 2)):
    return v4.make_grid(N, n, lo=(0.0, -1.0, -3.0, -2.5), hi=(2.0, 2.0, 3.0, 2.5), bc=bc, omega_c=omega_c,
                        pmax=pmax, mass_mode=mass_mode)


def fields(g, seed=1):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(g.flat_shape[:2]), rng.standard_normal(g.flat_shape[:2])


@pytest.mark.parametrize("mode", [0, 1])
def test_constant_state_has_zero_rhs(mode):
    g = grid4(mass_mode=mode)
    Ex, Ey = fields(g)
    r = v4.rhs(g, np.full(g.flat_shape, 1.3), Ex, Ey)
    assert np.max(np.abs(r)) < 1e-10


@pytest.mark.parametrize("mode", [0, 1])
def test_mass_conservation_all_periodic(mode):
    """sum W rhs = 0 (W = tensor LGL weights / Jacobians): the upwind flux is single-valued at every face."""
    g = grid4(mass_mode=mode)
    Ex, Ey = fields(g, 2)
    f = np.random.default_rng(3).random(g.flat_shape)
    r = v4.rhs(g, f, Ex, Ey)
    wx, wy = [np.tile(g.w[d] / g.J[d], g.nelem[d]) for d in (0, 1)]
    total = np.einsum("gh,g,h->", v4.density(g, r), wx, wy)
    scale = np.einsum("gh,g,h->", v4.density(g, np.abs(r)), wx, wy)
    assert abs(total) < 1e-13 * scale


@pytest.mark.parametrize("bc", [(0, 0, 0, 0), (0, 0, 1, 1)])
def test_y_independent_state_reduces_to_1d2v(bc):
    """f(x,u,v) copied along y, E_x = E(x), E_y = 0: the y term vanishes (consistency) and the rest is the 1D2V RHS."""
    g = grid4(bc=bc)
    g3 = vlasov.Grid(nelem=(3, 3, 4), order=(3, 4, 3), lo=(0.0, -3.0, -2.5), hi=(2.0, 3.0, 2.5),
                     bc=(bc[0], bc[2], bc[3]), omega_c=0.7, pmax=2)
    rng = np.random.default_rng(4)
    f3 = rng.random(g3.flat_shape)
    E = rng.standard_normal(g3.flat_shape[0])
    Gy = g.flat_shape[1]
    f = np.repeat(f3[:, None, :, :], Gy, axis=1)
    r = v4.rhs(g, f, np.repeat(E[:, None], Gy, axis=1), None)
    r3 = vlasov.rhs(g3, f3, E)
    assert np.max(np.abs(r - r3[:, None, :, :])) < 1e-12 * np.max(np.abs(r3))


def test_x_independent_state_reduces_to_1d2v_with_swapped_axes():
    """f(y,u,v) copied along x, E_x = 0: with x' = y, u' = v, v' = u the equation is the 1D2V one with omega_c -> -omega_c
    (a_v = -E_y + omega_c u = -E - omega' v', a_u = -omega_c v = omega' u').  Pins the signs of E_y and of both rotation terms."""
    g = grid4(bc=(0, 0, 1, 1))
    g3 = vlasov.Grid(nelem=(2, 4, 3), order=(4, 3, 4), lo=(-1.0, -2.5, -3.0), hi=(2.0, 2.5, 3.0),
                     bc=(0, 1, 1), omega_c=-0.7, pmax=2)
    rng = np.random.default_rng(5)
    f3 = rng.random(g3.flat_shape)                 # [y][v][u]
    E = rng.standard_normal(g3.flat_shape[0])
    Gx = g.flat_shape[0]
    f = np.repeat(np.transpose(f3, (0, 2, 1))[None], Gx, axis=0)          # [x][y][u][v]
    r = v4.rhs(g, f, None, np.repeat(E[None, :], Gx, axis=0))
    r3 = np.transpose(vlasov.rhs(g3, f3, E), (0, 2, 1))
    assert np.max(np.abs(r - r3[None])) < 1e-12 * np.max(np.abs(r3))


def test_rhs_at_matches_array_form():
    g = grid4(bc=(0, 0, 1, 1), mass_mode=0)
    Ex, Ey = fields(g, 6)
    f = np.random.default_rng(7).random(g.flat_shape)
    r = v4.rhs(g, f, Ex, Ey)
    rng = np.random.default_rng(8)
    for _ in range(60):
        node = tuple(int(rng.integers(0, G)) for G in g.flat_shape)
        assert abs(v4.rhs_at(g, f, Ex, Ey, node) - r[node]) < 1e-12 * np.max(np.abs(r))


def test_density_of_separable_state():
    g = grid4()
    x, y, u, v = [c.reshape(-1) for c in g.coords]
    f = (1 + 0.1 * x)[:, None, None, None] * (2 - y)[None, :, None, None] * (u ** 2)[None, None, :, None] * (1 + v)[None, None, None, :]
    rho = v4.density(g, f)
    # int u^2 du over [-3,3] = 18, int (1+v) dv over [-2.5,2.5] = 5 (exact: LGL with n >= 3 integrates degree <= 3)
    assert np.max(np.abs(rho - 90.0 * (1 + 0.1 * x)[:, None] * (2 - y)[None, :])) < 1e-11


@pytest.mark.parametrize("p,q", [(1, 0), (0, 2), (2, -1), (1, 1)])
def test_plane_wave_poisson_closed_form(p, q):
    """rho = 1 + A cos(kx x + ky y + phi)  =>  E = -(A/|k|^2) (kx, ky) sin(kx x + ky y + phi)   (div E = 1 - rho)."""
    N, n = (8, 6), (8, 8)
    g = v4.make_grid(N + (1, 1), n + (2, 2), lo=(0.0, 1.0, -1, -1), hi=(2 * np.pi, 4.0, 1, 1), pmax=(3, 3))
    x, y = g.coords[0].reshape(-1), g.coords[1].reshape(-1)
    kx, ky = 2 * np.pi * p / (2 * np.pi), 2 * np.pi * q / 3.0
    A, ph = 0.05, 0.4
    arg = kx * x[:, None] + ky * y[None, :] + ph
    Ex, Ey = v4.poisson_E(g, v4.fourier_project(g, 1.0 + A * np.cos(arg)))
    k2 = kx * kx + ky * ky
    assert np.max(np.abs(Ex + A * kx / k2 * np.sin(arg))) < 1e-10
    assert np.max(np.abs(Ey + A * ky / k2 * np.sin(arg))) < 1e-10


def test_y_uniform_density_gives_the_1d_field():
    """rho(x) copied along y: c_pq = 0 for q != 0 and E_x is the 1-D solve of oracle/fourier.py, E_y = 0."""
    from oracle import fourier
    g = v4.make_grid((6, 3, 1, 1), (6, 5, 2, 2), lo=(0.0, 0.0, -1, -1), hi=(4.0, 1.5, 1, 1), pmax=(4, 2))
    x = g.coords[0].reshape(-1)
    rho1 = 1 + 0.1 * np.cos(np.pi * x / 2 + 0.3) + 0.02 * np.sin(np.pi * x)
    Ex, Ey = v4.poisson_E(g, v4.fourier_project(g, np.repeat(rho1[:, None], g.flat_shape[1], axis=1)))
    E1 = fourier.poisson_E(0.0, 4.0, x, fourier.fourier_project(g.T, rho1))
    assert np.max(np.abs(Ex - E1[:, None])) < 1e-13
    assert np.max(np.abs(Ey)) < 1e-13


def test_step_conserves_mass():
    g = grid4(bc=(0, 0, 0, 0), N=(2, 2, 2, 2), n=(3, 3, 3, 3))
    f = 0.5 + np.random.default_rng(9).random(g.flat_shape)
    f1 = v4.ssprk3_step(g, f, 1e-3)
    wx, wy = [np.tile(g.w[d] / g.J[d], g.nelem[d]) for d in (0, 1)]
    m0 = np.einsum("gh,g,h->", v4.density(g, f), wx, wy)
    m1 = np.einsum("gh,g,h->", v4.density(g, f1), wx, wy)
    assert abs(m1 - m0) < 1e-13 * m0


def test_free_streaming_exact_solution_and_convergence():
    """omega_c = 0, E = 0, periodic x and y: f(x, y, u, v, t) = f0(x - u t, y - v t, u, v).  The nodal error of a smooth state
    falls by more than a factor 10 when the space elements are halved at order 5 (spectral convergence of the x and y operators and of
    the stepper together; a wrong sign or a swapped speed in the space terms gives an O(1) error)."""
    def run(N):
        g = v4.make_grid((N, N, 1, 1), (5, 5, 3, 3), lo=(0.0, 0.0, -1.0, -1.0), hi=(1.0, 1.0, 1.0, 1.0), bc=(0, 0, 0, 0), omega_c=0.0)
        x, y, u, v = [c.reshape(-1) for c in g.coords]
        def exact(t):
            X = x[:, None, None, None] - u[None, None, :, None] * t
            Y = y[None, :, None, None] - v[None, None, None, :] * t
            return np.ascontiguousarray(np.broadcast_to(1.0 + 0.3 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y), g.flat_shape))
        f, dt, steps = exact(0.0), 2.5e-4, 80
        for _ in range(steps):
            f = v4.ssprk3_step(g, f, dt, self_consistent=False)
        return np.max(np.abs(f - exact(dt * steps)))
    e4, e8 = run(4), run(8)
    assert e4 < 5e-4 and e8 < e4 / 10.0, (e4, e8)          # measured: 1.2e-4, 8.3e-6
