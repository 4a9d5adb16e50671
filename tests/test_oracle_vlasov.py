"""Pins for oracle/vlasov.py and oracle/pointwise.py: invariants, exact solutions, brute force."""
import itertools
import math

import numpy as np
import pytest

from oracle import basis, vlasov, pointwise


def small_grid(bc=(0, 0, 0), n=(4, 4, 4), N=(3, 4, 3), omega_c=0.7, mass_mode=0):
    return vlasov.Grid(nelem=N, order=n, lo=(0.0, -3.0, -2.5), hi=(2.0, 3.0, 2.5), bc=bc,
                       omega_c=omega_c, pmax=2, mass_mode=mass_mode)


@pytest.mark.parametrize("mode", [0, 1])
def test_constant_state_has_zero_rhs(mode):
    g = small_grid(mass_mode=mode)
    rng = np.random.default_rng(0)
    E = rng.standard_normal(g.flat_shape[0])
    r = vlasov.rhs(g, np.full(g.flat_shape, 1.7), E)
    assert np.max(np.abs(r)) < 1e-11


@pytest.mark.parametrize("mode", [0, 1])
def test_polynomial_exactness_interior(mode):
    """f = p(x) q(u) r(v), degrees <= n-1: rhs = -(a_x d_x + a_u d_u + a_v d_v) f exactly on
    elements whose upwind neighbours are interior (the global polynomial is continuous there)."""
    n = 4
    g = vlasov.Grid(nelem=(4, 4, 4), order=(n, n, n), lo=(0.0, -2.0, -2.0), hi=(2.0, 2.0, 2.0),
                    bc=(1, 1, 1), omega_c=0.9, mass_mode=mode)
    x, u, v = [c.reshape(-1) for c in g.coords]
    p = lambda s: 1 + 0.3 * s - 0.2 * s ** 2 + 0.1 * s ** 3
    dp = lambda s: 0.3 - 0.4 * s + 0.3 * s ** 2
    q = lambda s: 0.5 - 0.1 * s + 0.05 * s ** 3
    dq = lambda s: -0.1 + 0.15 * s ** 2
    E = 0.37 * np.ones_like(x)          # constant E keeps a_u polynomial-free in x
    f = p(x)[:, None, None] * q(u)[None, :, None] * p(v)[None, None, :]
    ax = u[None, :, None]
    au = -E[:, None, None] - g.omega_c * v[None, None, :]
    av = g.omega_c * u[None, :, None]
    exact = -(ax * dp(x)[:, None, None] * q(u)[None, :, None] * p(v)[None, None, :]
              + au * p(x)[:, None, None] * dq(u)[None, :, None] * p(v)[None, None, :]
              + av * p(x)[:, None, None] * q(u)[None, :, None] * dp(v)[None, None, :])
    r = vlasov.rhs(g, f, E)
    inner = slice(n, 3 * n)
    assert np.max(np.abs(r[inner, inner, inner] - exact[inner, inner, inner])) < 1e-11


@pytest.mark.parametrize("mode", [0, 1])
def test_mass_conservation_periodic(mode):
    """sum_nodes W rhs = 0 to round-off under all-periodic upwind flux (north_star pin)."""
    g = small_grid(mass_mode=mode)
    rng = np.random.default_rng(1)
    f = rng.random(g.flat_shape)
    E = rng.standard_normal(g.flat_shape[0])
    r = vlasov.rhs(g, f, E)
    W = [np.tile(g.w[d] / g.J[d], g.nelem[d]) for d in range(3)]
    tot = np.einsum("i,j,k,ijk->", W[0], W[1], W[2], r)
    scale = np.einsum("i,j,k,ijk->", W[0], W[1], W[2], np.abs(r))
    assert abs(tot) < 1e-13 * scale
    # density() is the same quadrature: its x-integral is the total mass
    assert abs(np.dot(W[0], vlasov.density(g, f)) - np.einsum("i,j,k,ijk->", W[0], W[1], W[2], f)) < 1e-12


def test_zero_inflow_mass_change_is_boundary_outflow():
    g = small_grid(bc=(0, 1, 1))
    rng = np.random.default_rng(2)
    f = rng.random(g.flat_shape)
    r = vlasov.rhs(g, f, None)
    W = [np.tile(g.w[d] / g.J[d], g.nelem[d]) for d in range(3)]
    dm = np.einsum("i,j,k,ijk->", W[0], W[1], W[2], r)
    u = g.coords[1].reshape(-1); v = g.coords[2].reshape(-1)
    # outflow through u = hi (a_u = -omega_c v > 0 where v < 0), u = lo (a_u < 0 where v > 0), same for v
    au = -g.omega_c * v
    av = g.omega_c * u
    out = 0.0
    out += np.einsum("i,k,ik->", W[0], W[2] * np.maximum(au, 0), f[:, -1, :])
    out += np.einsum("i,k,ik->", W[0], W[2] * np.maximum(-au, 0), f[:, 0, :])
    out += np.einsum("i,j,ij->", W[0], W[1] * np.maximum(av, 0), f[:, :, -1])
    out += np.einsum("i,j,ij->", W[0], W[1] * np.maximum(-av, 0), f[:, :, 0])
    assert abs(dm + out) < 1e-12 * abs(out)


@pytest.mark.parametrize("bc", [(0, 0, 0), (0, 1, 1)])
@pytest.mark.parametrize("mass_mode", [0, 1])
def test_weak_equals_strong_form(bc, mass_mode):
    """Eq. 15: du/dt = -D F + Xi (F - Flux) (vlasov.rhs_strong) must equal the weak form Eq. 14 (vlasov.rhs), with
    the exact-mass operators and with the lumped ones (both satisfy Upsilon + D = Xi_R e_R^T - Xi_L e_L^T)."""
    g = small_grid(bc=bc, mass_mode=mass_mode)
    rng = np.random.default_rng(3)
    f = rng.random(g.flat_shape)
    E = rng.standard_normal(g.flat_shape[0])
    weak = vlasov.rhs(g, f, E)
    strong = vlasov.rhs_strong(g, f, E)
    assert np.max(np.abs(weak - strong)) < 1e-10 * np.max(np.abs(weak))
    # the strong form differentiates: a polynomial of degree n-1 in x (one element wide pieces joined continuously
    # would need a global polynomial; here: f constant => -D F = 0 and all jumps vanish with periodic BCs)
    if bc == (0, 0, 0):
        assert np.max(np.abs(vlasov.rhs_strong(g, np.full(g.flat_shape, 0.7), E))) < 1e-11


def test_full_tensor_brute_force_eq18():
    """Volume term with the full N x N element tensors I (x) I (x) Ups etc. (Eq. 18) on a 2x2x2 grid."""
    n = 3
    g = vlasov.Grid(nelem=(2, 2, 2), order=(n, n, n), lo=(0, -1, -1), hi=(1, 1, 1), bc=(0, 0, 0), omega_c=0.4)
    rng = np.random.default_rng(4)
    f = rng.random(g.flat_shape)
    u = f.reshape(g.shape)
    a = vlasov.speeds(g, None)
    I = np.eye(n)
    full = [np.kron(np.kron(g.ups[0], I), I), np.kron(np.kron(I, g.ups[1]), I), np.kron(np.kron(I, I), g.ups[2])]
    vol = np.zeros(g.shape)
    for e in itertools.product(range(2), repeat=3):
        for d in range(3):
            flux = (a[d] * u)[e[0], :, e[1], :, e[2], :]
            flux = np.broadcast_to(flux, (n, n, n)).reshape(-1)
            vol[e[0], :, e[1], :, e[2], :] += g.J[d] * (full[d] @ flux).reshape(n, n, n)
    ours = sum(g.J[d] * vlasov.basis_product(a[d] * u, g.ups[d], g.sub_element_axis(d)) for d in range(3))
    assert np.allclose(vol, ours, atol=1e-12)


@pytest.mark.parametrize("bc,mode,ndim", [((0, 0, 0), 0, 3), ((0, 1, 1), 0, 3), ((0, 1, 1), 1, 3), ((1, 0, 1), 0, 3),
                                          ((0, 1), 0, 2), ((0, 0), 1, 2)])
def test_pointwise_loops_match_array_form(bc, mode, ndim):
    rng = np.random.default_rng(6)
    if ndim == 3:
        g = vlasov.Grid(nelem=(3, 2, 4), order=(3, 4, 2), lo=(0.0, -1.0, -2.0), hi=(1.5, 1.0, 2.0), bc=bc,
                        omega_c=1.3, mass_mode=mode)
    else:
        g = vlasov.Grid(nelem=(4, 6), order=(4, 3), lo=(0.0, -2.0), hi=(3.0, 2.0), bc=bc, mass_mode=mode)
    f = rng.random(g.flat_shape) - 0.3
    E = rng.standard_normal(g.flat_shape[0])
    r = vlasov.rhs(g, f, E)
    for idx in itertools.product(*[range(s) for s in g.flat_shape]):
        assert abs(pointwise.rhs_at(g, f, E, idx) - r[idx]) < 1e-11 * (1 + abs(r[idx])), idx
    rho = vlasov.density(g, f)
    for gx in range(g.flat_shape[0]):
        assert abs(pointwise.density_at(g, f, gx) - rho[gx]) < 1e-13


def test_upwind_direction_1d():
    """A step advected with a > 0 must take its face value from the LEFT (Eq. 23): in 1D1V with
    E = 0, f = indicator of one x-element, the element to the RIGHT feels it for v > 0 only."""
    g = vlasov.Grid(nelem=(4, 2), order=(3, 3), lo=(0.0, -1.0), hi=(4.0, 1.0), bc=(0, 0))
    f = np.zeros(g.flat_shape)
    f[3:6, :] = 1.0                                   # element 1 in x
    r = vlasov.rhs(g, f, None)
    v = g.coords[1].reshape(-1)
    assert np.all(np.abs(r[6:9][:, v > 0]).max(axis=0) > 0) and np.max(np.abs(r[6:9][:, v < 0])) == 0
    assert np.all(np.abs(r[0:3][:, v < 0]).max(axis=0) > 0) and np.max(np.abs(r[0:3][:, v > 0])) == 0


def test_density_of_maxwellian_and_ring():
    g = vlasov.Grid(nelem=(2, 16, 16), order=(3, 8, 8), lo=(0, -8.5, -8.5), hi=(1, 8.5, 8.5), omega_c=1.0)
    u, v = g.coords[1].reshape(-1), g.coords[2].reshape(-1)
    v2 = u[:, None] ** 2 + v[None, :] ** 2
    maxw = np.exp(-0.5 * v2) / (2 * np.pi)
    ring = (0.5 * v2) ** 3 * np.exp(-0.5 * v2) / (2 * np.pi * 6)     # Eq. 31, j = 3, alpha = 1
    for fv in (maxw, ring):
        rho = vlasov.density(g, np.broadcast_to(fv, g.flat_shape))
        assert np.max(np.abs(rho - 1)) < 1e-9
    assert abs(ring.max() - 27 * math.exp(-3) / (12 * math.pi)) < 1e-3


def test_free_streaming_exact_solution():
    """omega_c = 0, E = 0, periodic x: f(x - v t, v) (north_star pin). Error is discretisation
    limited and must fall fast under h-refinement."""
    errs = []
    for N in (4, 8):
        g = vlasov.Grid(nelem=(N, 2), order=(6, 4), lo=(0.0, -1.0), hi=(2 * np.pi, 1.0), bc=(0, 1))
        x, v = g.coords[0].reshape(-1), g.coords[1].reshape(-1)
        f0 = lambda xx: np.sin(xx)[:, None] * np.exp(-v ** 2)[None, :] + 2.0
        f = f0(x)
        dt, steps = 0.004, 125
        for _ in range(steps):
            f = vlasov.ssprk3_step(g, f, dt, self_consistent=False)
        t = dt * steps
        exact = np.sin(x[:, None] - v[None, :] * t) * np.exp(-v ** 2)[None, :] + 2.0
        errs.append(np.max(np.abs(f - exact)))
    assert errs[0] < 2e-4 and errs[1] < errs[0] / 20, errs


def test_ssprk3_third_order_in_dt():
    g = vlasov.Grid(nelem=(6, 2), order=(8, 3), lo=(0.0, 0.5), hi=(2 * np.pi, 1.0), bc=(0, 1))
    x, v = g.coords[0].reshape(-1), g.coords[1].reshape(-1)
    f0 = np.sin(x)[:, None] * np.ones_like(v)[None, :]
    def run(dt, T=0.4):
        f = f0.copy()
        for _ in range(int(round(T / dt))):
            f = vlasov.ssprk3_step(g, f, dt, self_consistent=False)
        return f
    ref = run(0.000625)
    e1 = np.max(np.abs(run(0.005) - ref)); e2 = np.max(np.abs(run(0.0025) - ref))
    assert 6.5 < e1 / e2 < 9.5, (e1, e2)


def test_cyclotron_rotation_is_counter_clockwise():
    """E = 0, x-uniform: f(u,v,t) = f0(u cos th + v sin th, -u sin th + v cos th), th = omega_c t
    (north_star pin; reading C15: a blob at (2,0) arrives at (0,2) after a quarter turn)."""
    errs = []
    for N in (8, 16):
        g = vlasov.Grid(nelem=(1, N, N), order=(2, 8, 8), lo=(0, -6, -6), hi=(1, 6, 6), bc=(0, 1, 1), omega_c=1.0)
        u, v = g.coords[1].reshape(-1), g.coords[2].reshape(-1)
        blob = lambda uu, vv: np.exp(-((uu - 2.0) ** 2 + vv ** 2) / (2 * 0.6 ** 2))
        f = np.broadcast_to(blob(u[:, None], v[None, :]), g.flat_shape).copy()
        steps = 400 if N == 8 else 800
        dt = (np.pi / 2) / steps
        for _ in range(steps):
            f = vlasov.ssprk3_step(g, f, dt, self_consistent=False)
        th = np.pi / 2
        U, V = u[:, None], v[None, :]
        exact = blob(U * np.cos(th) + V * np.sin(th), -U * np.sin(th) + V * np.cos(th))
        errs.append(np.max(np.abs(f[0] - exact)))
        iu, iv = np.unravel_index(np.argmax(f[0]), f[0].shape)
        assert abs(u[iu]) < 0.4 and abs(v[iv] - 2.0) < 0.4
    assert errs[0] < 5e-3 and errs[1] < errs[0] / 10, errs


@pytest.mark.slow
def test_landau_damping_rate():
    """Config-1 grid, self-consistent E each stage: the k = 0.5 field mode decays at the textbook
    Landau rate -0.1533 (pins the signs of E and of the v-speed together: a wrong sign grows)."""
    g = vlasov.Grid(nelem=(16, 32), order=(4, 4), lo=(0.0, -6.0), hi=(4 * np.pi, 6.0), bc=(0, 1), pmax=16)
    x, v = g.coords[0].reshape(-1), g.coords[1].reshape(-1)
    f = (1 + 0.01 * np.cos(0.5 * x))[:, None] * (np.exp(-0.5 * v ** 2) / np.sqrt(2 * np.pi))[None, :]
    E0 = vlasov.field_E(g, f)
    assert np.max(np.abs(E0 + 0.02 * np.sin(0.5 * x))) < 1e-7
    dt, steps = 0.01, 1500
    amp = []
    for s in range(steps):
        f = vlasov.ssprk3_step(g, f, dt)
        amp.append(np.max(np.abs(vlasov.field_E(g, f))))
    amp = np.array(amp); t = dt * (np.arange(steps) + 1)
    pk = [i for i in range(1, steps - 1) if amp[i] > amp[i - 1] and amp[i] > amp[i + 1]]
    assert len(pk) >= 5
    rate = np.polyfit(t[pk], np.log(amp[pk]), 1)[0]
    assert -0.165 < rate < -0.143, rate
    period = np.mean(np.diff(t[pk]))
    assert abs(period - np.pi / 1.4156) < 0.08          # half period of omega_r = 1.4156
