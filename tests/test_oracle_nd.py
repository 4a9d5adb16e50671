"""Pins of oracle/vlasov_nd.py (the d_x + d_v dimensional oracle): what the mathematics fixes, and the already pinned 1D2V and
2D2V oracles on their own shapes and as limits of the higher-dimensional ones."""
import math

import numpy as np
import pytest

from oracle import vlasov as ov
from oracle import vlasov2d2v as o4
from oracle import vlasov_nd as on
import workloads as wl


def relerr(a, b):
    return float(np.max(np.abs(np.asarray(a) - np.asarray(b))) / max(np.max(np.abs(b)), 1e-300))


def rnd(shape, seed):
    return wl.counter_uniform_chunked(seed, int(np.prod(shape))).reshape(shape)


def test_constant_state_has_zero_rhs_and_mass_is_conserved_3d3v():
    g = on.make_grid(3, 3, (2, 2, 2, 2, 2, 2), (3, 2, 3, 2, 3, 2), (0, 0, 0, -1, -1.5, -2), (1, 2, 1.5, 1, 1.5, 2), bc=(0,) * 6, omega_c=0.7)
    E = [0.3 * rnd(g.flat_shape[:3], 5 + i) - 0.15 for i in range(3)]
    assert np.max(np.abs(on.rhs(g, np.ones(g.flat_shape), E))) < 1e-11
    f = rnd(g.flat_shape, 11)
    r = on.rhs(g, f, E).reshape(g.shape)
    W = 1.0
    for d in range(6):
        shp = [1] * 12; shp[2 * d + 1] = g.order[d]
        W = W * (g.w[d] / g.J[d]).reshape(shp)
    assert abs(np.sum(W * r)) < 1e-11 * np.sum(np.abs(W * r))


def test_matches_the_1d2v_oracle_on_its_own_shape():
    nelem, order, lo, hi = (3, 2, 3), (4, 3, 5), (0.0, -2.0, -2.5), (2.0, 2.0, 2.5)
    g3 = ov.Grid(nelem=nelem, order=order, lo=lo, hi=hi, bc=(0, 1, 0), omega_c=0.8, pmax=3)
    gn = on.make_grid(1, 2, nelem, order, lo, hi, bc=(0, 1, 0), omega_c=0.8, pmax=(3,))
    f = rnd(g3.flat_shape, 3)
    E = 0.4 * rnd((g3.flat_shape[0],), 4) - 0.2
    assert relerr(on.rhs(gn, f, [E]), ov.rhs(g3, f, E)) < 1e-14
    assert relerr(on.density(gn, f), ov.density(g3, f)) < 1e-14
    assert relerr(on.field_E(gn, f)[0], ov.field_E(g3, f)) < 1e-13
    assert relerr(on.ssprk3_step(gn, f, 1e-3), ov.ssprk3_step(g3, f, 1e-3)) < 1e-13


def test_matches_the_1d1v_oracle():
    nelem, order, lo, hi = (4, 5), (4, 3), (0.0, -3.0), (4 * math.pi, 3.0)
    g2 = ov.Grid(nelem=nelem, order=order, lo=lo, hi=hi, bc=(0, 1), pmax=4)
    gn = on.make_grid(1, 1, nelem, order, lo, hi, bc=(0, 1), pmax=(4,))
    f = rnd(g2.flat_shape, 8)
    assert relerr(on.ssprk3_step(gn, f, 2e-3), ov.ssprk3_step(g2, f, 2e-3)) < 1e-13


def test_matches_the_2d2v_oracle_on_its_own_shape():
    nelem, order, lo, hi = (2, 3, 2, 2), (3, 2, 4, 3), (0.0, -1.0, -2.0, -2.5), (2.0, 2.0, 2.0, 2.5)
    g4 = o4.make_grid(nelem, order, lo, hi, bc=(0, 0, 1, 1), omega_c=0.6, pmax=(2, 3))
    gn = on.make_grid(2, 2, nelem, order, lo, hi, bc=(0, 0, 1, 1), omega_c=0.6, pmax=(2, 3))
    f = rnd(g4.flat_shape, 21)
    Ex, Ey = 0.4 * rnd(g4.flat_shape[:2], 22) - 0.2, 0.4 * rnd(g4.flat_shape[:2], 23) - 0.2
    assert relerr(on.rhs(gn, f, [Ex, Ey]), o4.rhs(g4, f, Ex, Ey)) < 1e-14
    rho = on.density(gn, f)
    assert relerr(rho, o4.density(g4, f)) < 1e-14
    assert relerr(on.fourier_project(gn, rho), o4.fourier_project(g4, rho)) < 1e-13
    En, E4 = on.field_E(gn, f), o4.field_E(g4, f)
    assert relerr(En[0], E4[0]) < 1e-12 and relerr(En[1], E4[1]) < 1e-12
    assert relerr(on.ssprk3_step(gn, f, 1e-3), o4.ssprk3_step(g4, f, 1e-3)) < 1e-13


def test_3d3v_state_independent_of_z_and_separable_in_w_reduces_to_2d2v():
    """f(x, y, u, v) g(w), uniform in z: a_z d_z f = 0, E_z = 0, so the 3D3V RHS is the 2D2V RHS times g(w); the density is the
    2D2V density times the quadrature of g, repeated along z."""
    N4, n4 = (2, 2, 2, 2), (3, 3, 3, 2)
    lo4, hi4 = (0.0, 0.0, -2.0, -2.0), (2.0, 3.0, 2.0, 2.0)
    g4 = o4.make_grid(N4, n4, lo4, hi4, bc=(0, 0, 1, 1), omega_c=0.9, pmax=(2, 2))
    nelem = (2, 2, 2, 2, 2, 3); order = (3, 3, 2, 3, 2, 4)
    lo = (0.0, 0.0, 0.0, -2.0, -2.0, -1.5); hi = (2.0, 3.0, 1.0, 2.0, 2.0, 1.5)
    g6 = on.make_grid(3, 3, nelem, order, lo, hi, bc=(0, 0, 0, 1, 1, 1), omega_c=0.9, pmax=(2, 2, 1))
    f4 = rnd(g4.flat_shape, 31)
    w = g6.coords[5].reshape(-1)
    gw = np.exp(-w * w)
    f6 = f4[:, :, None, :, :, None] * gw[None, None, None, None, None, :] * np.ones((1, 1, g6.flat_shape[2], 1, 1, 1))
    Ex, Ey = 0.3 * rnd(g4.flat_shape[:2], 32) - 0.15, 0.3 * rnd(g4.flat_shape[:2], 33) - 0.15
    ones_z = np.ones((1, 1, g6.flat_shape[2]))
    E6 = [Ex[:, :, None] * ones_z, Ey[:, :, None] * ones_z, None]
    r6 = on.rhs(g6, f6, E6)
    ref = o4.rhs(g4, f4, Ex, Ey)[:, :, None, :, :, None] * gw[None, None, None, None, None, :] * np.ones((1, 1, g6.flat_shape[2], 1, 1, 1))
    assert relerr(r6, ref) < 1e-13
    qw = float(np.sum(np.tile(g6.w[5] / g6.J[5], g6.nelem[5]) * gw))
    assert relerr(on.density(g6, f6), o4.density(g4, f4)[:, :, None] * qw * ones_z) < 1e-13
    # the self-consistent field of the z-uniform density: the 2D2V field, and no z component
    E = on.field_E(g6, f6)
    E4 = o4.field_E(g4, f4)
    assert relerr(E[0], E4[0][:, :, None] * qw * ones_z) < 1e-12 and relerr(E[1], E4[1][:, :, None] * qw * ones_z) < 1e-12
    assert np.max(np.abs(E[2])) < 1e-13 * np.max(np.abs(E[0]))


def test_1d3v_with_w_dependence_reduces_to_1d2v():
    """1D3V: a_w = 0 (no E_z, B along z): f(x, u, v) g(w) evolves as the 1D2V state times g."""
    nelem3, order3, lo3, hi3 = (3, 2, 2), (3, 4, 3), (0.0, -2.0, -2.0), (3.0, 2.0, 2.0)
    g3 = ov.Grid(nelem=nelem3, order=order3, lo=lo3, hi=hi3, bc=(0, 1, 1), omega_c=1.1, pmax=3)
    gn = on.make_grid(1, 3, nelem3 + (2,), order3 + (3,), lo3 + (-1.0,), hi3 + (1.0,), bc=(0, 1, 1, 1), omega_c=1.1, pmax=(3,))
    f3 = rnd(g3.flat_shape, 41)
    w = gn.coords[3].reshape(-1)
    gw = 1.0 + 0.3 * w
    f = f3[..., None] * gw
    qw = float(np.sum(np.tile(gn.w[3] / gn.J[3], gn.nelem[3]) * gw))
    # one self-consistent step: the field of the 1D3V state is qw times that of f3, i.e. that of the 1D2V state qw f3 / qw ...
    E3 = ov.field_E(g3, f3 * qw)
    assert relerr(on.field_E(gn, f)[0], E3) < 1e-12
    assert relerr(on.rhs(gn, f, [E3]), ov.rhs(g3, f3, E3)[..., None] * gw) < 1e-13


@pytest.mark.parametrize("p", [(1, 0, 0), (0, 2, 0), (0, 0, 1), (1, -1, 1), (2, 1, -1)])
def test_plane_wave_field_closed_form_3d(p):
    """rho = 1 + A cos(k.x + phi)  =>  E = -(A / |k|^2) k sin(k.x + phi)  (Eq. 68/71 with E = -grad Phi, d_x E = 1 - rho)."""
    N, n = (5, 4, 3), (6, 6, 6)
    lo, hi = (0.0, -1.0, 0.5), (2.0, 2.0, 2.0)
    g = on.make_grid(3, 3, N + (1, 1, 1), n + (2, 2, 2), lo + (-1, -1, -1), hi + (1, 1, 1), bc=(0,) * 6, pmax=(3, 3, 3))
    xs = [g.coords[i].reshape(-1) for i in range(3)]
    k = [2 * math.pi * p[i] / (hi[i] - lo[i]) for i in range(3)]
    A, ph = 0.05, 0.3
    arg = k[0] * xs[0][:, None, None] + k[1] * xs[1][None, :, None] + k[2] * xs[2][None, None, :] + ph
    rho = 1.0 + A * np.cos(arg)
    E = on.poisson_E(g, on.fourier_project(g, rho))
    k2 = sum(ki * ki for ki in k)
    for i in range(3):
        exact = -(A / k2) * k[i] * np.sin(arg)
        # discretisation error of the n = 6 projection at 2-5 elements per wavelength; a wrong sign or factor is O(1)
        assert np.max(np.abs(E[i] - exact)) < 1e-4 * A / math.sqrt(k2), (i, np.max(np.abs(E[i] - exact)))


# ---------------------------------------------------------------------------------------------
# the third force component, a_{v_3} = -E_3 (Eq. 28 carried to three space dimensions; "n-dimensions",
# PAPER.md:43).  Both pins below fail when the sign of E in the i >= 2 branch of `speeds` is flipped.
# ---------------------------------------------------------------------------------------------
def test_3d3v_unmagnetised_rhs_commutes_with_swapping_the_first_and_third_pair():
    """Without B the Vlasov equation does not know which (x_i, v_i) pair is which: relabelling (x_1, v_1) <-> (x_3, v_3) of the
    state and of the field must relabel the RHS.  The first component is pinned (1D2V / 2D2V oracles), so this carries its sign
    and its field indexing over to the third."""
    pair = dict(nelem=(2, 3, 2), order=(3, 2, 3), lo=(0.0, -1.0, 0.0), hi=(1.5, 2.0, 1.5))       # dims 0 and 2 alike
    vel = dict(nelem=(2, 2, 2), order=(3, 4, 3), lo=(-2.0, -1.5, -2.0), hi=(2.0, 2.5, 2.0))      # dims 3 and 5 alike
    g = on.make_grid(3, 3, pair["nelem"] + vel["nelem"], pair["order"] + vel["order"], pair["lo"] + vel["lo"], pair["hi"] + vel["hi"],
                     bc=(0, 0, 0, 1, 0, 1), omega_c=0.0, pmax=(1, 1, 1))
    f = rnd(g.flat_shape, 51)
    E = [0.6 * rnd(g.flat_shape[:3], 52 + i) - 0.3 for i in range(3)]
    swap6 = lambda a: np.ascontiguousarray(np.transpose(a, (2, 1, 0, 5, 4, 3)))
    swap3 = lambda a: np.ascontiguousarray(np.transpose(a, (2, 1, 0)))
    lhs = on.rhs(g, swap6(f), [swap3(E[2]), swap3(E[1]), swap3(E[0])])
    assert relerr(lhs, swap6(on.rhs(g, f, E))) < 1e-13
    # and the relabelled problem really exercises E_3: dropping it changes the answer at O(1)
    assert relerr(on.rhs(g, f, [E[0], E[1], None]), on.rhs(g, f, E)) > 1e-2


def test_3d3v_z_only_problem_reduces_to_the_1d1v_oracle():
    """f = h(z, w) a(u) b(v), uniform in x and y, E = (0, 0, E_3(z)), no B: every term but the (z, w) pair vanishes (zero speed
    in u and v, no gradient in x and y) and the 3D3V RHS is the pinned 1D1V RHS of h on (z, w), times a(u) b(v)."""
    Nz, nz, Nw, nw = 4, 4, 5, 3
    loz, hiz, low, hiw = 0.0, 4 * math.pi, -3.0, 3.5
    g2 = ov.Grid(nelem=(Nz, Nw), order=(nz, nw), lo=(loz, low), hi=(hiz, hiw), bc=(0, 1), pmax=3)
    g6 = on.make_grid(3, 3, (1, 2, Nz, 2, 1, Nw), (2, 2, nz, 3, 2, nw), (0.0, 0.0, loz, -1.0, -2.0, low), (1.0, 2.0, hiz, 1.0, 2.0, hiw),
                      bc=(0, 0, 0, 1, 1, 1), omega_c=0.0, pmax=(1, 1, 3))
    h = rnd(g2.flat_shape, 61)
    E3 = 0.8 * rnd((g2.flat_shape[0],), 62) - 0.4
    u, v = g6.coords[3].reshape(-1), g6.coords[4].reshape(-1)
    au, bv = 1.0 + 0.2 * u, np.exp(-v * v)
    lift = lambda a2: (a2[None, None, :, None, None, :] * au[None, None, None, :, None, None] * bv[None, None, None, None, :, None]
                       * np.ones((g6.flat_shape[0], g6.flat_shape[1], 1, 1, 1, 1)))
    E6 = [None, None, E3[None, None, :] * np.ones(g6.flat_shape[:2] + (1,))]
    assert relerr(on.rhs(g6, lift(h), E6), lift(ov.rhs(g2, h, E3))) < 1e-13
    # one self-consistent step: the field of the lifted state is along z only and is the 1D1V field scaled by the u, v quadratures
    qu = float(np.sum(np.tile(g6.w[3] / g6.J[3], g6.nelem[3]) * au)); qv = float(np.sum(np.tile(g6.w[4] / g6.J[4], g6.nelem[4]) * bv))
    En = on.field_E(g6, lift(h))
    assert relerr(En[2], (qu * qv) * ov.field_E(g2, h)[None, None, :] * np.ones(g6.flat_shape[:2] + (1,))) < 1e-12
    assert max(np.max(np.abs(En[0])), np.max(np.abs(En[1]))) < 1e-12 * np.max(np.abs(En[2]))
