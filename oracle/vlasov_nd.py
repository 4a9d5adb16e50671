"""ORACLE (test infrastructure, not product code) -- tensor-product DG Vlasov-Poisson in d_x + d_v dimensions.

The paper writes its method for any number of dimensions (Section 2, Eq. 18-21; Section 3,
PAPER.md:43: "computing the semi-discrete equation in n-dimensions") and runs it in 1D2V.  This module is the same
sequence of steps for a phase space (x_1..x_dx, v_1..v_dv), 1 <= d_x <= d_v <= 3 (1D1V, 1D2V, 1D3V, 2D2V, 2D3V, 3D3V),
array f[g_x1]..[g_xdx][g_v1]..[g_vdv] (the paper's u[a0,b0,...] in C order), built from the
dimension-generic `basis_product` and `flux_in_dim` of oracle/vlasov.py (Appendix A).  Plain NumPy,
fp64; shares no code with the CUDA path.

Speeds (Eq. 28, with all space dimensions restored; E = -grad Phi, B = omega_c z^):
    a_{x_i} = v_i                          i < d_x
    a_{v_1} = -E_1 - omega_c v_2           (no magnetic term when d_v = 1)
    a_{v_2} = -E_2 + omega_c v_1           (E_2 = 0 when d_x < 2)
    a_{v_3} = -E_3                         (E_3 = 0 when d_x < 3; B along z does not act on v_3)
Every a_d is independent of its own coordinate, so the conservative flux a_d f is the advective one (reading C13).
Density (Eq. 27): rho[x] = sum over all velocity nodes of prod_i (w/J_{v_i}) f.
Field (reading C27 of DESIGN.md carried to d_x dimensions): the tensor product of Eq. 63 over the space
dimensions, c_p = sum_x prod_i T^{(i)}_{p_i}[g_{x_i}] rho[x], |p_i| <= pmax_i, and Eq. 68/71 with
k^2 = sum k_{p_i}^2: Phi_p = -c_p / k^2, E_p = -i k_p Phi_p, p = 0 dropped (reading C5).

Pins: tests/test_oracle_nd.py -- constant state, mass conservation, exact agreement with the pinned 1D2V and 2D2V oracles on
their shapes, reduction of 3D3V / 2D3V / 1D3V states that do not depend on the extra dimensions to those oracles, plane-wave
closed form of E in three dimensions.  The third force component a_{v_3} = -E_3 (the i >= 2 branch of `speeds`) is pinned by
the relabelling symmetry (x_1, v_1) <-> (x_3, v_3) of the unmagnetised equation and by a z-only problem that must equal the
pinned 1D1V oracle on (z, w); flipping that sign fails both.
"""
from __future__ import annotations

import itertools

import numpy as np

from . import fourier
from .vlasov import Grid, basis_product, flux_in_dim


def make_grid(dx, dv, nelem, order, lo, hi, bc=None, omega_c=0.0, pmax=None, mass_mode=0) -> Grid:
    """Grid of oracle/vlasov.py with ndim = dx + dv, plus one DG->Fourier tensor per space dimension.
    pmax: per space dimension, 0 -> N."""
    assert 1 <= dx <= dv <= 3 and len(nelem) == dx + dv
    if bc is None:
        bc = (0,) * dx + (1,) * dv
    pmax = tuple(pmax) if pmax is not None else (0,) * dx
    g = Grid(tuple(nelem), tuple(order), tuple(lo), tuple(hi), tuple(bc), omega_c, pmax[0], mass_mode)
    g.dx, g.dv = dx, dv
    g.pmaxs = tuple(pmax[i] if pmax[i] else nelem[i] for i in range(dx))
    g.Ts = [fourier.transform_tensor(lo[i], hi[i], nelem[i], order[i], g.pmaxs[i]) for i in range(dx)]
    return g


def _shaped(grid: Grid, arr2d, d):
    shp = [1] * (2 * grid.ndim)
    shp[2 * d], shp[2 * d + 1] = arr2d.shape
    return arr2d.reshape(shp)


def _field_shaped(grid: Grid, E):
    """E component on the space nodes [G_x1]..[G_xdx] -> broadcast shape over the paper's index pairs."""
    if E is None:
        return 0.0
    shp = [s for i in range(grid.dx) for s in (grid.nelem[i], grid.order[i])] + [1] * (2 * grid.dv)
    return np.asarray(E, dtype=np.float64).reshape(shp)


def speeds(grid: Grid, E):
    """Eq. 28 in d_x + d_v dimensions.  E: sequence of d_x arrays [G_x1]..[G_xdx] (entries or E itself may be None = 0)."""
    dx, dv = grid.dx, grid.dv
    E = [None] * dx if E is None else list(E)
    v = [_shaped(grid, grid.coords[dx + i], dx + i) for i in range(dv)]
    a = [v[i] for i in range(dx)]
    for i in range(dv):
        e = _field_shaped(grid, E[i]) if i < dx else 0.0
        if i == 0:
            a.append(-e - (grid.omega_c * v[1] if dv >= 2 else np.zeros([1] * (2 * grid.ndim))))
        elif i == 1:
            a.append(-e + grid.omega_c * v[0])
        else:
            a.append(-e + np.zeros([1] * (2 * grid.ndim)))      # independent of v_3 itself (no magnetic term along B)
    return a


def rhs(grid: Grid, f, E=None) -> np.ndarray:
    """Weak form Eq. 14 reduced by Eq. 20-21, one term per dimension."""
    u = np.asarray(f, dtype=np.float64).reshape(grid.shape)
    a = speeds(grid, E)
    out = np.zeros(grid.shape)
    for d in range(grid.ndim):
        flux = a[d] * u
        out += grid.J[d] * (basis_product(flux, grid.ups[d], grid.sub_element_axis(d)) - flux_in_dim(grid, flux, a[d], d))
    return out.reshape(grid.flat_shape)


def density(grid: Grid, f) -> np.ndarray:
    """Eq. 27 by LGL quadrature over every velocity dimension: [G_x1]..[G_xdx]."""
    u = np.asarray(f, dtype=np.float64).reshape(grid.shape)
    for d in range(grid.ndim - 1, grid.dx - 1, -1):
        wq = np.tile(grid.w[d] / grid.J[d], (grid.nelem[d], 1))
        u = np.tensordot(u, wq, axes=([2 * d, 2 * d + 1], [0, 1]))
    return u.reshape(grid.flat_shape[:grid.dx])


def _mode_axes(grid: Grid):
    """Mode numbers kept per space dimension: p_1 = 0..pmax_1 (the other half-space by conjugation, rho is real),
    p_i = -pmax_i..pmax_i for i > 1."""
    return [np.arange(0, grid.pmaxs[0] + 1)] + [np.arange(-grid.pmaxs[i], grid.pmaxs[i] + 1) for i in range(1, grid.dx)]


def fourier_project(grid: Grid, rho) -> np.ndarray:
    """c[p_1][p_2'][p_3'] with p_i' = p_i + pmax_i for i > 1 (T_{-p} = conj T_p, Eq. 63), one contraction per dimension."""
    c = np.asarray(rho, dtype=np.float64).astype(np.complex128)
    for i in range(grid.dx):
        T = grid.Ts[i] if i == 0 else np.concatenate((np.conj(grid.Ts[i][:0:-1]), grid.Ts[i]), axis=0)
        c = np.moveaxis(np.tensordot(T, c, axes=([1], [i])), 0, i)
    return c


def poisson_E(grid: Grid, c):
    """Eq. 68 + Eq. 71 in d_x dimensions, mode by mode.  Real rho: c_{-p} = conj c_p, so the sum over the full lattice is
    the kept half-space (p_1 > 0, or p_1 = 0 and the first non-zero of the remaining p_i positive) doubled and made real."""
    dx = grid.dx
    xs = [grid.coords[i].reshape(-1) for i in range(dx)]
    Ls = [grid.hi[i] - grid.lo[i] for i in range(dx)]
    E = [np.zeros([x.size for x in xs]) for _ in range(dx)]
    axes = _mode_axes(grid)
    for idx in itertools.product(*[range(a.size) for a in axes]):
        p = [int(axes[i][idx[i]]) for i in range(dx)]
        first = next((q for q in p if q != 0), 0)
        if first <= 0:
            continue                                   # the zero mode, and the half-space given by conjugation
        k = [2.0 * np.pi * p[i] / Ls[i] for i in range(dx)]
        phi = -c[idx] / sum(ki * ki for ki in k)
        wave = np.ones([1] * dx, dtype=np.complex128)
        for i in range(dx):
            shp = [1] * dx; shp[i] = xs[i].size
            wave = wave * np.exp(1j * k[i] * xs[i]).reshape(shp)
        for i in range(dx):
            E[i] += 2.0 * np.real(-1j * k[i] * phi * wave)
    return E


def field_E(grid: Grid, f):
    return poisson_E(grid, fourier_project(grid, density(grid, f)))


def ssprk3_step(grid: Grid, f, dt: float, self_consistent: bool = True, E_fixed=None) -> np.ndarray:
    """Shu-Osher SSP-RK3 (readings C3, C4)."""
    def L(u):
        return rhs(grid, u, field_E(grid, u) if self_consistent else E_fixed)
    u = np.asarray(f, dtype=np.float64).reshape(grid.flat_shape)
    u1 = u + dt * L(u)
    u2 = 0.75 * u + 0.25 * (u1 + dt * L(u1))
    return (1.0 / 3.0) * u + (2.0 / 3.0) * (u2 + dt * L(u2))
