"""ORACLE (test infrastructure, not product code) -- 2D2V tensor-product DG Vlasov-Poisson.

The paper's method is written for any number of dimensions (Section 2, Eq. 18-21; Section 3,
PAPER.md:43: "computing the semi-discrete equation in n-dimensions"); its example is 1D2V.  This module applies the
same steps to four phase-space dimensions (x, y, u, v) = (x, y, v_x, v_y), array f[g_x][g_y][g_u][g_v]
(the paper's u[a0,b0,...,a3,b3] in C order), reusing the dimension-generic `basis_product` and
`flux_in_dim` of oracle/vlasov.py (Appendix A).  Plain NumPy, fp64; shares no code with the CUDA path.

Speeds (Eq. 28, with the second space dimension restored; E = -grad Phi, B = omega_c z^):
    a_x = u,  a_y = v,  a_u = -E_x(x,y) - omega_c v,  a_v = -E_y(x,y) + omega_c u.
Density (Eq. 27): rho[g_x][g_y] = sum_{g_u,g_v} (w/J_u)(w/J_v) f.
Field (reading C27 of DESIGN.md): the tensor product of Eq. 63 in x and y,
    c_pq = sum T^x_p[g_x] T^y_q[g_y] rho[g_x][g_y],   |p| <= pmax_x, |q| <= pmax_y,
and Eq. 68/71 with k^2 = k_p^2 + k_q^2:  Phi_pq = -c_pq / k^2,  E_pq = -i (k_p, k_q) Phi_pq,
(p,q) = (0,0) dropped (reading C5).

Pins: tests/test_oracle_2d2v.py (constant state, mass conservation, reduction to the 1D2V oracle for y-independent and,
with the axes swapped and omega_c -> -omega_c, x-independent states, plane-wave closed form of E, node-by-node loops).
"""
from __future__ import annotations

import numpy as np

from . import fourier
from .vlasov import Grid, basis_product, flux_in_dim


def make_grid(nelem, order, lo, hi, bc=None, omega_c=0.0, pmax=(0, 0), mass_mode=0) -> Grid:
    """Grid of oracle/vlasov.py with ndim = 4 plus the y transform; pmax = (pmax_x, pmax_y), 0 -> N_x, N_y."""
    if bc is None:
        bc = (0, 0, 1, 1)
    g = Grid(tuple(nelem), tuple(order), tuple(lo), tuple(hi), tuple(bc), omega_c, pmax[0], mass_mode)
    g.pmax_y = pmax[1] if pmax[1] else nelem[1]
    g.Ty = fourier.transform_tensor(lo[1], hi[1], nelem[1], order[1], g.pmax_y)
    return g


def _shaped(arr2d, d, nd=4):
    shp = [1] * (2 * nd)
    shp[2 * d], shp[2 * d + 1] = arr2d.shape
    return arr2d.reshape(shp)


def speeds(grid: Grid, Ex, Ey):
    """Eq. 28 with two space dimensions; Ex, Ey: [G_x][G_y] or None (= 0)."""
    Nx, nx, Ny, ny = grid.nelem[0], grid.order[0], grid.nelem[1], grid.order[1]
    def field(E):
        if E is None:
            return 0.0
        return np.asarray(E, dtype=np.float64).reshape(Nx, nx, Ny, ny, 1, 1, 1, 1)
    u, v = _shaped(grid.coords[2], 2), _shaped(grid.coords[3], 3)
    return [u, v, -field(Ex) - grid.omega_c * v, -field(Ey) + grid.omega_c * u]


def rhs(grid: Grid, f, Ex=None, Ey=None) -> np.ndarray:
    """Weak form Eq. 14 reduced by Eq. 20-21, four dimensions."""
    u = np.asarray(f, dtype=np.float64).reshape(grid.shape)
    a = speeds(grid, Ex, Ey)
    out = np.zeros(grid.shape)
    for d in range(4):
        flux = a[d] * u
        out += grid.J[d] * (basis_product(flux, grid.ups[d], grid.sub_element_axis(d))
                            - flux_in_dim(grid, flux, a[d], d))
    return out.reshape(grid.flat_shape)


def density(grid: Grid, f) -> np.ndarray:
    """Eq. 27 by LGL quadrature over (u, v): [G_x][G_y]."""
    u = np.asarray(f, dtype=np.float64).reshape(grid.shape)
    for d in (3, 2):
        wq = np.tile(grid.w[d] / grid.J[d], (grid.nelem[d], 1))
        u = np.tensordot(u, wq, axes=([2 * d, 2 * d + 1], [0, 1]))
    return u.reshape(grid.flat_shape[0], grid.flat_shape[1])


def fourier_project(grid: Grid, rho) -> np.ndarray:
    """c[p][q'] , p = 0..pmax_x, q' = q + pmax_y for q = -pmax_y..pmax_y (T_{-q} = conj T_q, Eq. 63)."""
    Tx = grid.T
    Ty2 = np.concatenate((np.conj(grid.Ty[:0:-1]), grid.Ty), axis=0)          # q = -pmax_y .. pmax_y
    return np.einsum("pg,qh,gh->pq", Tx, Ty2, np.asarray(rho, dtype=np.float64))


def poisson_E(grid: Grid, c):
    """Eq. 68 + Eq. 71 in two dimensions.  Real rho: c_{-p,-q} = conj c_{pq}, so the sum over all (p,q) is
    the p = 0, q > 0 and the p > 0 terms doubled and made real."""
    x, y = grid.coords[0].reshape(-1), grid.coords[1].reshape(-1)
    Lx, Ly = grid.hi[0] - grid.lo[0], grid.hi[1] - grid.lo[1]
    Ex = np.zeros((x.size, y.size)); Ey = np.zeros((x.size, y.size))
    for p in range(0, grid.pmax + 1):
        kp = 2.0 * np.pi * p / Lx
        for q in range(-grid.pmax_y, grid.pmax_y + 1):
            if p == 0 and q <= 0:
                continue
            kq = 2.0 * np.pi * q / Ly
            phi = -c[p, q + grid.pmax_y] / (kp * kp + kq * kq)
            wave = np.exp(1j * kp * x)[:, None] * np.exp(1j * kq * y)[None, :]
            Ex += 2.0 * np.real(-1j * kp * phi * wave)
            Ey += 2.0 * np.real(-1j * kq * phi * wave)
    return Ex, Ey


def field_E(grid: Grid, f):
    return poisson_E(grid, fourier_project(grid, density(grid, f)))


def ssprk3_step(grid: Grid, f, dt: float, self_consistent: bool = True, E_fixed=(None, None)) -> np.ndarray:
    """Shu-Osher SSP-RK3 (readings C3, C4)."""
    def L(u):
        Ex, Ey = field_E(grid, u) if self_consistent else E_fixed
        return rhs(grid, u, Ex, Ey)
    u = np.asarray(f, dtype=np.float64).reshape(grid.flat_shape)
    u1 = u + dt * L(u)
    u2 = 0.75 * u + 0.25 * (u1 + dt * L(u1))
    return (1.0 / 3.0) * u + (2.0 / 3.0) * (u2 + dt * L(u2))


def rhs_at(grid: Grid, f, Ex, Ey, g) -> float:
    """The same RHS at one node g = (g_x, g_y, g_u, g_v), scalar loops straight from Eq. 20, 21, 23, 14."""
    f = np.asarray(f).reshape(grid.flat_shape)
    def coord(dim, gi):
        return grid.coords[dim][gi // grid.order[dim], gi % grid.order[dim]]
    ex = 0.0 if Ex is None else Ex[g[0], g[1]]
    ey = 0.0 if Ey is None else Ey[g[0], g[1]]
    a_all = (coord(2, g[2]), coord(3, g[3]), -ex - grid.omega_c * coord(3, g[3]), -ey + grid.omega_c * coord(2, g[2]))
    total = 0.0
    for d in range(4):
        n, N = grid.order[d], grid.nelem[d]
        e, j = g[d] // n, g[d] % n
        a = a_all[d]
        def val(elem, node):
            idx = list(g); idx[d] = elem * n + node
            return f[tuple(idx)]
        vol = sum(grid.ups[d][j, k] * (a * val(e, k)) for k in range(n))
        uLm = val(e - 1, n - 1) if e > 0 else (val(N - 1, n - 1) if grid.bc[d] == 0 else 0.0)
        uRp = val(e + 1, 0) if e < N - 1 else (val(0, 0) if grid.bc[d] == 0 else 0.0)
        ap, am = max(a, 0.0), min(a, 0.0)
        total += grid.J[d] * (vol - grid.lift[d][j, 1] * (ap * val(e, n - 1) + am * uRp)
                              + grid.lift[d][j, 0] * (ap * uLm + am * val(e, 0)))
    return total
