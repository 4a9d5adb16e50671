"""ORACLE (test infrastructure, not product code) -- the same RHS, one node at a time.

Scalar Python loops straight from Eq. 20 (volume term), Eq. 21 + Eq. 23 (upwind face term)
and Eq. 14 (weak form) of PAPER.md, on the flat array f[g_x][g_u][g_v] (g = a*n + b).  It is
(i) a brute-force cross-check of oracle/vlasov.py's array formulation on small grids and
(ii) the way single outputs are sampled at BASELINE.json's full sizes, where the array
oracle is slow.  It shares nothing with the CUDA path.
"""
from __future__ import annotations

import numpy as np

from .vlasov import Grid


def _speed(grid: Grid, E, d: int, g):
    """Eq. 28, E = -d_x Phi (reading C15). g = tuple of flat node indices."""
    def coord(dim, gi):
        n = grid.order[dim]
        return grid.coords[dim][gi // n, gi % n]
    Ex = 0.0 if E is None else E[g[0]]
    if grid.ndim == 2:
        return coord(1, g[1]) if d == 0 else -Ex
    if d == 0:
        return coord(1, g[1])
    if d == 1:
        return -Ex - grid.omega_c * coord(2, g[2])
    return grid.omega_c * coord(1, g[1])


def rhs_at(grid: Grid, f: np.ndarray, E, g) -> float:
    """du/dt at flat node g = (g_x, g_u[, g_v]):
    sum_d J_d ( a_d sum_k Ups[j,k] f_k  -  Xi[j,R] Flux_R  +  Xi[j,L] Flux_L ),
    Flux = a^+ u_left + a^- u_right (Eq. 23), neighbour periodic (bc 0) or zero exterior (bc 1)."""
    f = f.reshape(grid.flat_shape)
    total = 0.0
    for d in range(grid.ndim):
        n, N = grid.order[d], grid.nelem[d]
        e, j = g[d] // n, g[d] % n
        a = _speed(grid, E, d, g)

        def val(elem, node):
            idx = list(g)
            idx[d] = elem * n + node
            return f[tuple(idx)]

        vol = 0.0
        for k in range(n):
            vol += grid.ups[d][j, k] * (a * val(e, k))
        # exterior states
        if e > 0:
            uLm = val(e - 1, n - 1)
        else:
            uLm = val(N - 1, n - 1) if grid.bc[d] == 0 else 0.0
        if e < N - 1:
            uRp = val(e + 1, 0)
        else:
            uRp = val(0, 0) if grid.bc[d] == 0 else 0.0
        ap, am = max(a, 0.0), min(a, 0.0)
        flux_L = ap * uLm + am * val(e, 0)          # left face: left state is the neighbour
        flux_R = ap * val(e, n - 1) + am * uRp      # right face: right state is the neighbour
        total += grid.J[d] * (vol - grid.lift[d][j, 1] * flux_R + grid.lift[d][j, 0] * flux_L)
    return total


def density_at(grid: Grid, f: np.ndarray, gx: int) -> float:
    """Eq. 27 at one x node, LGL quadrature, plain loops."""
    f = f.reshape(grid.flat_shape)
    tot = 0.0
    if grid.ndim == 2:
        for gv in range(grid.flat_shape[1]):
            tot += grid.w[1][gv % grid.order[1]] / grid.J[1] * f[gx, gv]
        return tot
    for gu in range(grid.flat_shape[1]):
        wu = grid.w[1][gu % grid.order[1]] / grid.J[1]
        row = 0.0
        for gv in range(grid.flat_shape[2]):
            row += grid.w[2][gv % grid.order[2]] / grid.J[2] * f[gx, gu, gv]
        tot += wu * row
    return tot
