"""ORACLE (test infrastructure, not product code) -- tensor-product DG Vlasov RHS + SSP-RK3.

Plain NumPy, fp64, following PAPER.md step by step in the paper's own array formulation:
data array u[a0,b0,a1,b1,(a2,b2)] (Section 3.1), `basis_product` = tensordot +
transpose (Section 3.1), upwind numerical flux by roll / sign masks
(Appendix A listing `flux_in_dim`), weak form Eq. 14, speeds of
Eq. 28, density Eq. 27, Shu-Osher SSP-RK3 with Poisson solved at
each stage.  Shares no code with the CUDA path (paper_2202_13532_b200/).

Pins: tests/test_oracle_vlasov.py (constant state, polynomial exactness, mass conservation,
weak == strong form, full-tensor Eq. 18 brute force, pointwise loop version, free streaming,
cyclotron rotation, Landau damping rate).
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

from . import basis, fourier


@dataclass
class Grid:
    """Rectilinear phase-space grid. ndim = 2: (x, v) [1D1V]; ndim = 3: (x, u, v) = (x, v_x, v_y)."""
    nelem: tuple
    order: tuple
    lo: tuple
    hi: tuple
    bc: tuple = None            # per dim: 0 periodic (the paper's roll), 1 zero-inflow (reading C2)
    omega_c: float = 0.0        # B_ext of Eq. 28
    pmax: int = 0               # Fourier modes kept; 0 -> nelem[0]
    mass_mode: int = 0          # 0 exact LGL mass (paper), 1 lumped (reading C1)
    ndim: int = field(init=False)

    def __post_init__(self):
        self.ndim = len(self.nelem)
        if self.bc is None:
            self.bc = (0,) + (1,) * (self.ndim - 1)
        if self.pmax == 0:
            self.pmax = self.nelem[0]
        self.J = [2.0 * self.nelem[d] / (self.hi[d] - self.lo[d]) for d in range(self.ndim)]  # Eq. 61
        self.xi, self.w, self.ups, self.lift = [], [], [], []
        for d in range(self.ndim):
            xi, w, ups, lift = basis.operators(self.order[d], self.mass_mode)
            self.xi.append(xi); self.w.append(w); self.ups.append(ups); self.lift.append(lift)
        # node coordinates per dim, shape [N_d, n_d]
        self.coords = [fourier.node_coordinates(self.lo[d], self.hi[d], self.nelem[d], self.order[d])
                       .reshape(self.nelem[d], self.order[d]) for d in range(self.ndim)]
        self.shape = tuple(s for d in range(self.ndim) for s in (self.nelem[d], self.order[d]))
        self.flat_shape = tuple(self.nelem[d] * self.order[d] for d in range(self.ndim))
        self._T = None

    # paper's index bookkeeping: element axis 2d, sub-element axis 2d+1
    def grid_axis(self, d):
        return 2 * d

    def sub_element_axis(self, d):
        return 2 * d + 1

    @property
    def T(self):
        if self._T is None:
            self._T = fourier.transform_tensor(self.lo[0], self.hi[0], self.nelem[0], self.order[0], self.pmax)
        return self._T

    def x_nodes(self):
        return self.coords[0].reshape(-1)


def basis_product(flux: np.ndarray, basis_matrix: np.ndarray, axis: int) -> np.ndarray:
    """Section 3.1 (the listing itself is lost, reading C18): contract the
    sub-element axis `axis` of `flux` with the column index of `basis_matrix[j, k]` by
    tensordot, then transpose the new (last) axis back to position `axis`."""
    out = np.tensordot(flux, basis_matrix, axes=([axis], [1]))
    nd = flux.ndim
    permutation = list(range(axis)) + [nd - 1] + list(range(axis, nd - 1))
    return np.transpose(out, permutation)


def speeds(grid: Grid, E):
    """Eq. 28 with E = -d_x Phi (reading C15), broadcast-shaped per dim.
    1D2V: a_x = u, a_u = -E(x) - omega_c v, a_v = omega_c u.   1D1V: a_x = v, a_v = -E(x)."""
    nd = grid.ndim
    def shaped(arr2d, d):
        shp = [1] * (2 * nd)
        shp[2 * d], shp[2 * d + 1] = arr2d.shape
        return arr2d.reshape(shp)
    Ex = np.zeros((grid.nelem[0], grid.order[0])) if E is None else np.asarray(E).reshape(grid.nelem[0], grid.order[0])
    if nd == 2:
        return [shaped(grid.coords[1], 1), -shaped(Ex, 0)]
    return [shaped(grid.coords[1], 1),
            -shaped(Ex, 0) - grid.omega_c * shaped(grid.coords[2], 2),
            grid.omega_c * shaped(grid.coords[1], 1)]


def flux_in_dim(grid: Grid, flux: np.ndarray, speed: np.ndarray, d: int) -> np.ndarray:
    """Appendix A `flux_in_dim`: build the numerical-flux array of shape
    [..., N_d, 2, ...] with the upwind rule Eq. 23, left face stored with its
    outward normal -1, right face with +1, then contract with Xi.  `roll` supplies the periodic
    neighbour; for bc = 1 (zero inflow, reading C2) the wrapped-around exterior state is zero."""
    one_negatives = np.where(speed < 0, 1.0, 0.0)
    one_positives = np.where(speed > 0, 1.0, 0.0)
    ax_e, ax_s = grid.grid_axis(d), grid.sub_element_axis(d)
    n = grid.order[d]
    left = [slice(None)] * flux.ndim;  left[ax_s] = slice(0, 1)           # boundary_slices[d][0]
    right = [slice(None)] * flux.ndim; right[ax_s] = slice(n - 1, n)       # boundary_slices[d][1]
    left, right = tuple(left), tuple(right)
    from_left = np.roll(flux[right], shift=1, axis=ax_e)     # right face of element e-1
    from_right = np.roll(flux[left], shift=-1, axis=ax_e)    # left face of element e+1
    if grid.bc[d] == 1:
        first = [slice(None)] * flux.ndim; first[ax_e] = slice(0, 1)
        last = [slice(None)] * flux.ndim;  last[ax_e] = slice(grid.nelem[d] - 1, grid.nelem[d])
        from_left = from_left.copy();  from_left[tuple(first)] = 0.0
        from_right = from_right.copy(); from_right[tuple(last)] = 0.0
    # the speed does not depend on its own coordinate (Eq. 28), so its masks broadcast over axis d
    num_flux_left = -1.0 * (from_left * one_positives + flux[left] * one_negatives)
    num_flux_right = flux[right] * one_positives + from_right * one_negatives
    num_flux = np.concatenate((num_flux_left, num_flux_right), axis=ax_s)
    return basis_product(num_flux, grid.lift[d], ax_s)


def rhs(grid: Grid, f: np.ndarray, E=None) -> np.ndarray:
    """Weak form Eq. 14 reduced by Eq. 20-21:
    du/dt = sum_d J_d ( Upsilon_d F_d - Xi_d NumFlux_d ),  F_d = a_d u (conservative, reading C13)."""
    u = np.asarray(f, dtype=np.float64).reshape(grid.shape)
    a = speeds(grid, E)
    out = np.zeros(grid.shape)
    for d in range(grid.ndim):
        flux = a[d] * u
        out += grid.J[d] * (basis_product(flux, grid.ups[d], grid.sub_element_axis(d))
                            - flux_in_dim(grid, flux, a[d], d))
    return out.reshape(grid.flat_shape)


def rhs_strong(grid: Grid, f: np.ndarray, E=None) -> np.ndarray:
    """Strong form Eq. 15: du/dt = sum_d J_d ( -D_d F_d + Xi_d (F_d|faces - NumFlux_d) ), with
    D = Eq. 55 and the boundary values of F signed by the outward normal like the numerical flux
    (Appendix A).  Equal to rhs() up to rounding (tests/test_oracle_vlasov.py)."""
    u = np.asarray(f, dtype=np.float64).reshape(grid.shape)
    a = speeds(grid, E)
    out = np.zeros(grid.shape)
    for d in range(grid.ndim):
        n = grid.order[d]
        D = basis.lagrange_derivative_matrix(n)
        flux = a[d] * u
        ax = grid.sub_element_axis(d)
        left = [slice(None)] * flux.ndim;  left[ax] = slice(0, 1)
        right = [slice(None)] * flux.ndim; right[ax] = slice(n - 1, n)
        face_flux = np.concatenate((-flux[tuple(left)], flux[tuple(right)]), axis=ax)
        out += grid.J[d] * (-basis_product(flux, D, ax) + basis_product(face_flux, grid.lift[d], ax)
                            - flux_in_dim(grid, flux, a[d], d))
    return out.reshape(grid.flat_shape)


def density(grid: Grid, f: np.ndarray) -> np.ndarray:
    """Eq. 27 zeroth moment by LGL quadrature (reading C14):
    rho[g_x] = sum over velocity nodes of prod_d (w_b / J_d) f."""
    u = np.asarray(f, dtype=np.float64).reshape(grid.shape)
    for d in range(grid.ndim - 1, 0, -1):
        wq = np.tile(grid.w[d] / grid.J[d], (grid.nelem[d], 1))        # [N_d, n_d]
        u = np.tensordot(u, wq, axes=([2 * d, 2 * d + 1], [0, 1]))
    return u.reshape(-1)


def field_E(grid: Grid, f: np.ndarray) -> np.ndarray:
    """rho -> c_p (Eq. 63) -> E (Eq. 71)."""
    rho = density(grid, f)
    c = fourier.fourier_project(grid.T, rho)
    return fourier.poisson_E(grid.lo[0], grid.hi[0], grid.x_nodes(), c)


def ssprk3_step(grid: Grid, f: np.ndarray, dt: float, self_consistent: bool = True, E_fixed=None, strong: bool = False) -> np.ndarray:
    """Shu-Osher SSP-RK3 (reading C3), E from each stage's input (reading C4):
    u1 = u + dt L(u); u2 = 3/4 u + 1/4 (u1 + dt L(u1)); u+ = 1/3 u + 2/3 (u2 + dt L(u2))."""
    def L(u):
        E = field_E(grid, u) if self_consistent else E_fixed
        return rhs_strong(grid, u, E) if strong else rhs(grid, u, E)
    u = np.asarray(f, dtype=np.float64).reshape(grid.flat_shape)
    u1 = u + dt * L(u)
    u2 = 0.75 * u + 0.25 * (u1 + dt * L(u1))
    return (1.0 / 3.0) * u + (2.0 / 3.0) * (u2 + dt * L(u2))
