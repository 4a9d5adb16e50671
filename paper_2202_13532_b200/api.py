"""Thin Python binding over the C ABI (include/dgvlasov.h): argument marshalling only.

torch provides device memory and streams; every step of the path runs in the library's kernels.
Method names mirror the C entry points (dg_rhs -> DGContext.rhs, ...)."""
from __future__ import annotations

import ctypes as C

import numpy as np
import torch

from . import _lib

_L = _lib.load()

OPT_RHS_KERNEL = 1
OPT_FIELD_KERNEL = 2
OPT_PROFILE = 3
OPT_PDL = 4
OPT_FORM = 5
FORM_WEAK, FORM_STRONG = 0, 1
KERNEL_AUTO, KERNEL_GENERIC, KERNEL_TILED = 0, 1, 2
FIELD_AUTO, FIELD_SIMPLE, FIELD_DMMA, FIELD_DFMA, FIELD_FFT = 0, 1, 2, 3, 4
BC_PERIODIC, BC_ZERO_INFLOW, BC_HALO = 0, 1, 2


class DGError(RuntimeError):
    pass


def _check(rc: int, what: str):
    if rc != 0:
        raise DGError(f"{what} failed ({rc}): {_L.dg_last_error().decode()}")


def _ptr(t):
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise DGError("expected a contiguous float64 CUDA tensor")
    return t.data_ptr()


def _stream(device):
    return torch.cuda.current_stream(device).cuda_stream


def version() -> str:
    return _L.dg_version().decode()


def ssprk3_stage_coeffs(stage: int):
    """dg_ssprk3_stage_coeffs: (c0, c1) of Shu-Osher stage 0, 1, 2 -- the table lives in the library."""
    c0, c1 = C.c_double(0.0), C.c_double(0.0)
    _check(_L.dg_ssprk3_stage_coeffs(int(stage), C.byref(c0), C.byref(c1)), "dg_ssprk3_stage_coeffs")
    return c0.value, c1.value


def fp64_peak(device=0, variant=0, iters=20000) -> float:
    """dg_fp64_peak: measured FP64 TFLOP/s of the device (variant 0 DFMA, 1 DMMA)."""
    tf = C.c_double(0.0)
    _check(_L.dg_fp64_peak(int(device), int(variant), int(iters), C.byref(tf)), "dg_fp64_peak")
    return tf.value


STATIC_MAX_GX = 16384      # DG_STATIC_MAX_GX of include/dgvlasov_noalloc.h


def density_static(f, wq_u, wq_v, out):
    """dg_density_static: the density moment (Eq. 27) without a context or a workspace, for callers that must not
    allocate device memory where they stand (a hook inside another code's time loop that owns all of the HBM, a
    latency-critical callback that cannot afford the device-wide stall of cudaMalloc).  The partial sums go to a 2 MiB
    array built into the library, shared by every call on the device: keep calls on one stream or order them with
    events, and make the first call on each device at start-up (it looks up the array's address).
    f: [G_x][G_u][G_v] or [G_x][G_v]; wq_u / wq_v: per-node quadrature weights [G_u] / [G_v] (wq_v None for 1D1V);
    out: [G_x], required -- this wrapper allocates nothing either.  G_x <= STATIC_MAX_GX."""
    if out is None:
        raise DGError("density_static: pass the output tensor (nothing is allocated on this path)")
    G_x, G_u = int(f.shape[0]), int(f.shape[1])
    G_v = int(f.shape[2]) if f.dim() == 3 else 1
    _check(_L.dg_density_static(_ptr(f), G_x, G_u, G_v, _ptr(wq_u), _ptr(wq_v), _ptr(out), f.device.index or 0,
                                _stream(f.device)), "dg_density_static")
    return out


class DGContext:
    """dg_create / dg_destroy plus one method per C entry point."""

    def __init__(self, nelem, order, lo, hi, bc=None, omega_c=0.0, pmax=0, mass_mode=0, device=0,
                 workspace=True, field_batch=1):
        ndim = len(nelem)
        if bc is None:
            bc = (0,) + (1,) * (ndim - 1)
        d = _lib.GridDesc()
        d.ndim = ndim
        for i in range(3):
            d.nelem[i] = int(nelem[i]) if i < ndim else 0
            d.order[i] = int(order[i]) if i < ndim else 0
            d.lo[i] = float(lo[i]) if i < ndim else 0.0
            d.hi[i] = float(hi[i]) if i < ndim else 0.0
            d.bc[i] = int(bc[i]) if i < ndim else 0
        d.omega_c, d.pmax, d.mass_mode, d.device = float(omega_c), int(pmax), int(mass_mode), int(device)
        self._h = C.c_void_p()
        _check(_L.dg_create(C.byref(d), C.byref(self._h)), "dg_create")
        self.ndim, self.nelem, self.order = ndim, tuple(nelem), tuple(order)
        self.device = torch.device("cuda", device)
        self.flat_shape = tuple(int(nelem[i]) * int(order[i]) for i in range(ndim))
        self.pmax = int(pmax) if pmax > 0 else int(nelem[0])
        self._ws = None
        if workspace:
            nbytes = _L.dg_field_workspace_bytes(self._h, int(field_batch))
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self._ws.data_ptr() + 255) // 256 * 256
            _check(_L.dg_set_workspace(self._h, base, nbytes), "dg_set_workspace")

    @classmethod
    def field_nonuniform(cls, edges, order, pmax=0, device=0, field_batch=1):
        """dg_create_field_nonuniform: x-only context with explicitly given element edges (Eq. 63's (Delta x)_m)."""
        e = np.ascontiguousarray(edges, dtype=np.float64)
        self = cls.__new__(cls)
        self._h = C.c_void_p()
        nelem = e.size - 1
        _check(_L.dg_create_field_nonuniform(e.ctypes.data_as(C.POINTER(C.c_double)), nelem, int(order), int(pmax), int(device),
                                             C.byref(self._h)), "dg_create_field_nonuniform")
        self.ndim, self.nelem, self.order = 1, (nelem,), (int(order),)
        self.device = torch.device("cuda", device)
        self.flat_shape = (nelem * int(order),)
        self.pmax = int(pmax) if pmax > 0 else nelem
        nbytes = _L.dg_field_workspace_bytes(self._h, int(field_batch))
        self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self._ws.data_ptr() + 255) // 256 * 256
        _check(_L.dg_set_workspace(self._h, base, nbytes), "dg_set_workspace")
        return self

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            _L.dg_destroy(self._h)
            self._h = C.c_void_p()
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # --- compute entry points -----------------------------------------------------------------
    def rhs(self, f, E=None, out=None):
        out = torch.empty_like(f) if out is None else out
        _check(_L.dg_rhs(self._h, _ptr(f), _ptr(E), _ptr(out), _stream(self.device)), "dg_rhs")
        return out

    def set_xhalo(self, halo):
        """halo: [2][G_u][G_v] exterior x-face planes of an x-slab context (bc[0] = BC_HALO); kept alive here."""
        self._xhalo = halo
        _check(_L.dg_set_xhalo(self._h, _ptr(halo)), "dg_set_xhalo")

    def set_xhalo_push(self, left_dst, right_dst):
        """left_dst / right_dst: [G_u][G_v] planes in the x-neighbours' halo buffers (or None); kept alive here."""
        self._push = (left_dst, right_dst)
        _check(_L.dg_set_xhalo_push(self._h, _ptr(left_dst), _ptr(right_dst)), "dg_set_xhalo_push")

    def rk_stage(self, f_s, f_n, E, out, c0, c1, dt, rho_out=None):
        _check(_L.dg_rk_stage(self._h, _ptr(f_s), _ptr(f_n), _ptr(E), _ptr(out), float(c0), float(c1), float(dt),
                              _ptr(rho_out), _stream(self.device)), "dg_rk_stage")
        return out

    def ssprk3_step(self, f, dt, self_consistent=True):
        _check(_L.dg_ssprk3_step(self._h, _ptr(f), float(dt), int(bool(self_consistent)), _stream(self.device)), "dg_ssprk3_step")
        return f

    def ssprk3_run(self, f, dt, nsteps, self_consistent=True):
        _check(_L.dg_ssprk3_run(self._h, _ptr(f), float(dt), int(nsteps), int(bool(self_consistent)), _stream(self.device)), "dg_ssprk3_run")
        return f

    def ssprk3_run_host(self, f_host, dt, nsteps, self_consistent=True):
        """f_host: contiguous float64 CPU tensor or NumPy array, updated in place."""
        if isinstance(f_host, np.ndarray):
            assert f_host.dtype == np.float64 and f_host.flags["C_CONTIGUOUS"]
            p = f_host.ctypes.data
        else:
            assert f_host.dtype == torch.float64 and f_host.is_contiguous() and not f_host.is_cuda
            p = f_host.data_ptr()
        _check(_L.dg_ssprk3_run_host(self._h, p, float(dt), int(nsteps), int(bool(self_consistent))), "dg_ssprk3_run_host")
        return f_host

    def density(self, f, out=None):
        out = torch.empty(self.flat_shape[0], dtype=torch.float64, device=self.device) if out is None else out
        _check(_L.dg_density(self._h, _ptr(f), _ptr(out), _stream(self.device)), "dg_density")
        return out

    def fourier_project(self, rho, out=None):
        rho2 = rho.reshape(-1, self.flat_shape[0])
        batch = rho2.shape[0]
        out = torch.empty((batch, self.pmax + 1, 2), dtype=torch.float64, device=self.device) if out is None else out
        _check(_L.dg_fourier_project(self._h, _ptr(rho2), batch, _ptr(out), _stream(self.device)), "dg_fourier_project")
        return out

    def poisson_E(self, rho, out=None):
        rho2 = rho.reshape(-1, self.flat_shape[0])
        batch = rho2.shape[0]
        out = torch.empty_like(rho2) if out is None else out
        _check(_L.dg_poisson_E(self._h, _ptr(rho2), batch, _ptr(out), _stream(self.device)), "dg_poisson_E")
        return out.reshape(rho.shape)

    def poisson_phi(self, rho, out=None):
        rho2 = rho.reshape(-1, self.flat_shape[0])
        batch = rho2.shape[0]
        out = torch.empty_like(rho2) if out is None else out
        _check(_L.dg_poisson_phi(self._h, _ptr(rho2), batch, _ptr(out), _stream(self.device)), "dg_poisson_phi")
        return out.reshape(rho.shape)

    def broken_l2(self, u, v=None, out=None):
        u2 = u.reshape(-1, self.flat_shape[0])
        v2 = None if v is None else v.reshape(-1, self.flat_shape[0])
        batch = u2.shape[0]
        out = torch.empty(batch, dtype=torch.float64, device=self.device) if out is None else out
        _check(_L.dg_broken_l2(self._h, _ptr(u2), _ptr(v2), batch, _ptr(out), _stream(self.device)), "dg_broken_l2")
        return out

    def field_energy(self, E, out=None):
        """dg_field_energy: W = (1/2) int E^2 dx per vector (Fig. 10), exact LGL mass matrix."""
        E2 = E.reshape(-1, self.flat_shape[0])
        batch = E2.shape[0]
        out = torch.empty(batch, dtype=torch.float64, device=self.device) if out is None else out
        _check(_L.dg_field_energy(self._h, _ptr(E2), batch, _ptr(out), _stream(self.device)), "dg_field_energy")
        return out

    # --- introspection ------------------------------------------------------------------------
    def operators(self, dim):
        n = self.order[dim]
        xi, w = np.empty(n), np.empty(n)
        ups, lift = np.empty((n, n)), np.empty((n, 2))
        dp = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
        _check(_L.dg_get_operators(self._h, dim, dp(xi), dp(w), dp(ups), dp(lift)), "dg_get_operators")
        return xi, w, ups, lift

    def dmatrix(self, dim):
        n = self.order[dim]
        D = np.empty((n, n))
        _check(_L.dg_get_dmatrix(self._h, dim, D.ctypes.data_as(C.POINTER(C.c_double))), "dg_get_dmatrix")
        return D

    def nodes(self, dim):
        x = np.empty(self.flat_shape[dim])
        _check(_L.dg_get_nodes(self._h, dim, x.ctypes.data_as(C.POINTER(C.c_double))), "dg_get_nodes")
        return x

    def transform(self, p_first=0, p_count=None):
        p_count = self.pmax + 1 - p_first if p_count is None else p_count
        T = np.empty((p_count, self.flat_shape[0], 2))
        _check(_L.dg_get_transform(self._h, p_first, p_count, T.ctypes.data_as(C.POINTER(C.c_double))), "dg_get_transform")
        return T[..., 0] + 1j * T[..., 1]

    def max_stable_dt(self, E_bound=0.0):
        return float(_L.dg_max_stable_dt(self._h, float(E_bound)))

    def set_option(self, key, value):
        _check(_L.dg_set_option(self._h, int(key), int(value)), "dg_set_option")

    def get_profile(self, reset=True):
        ms, cnt = C.c_double(0.0), C.c_int64(0)
        _check(_L.dg_get_profile(self._h, C.byref(ms), C.byref(cnt), int(bool(reset))), "dg_get_profile")
        return ms.value, cnt.value

    def get_profile_stages(self, reset=True):
        """([ms] * 4, [launches] * 4): index 0 = RHS launches outside dg_ssprk3_*, 1..3 = RK stages 1..3."""
        ms, cnt = (C.c_double * 4)(), (C.c_int64 * 4)()
        _check(_L.dg_get_profile_stages(self._h, ms, cnt, int(bool(reset))), "dg_get_profile_stages")
        return list(ms), list(cnt)

    def check_finite(self, f, flag=None):
        """dg_check_finite: int32 device flag, 0 = every value of f finite, 1 = some Inf/NaN (asynchronous)."""
        flag = torch.empty(1, dtype=torch.int32, device=self.device) if flag is None else flag
        _check(_L.dg_check_finite(self._h, _ptr(f), flag.data_ptr(), _stream(self.device)), "dg_check_finite")
        return flag

    @property
    def launch_count(self):
        return int(_L.dg_launch_count(self._h))

    @property
    def last_kernel(self):
        return _L.dg_last_kernel(self._h).decode()

    @property
    def last_field_kernel(self):
        return _L.dg_last_field_kernel(self._h).decode()


OPT4_RHS_KERNEL, OPT4_PROFILE = 1, 3
KERNEL4_AUTO, KERNEL4_GENERIC, KERNEL4_TILED, KERNEL4_ELEMENT, KERNEL4_LINE = 0, 1, 2, 3, 4


class DG4Context:
    """2D2V variant (include/dgvlasov2d2v.h): dg4_create / dg4_destroy plus one method per C entry point.
    f: [G_x][G_y][G_u][G_v]; fields and density: [G_x][G_y]."""

    def __init__(self, nelem, order, lo, hi, bc=(0, 0, 1, 1), omega_c=0.0, pmax=(0, 0), mass_mode=0, device=0, workspace=True):
        d = _lib.GridDesc4()
        for i in range(4):
            d.nelem[i], d.order[i], d.lo[i], d.hi[i], d.bc[i] = int(nelem[i]), int(order[i]), float(lo[i]), float(hi[i]), int(bc[i])
        d.pmax[0], d.pmax[1] = int(pmax[0]), int(pmax[1])
        d.omega_c, d.mass_mode, d.device = float(omega_c), int(mass_mode), int(device)
        self._h = C.c_void_p()
        _check(_L.dg4_create(C.byref(d), C.byref(self._h)), "dg4_create")
        self.nelem, self.order = tuple(nelem), tuple(order)
        self.device = torch.device("cuda", device)
        self.flat_shape = tuple(int(nelem[i]) * int(order[i]) for i in range(4))
        self.pmax = (int(pmax[0]) or int(nelem[0]), int(pmax[1]) or int(nelem[1]))
        self._ws = None
        if workspace:
            nbytes = _L.dg4_workspace_bytes(self._h)
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self._ws.data_ptr() + 255) // 256 * 256
            _check(_L.dg4_set_workspace(self._h, base, nbytes), "dg4_set_workspace")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            _L.dg4_destroy(self._h)
            self._h = C.c_void_p()
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _field(self):
        return torch.empty(self.flat_shape[:2], dtype=torch.float64, device=self.device)

    def rhs(self, f, Ex=None, Ey=None, out=None):
        out = torch.empty_like(f) if out is None else out
        _check(_L.dg4_rhs(self._h, _ptr(f), _ptr(Ex), _ptr(Ey), _ptr(out), _stream(self.device)), "dg4_rhs")
        return out

    def rk_stage(self, f_s, f_n, Ex, Ey, out, c0, c1, dt, rho_out=None):
        _check(_L.dg4_rk_stage(self._h, _ptr(f_s), _ptr(f_n), _ptr(Ex), _ptr(Ey), _ptr(out), float(c0), float(c1), float(dt),
                               _ptr(rho_out), _stream(self.device)), "dg4_rk_stage")
        return out

    def set_xhalo(self, halo):
        """halo: [2][G_y][G_u][G_v] exterior x-face planes of an x-slab context (bc[0] = BC_HALO); kept alive here."""
        self._xhalo = halo
        _check(_L.dg4_set_xhalo(self._h, _ptr(halo)), "dg4_set_xhalo")

    def density(self, f, out=None):
        out = self._field() if out is None else out
        _check(_L.dg4_density(self._h, _ptr(f), _ptr(out), _stream(self.device)), "dg4_density")
        return out

    def fourier_project(self, rho, out=None):
        out = torch.empty((self.pmax[0] + 1, 2 * self.pmax[1] + 1, 2), dtype=torch.float64, device=self.device) if out is None else out
        _check(_L.dg4_fourier_project(self._h, _ptr(rho), _ptr(out), _stream(self.device)), "dg4_fourier_project")
        return out

    def poisson_E(self, rho, Ex=None, Ey=None):
        Ex = self._field() if Ex is None else Ex
        Ey = self._field() if Ey is None else Ey
        _check(_L.dg4_poisson_E(self._h, _ptr(rho), _ptr(Ex), _ptr(Ey), _stream(self.device)), "dg4_poisson_E")
        return Ex, Ey

    def ssprk3_run(self, f, dt, nsteps, self_consistent=True):
        _check(_L.dg4_ssprk3_run(self._h, _ptr(f), float(dt), int(nsteps), int(bool(self_consistent)), _stream(self.device)), "dg4_ssprk3_run")
        return f

    def ssprk3_run_host(self, f_host, dt, nsteps, self_consistent=True):
        p = f_host.ctypes.data if isinstance(f_host, np.ndarray) else f_host.data_ptr()
        _check(_L.dg4_ssprk3_run_host(self._h, p, float(dt), int(nsteps), int(bool(self_consistent))), "dg4_ssprk3_run_host")
        return f_host

    def nodes(self, dim):
        x = np.empty(self.flat_shape[dim])
        _check(_L.dg4_get_nodes(self._h, dim, x.ctypes.data_as(C.POINTER(C.c_double))), "dg4_get_nodes")
        return x

    def max_stable_dt(self, E_bound=0.0):
        return float(_L.dg4_max_stable_dt(self._h, float(E_bound)))

    def set_option(self, key, value):
        _check(_L.dg4_set_option(self._h, int(key), int(value)), "dg4_set_option")

    def get_profile(self, reset=True):
        ms, cnt = C.c_double(0.0), C.c_int64(0)
        _check(_L.dg4_get_profile(self._h, C.byref(ms), C.byref(cnt), int(bool(reset))), "dg4_get_profile")
        return ms.value, cnt.value

    @property
    def launch_count(self):
        return int(_L.dg4_launch_count(self._h))

    @property
    def last_kernel(self):
        return _L.dg4_last_kernel(self._h).decode()


class DGNContext:
    """Dimension-generic variant (include/dgvlasov_nd.h): dgn_create / dgn_destroy plus one method per C entry point.
    Phase space (x_1..x_dx, v_1..v_dv), 1 <= dx <= dv <= 3; f: [G_x1]..[G_vdv]; E: [dx][G_x1]..[G_xdx]; rho: [G_x1]..[G_xdx]."""

    def __init__(self, dx, dv, nelem, order, lo, hi, bc=None, omega_c=0.0, pmax=None, mass_mode=0, device=0, workspace=True):
        nd = dx + dv
        if bc is None:
            bc = (0,) * dx + (1,) * dv
        pmax = tuple(pmax) if pmax is not None else (0,) * dx
        d = _lib.GridDescN()
        d.dx, d.dv = int(dx), int(dv)
        for i in range(nd):
            d.nelem[i], d.order[i], d.lo[i], d.hi[i], d.bc[i] = int(nelem[i]), int(order[i]), float(lo[i]), float(hi[i]), int(bc[i])
        for i in range(dx):
            d.pmax[i] = int(pmax[i])
        d.omega_c, d.mass_mode, d.device = float(omega_c), int(mass_mode), int(device)
        self._h = C.c_void_p()
        _check(_L.dgn_create(C.byref(d), C.byref(self._h)), "dgn_create")
        self.dx, self.dv, self.ndim = int(dx), int(dv), nd
        self.nelem, self.order = tuple(nelem), tuple(order)
        self.device = torch.device("cuda", device)
        self.flat_shape = tuple(int(nelem[i]) * int(order[i]) for i in range(nd))
        self._ws = None
        if workspace:
            nbytes = _L.dgn_workspace_bytes(self._h)
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self._ws.data_ptr() + 255) // 256 * 256
            _check(_L.dgn_set_workspace(self._h, base, nbytes), "dgn_set_workspace")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            _L.dgn_destroy(self._h)
            self._h = C.c_void_p()
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def rhs(self, f, E=None, out=None):
        out = torch.empty_like(f) if out is None else out
        _check(_L.dgn_rhs(self._h, _ptr(f), _ptr(E), _ptr(out), _stream(self.device)), "dgn_rhs")
        return out

    def rk_stage(self, f_s, f_n, E, out, c0, c1, dt):
        _check(_L.dgn_rk_stage(self._h, _ptr(f_s), _ptr(f_n), _ptr(E), _ptr(out), float(c0), float(c1), float(dt),
                               _stream(self.device)), "dgn_rk_stage")
        return out

    def density(self, f, out=None):
        out = torch.empty(self.flat_shape[:self.dx], dtype=torch.float64, device=self.device) if out is None else out
        _check(_L.dgn_density(self._h, _ptr(f), _ptr(out), _stream(self.device)), "dgn_density")
        return out

    def poisson_E(self, rho, out=None):
        out = torch.empty((self.dx,) + self.flat_shape[:self.dx], dtype=torch.float64, device=self.device) if out is None else out
        _check(_L.dgn_poisson_E(self._h, _ptr(rho), _ptr(out), _stream(self.device)), "dgn_poisson_E")
        return out

    def ssprk3_run(self, f, dt, nsteps, self_consistent=True):
        _check(_L.dgn_ssprk3_run(self._h, _ptr(f), float(dt), int(nsteps), int(bool(self_consistent)), _stream(self.device)), "dgn_ssprk3_run")
        return f

    def nodes(self, dim):
        x = np.empty(self.flat_shape[dim])
        _check(_L.dgn_get_nodes(self._h, dim, x.ctypes.data_as(C.POINTER(C.c_double))), "dgn_get_nodes")
        return x

    @property
    def launch_count(self):
        return int(_L.dgn_launch_count(self._h))
