"""ctypes loader for libdgvlasov.so -- the C ABI declared in include/dgvlasov.h, include/dgvlasov2d2v.h, include/dgvlasov_nd.h and
include/dgvlasov_noalloc.h.

There is no fallback: if the library has not been built (python -m paper_2202_13532_b200.build)
importing the binding raises."""
from __future__ import annotations

import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
# DGVLASOV_LIB: another build of the same library (kernel A/B comparisons); default: the in-tree build
LIB_PATH = os.environ.get("DGVLASOV_LIB") or os.path.join(HERE, "libdgvlasov.so")


class GridDesc(C.Structure):
    _fields_ = [
        ("ndim", C.c_int32),
        ("nelem", C.c_int32 * 3),
        ("order", C.c_int32 * 3),
        ("lo", C.c_double * 3),
        ("hi", C.c_double * 3),
        ("bc", C.c_int32 * 3),
        ("omega_c", C.c_double),
        ("pmax", C.c_int32),
        ("mass_mode", C.c_int32),
        ("device", C.c_int32),
    ]


class GridDesc4(C.Structure):
    """dg4_grid_desc of include/dgvlasov2d2v.h."""
    _fields_ = [
        ("nelem", C.c_int32 * 4),
        ("order", C.c_int32 * 4),
        ("lo", C.c_double * 4),
        ("hi", C.c_double * 4),
        ("bc", C.c_int32 * 4),
        ("omega_c", C.c_double),
        ("pmax", C.c_int32 * 2),
        ("mass_mode", C.c_int32),
        ("device", C.c_int32),
    ]


class GridDescN(C.Structure):
    """dgn_grid_desc of include/dgvlasov_nd.h."""
    _fields_ = [
        ("dx", C.c_int32),
        ("dv", C.c_int32),
        ("nelem", C.c_int32 * 6),
        ("order", C.c_int32 * 6),
        ("lo", C.c_double * 6),
        ("hi", C.c_double * 6),
        ("bc", C.c_int32 * 6),
        ("omega_c", C.c_double),
        ("pmax", C.c_int32 * 3),
        ("mass_mode", C.c_int32),
        ("device", C.c_int32),
    ]


_vp, _dp, _i32, _i64, _dbl = C.c_void_p, C.POINTER(C.c_double), C.c_int32, C.c_int64, C.c_double

# name -> (restype, argtypes); must list every symbol include/dgvlasov.h declares
SIGNATURES = {
    "dg_create": (C.c_int, [C.POINTER(GridDesc), C.POINTER(_vp)]),
    "dg_destroy": (C.c_int, [_vp]),
    "dg_create_field_nonuniform": (C.c_int, [_dp, _i32, _i32, _i32, _i32, C.POINTER(_vp)]),
    "dg_workspace_bytes": (C.c_size_t, [_vp]),
    "dg_field_workspace_bytes": (C.c_size_t, [_vp, _i32]),
    "dg_set_workspace": (C.c_int, [_vp, _vp, C.c_size_t]),
    "dg_rhs": (C.c_int, [_vp, _vp, _vp, _vp, _vp]),
    "dg_ssprk3_step": (C.c_int, [_vp, _vp, _dbl, _i32, _vp]),
    "dg_ssprk3_run": (C.c_int, [_vp, _vp, _dbl, _i32, _i32, _vp]),
    "dg_ssprk3_run_host": (C.c_int, [_vp, _vp, _dbl, _i32, _i32]),
    "dg_set_xhalo": (C.c_int, [_vp, _vp]),
    "dg_set_xhalo_push": (C.c_int, [_vp, _vp, _vp]),
    "dg_rk_stage": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _dbl, _dbl, _dbl, _vp, _vp]),
    "dg_density": (C.c_int, [_vp, _vp, _vp, _vp]),
    "dg_fourier_project": (C.c_int, [_vp, _vp, _i32, _vp, _vp]),
    "dg_poisson_E": (C.c_int, [_vp, _vp, _i32, _vp, _vp]),
    "dg_poisson_phi": (C.c_int, [_vp, _vp, _i32, _vp, _vp]),
    "dg_broken_l2": (C.c_int, [_vp, _vp, _vp, _i32, _vp, _vp]),
    "dg_get_operators": (C.c_int, [_vp, _i32, _dp, _dp, _dp, _dp]),
    "dg_get_nodes": (C.c_int, [_vp, _i32, _dp]),
    "dg_get_dmatrix": (C.c_int, [_vp, _i32, _dp]),
    "dg_get_transform": (C.c_int, [_vp, _i32, _i32, _dp]),
    "dg_max_stable_dt": (_dbl, [_vp, _dbl]),
    "dg_set_option": (C.c_int, [_vp, _i32, _i64]),
    "dg_get_profile": (C.c_int, [_vp, _dp, C.POINTER(_i64), _i32]),
    "dg_get_profile_stages": (C.c_int, [_vp, _dp, C.POINTER(_i64), _i32]),
    "dg_ssprk3_stage_coeffs": (C.c_int, [_i32, _dp, _dp]),
    "dg_check_finite": (C.c_int, [_vp, _vp, _vp, _vp]),
    "dg_fp64_peak": (C.c_int, [_i32, _i32, _i32, _dp]),
    "dg_launch_count": (_i64, [_vp]),
    "dg_last_kernel": (C.c_char_p, [_vp]),
    "dg_last_field_kernel": (C.c_char_p, [_vp]),
    "dg_last_error": (C.c_char_p, []),
    "dg_version": (C.c_char_p, []),
    "dg_field_energy": (C.c_int, [_vp, _vp, _i32, _vp, _vp]),
    # include/dgvlasov_noalloc.h
    "dg_density_static": (C.c_int, [_vp, _i32, _i32, _i32, _vp, _vp, _vp, _i32, _vp]),
    # include/dgvlasov2d2v.h
    "dg4_create": (C.c_int, [C.POINTER(GridDesc4), C.POINTER(_vp)]),
    "dg4_destroy": (C.c_int, [_vp]),
    "dg4_workspace_bytes": (C.c_size_t, [_vp]),
    "dg4_set_workspace": (C.c_int, [_vp, _vp, C.c_size_t]),
    "dg4_rhs": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _vp]),
    "dg4_rk_stage": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _vp, _dbl, _dbl, _dbl, _vp, _vp]),
    "dg4_set_xhalo": (C.c_int, [_vp, _vp]),
    "dg4_density": (C.c_int, [_vp, _vp, _vp, _vp]),
    "dg4_fourier_project": (C.c_int, [_vp, _vp, _vp, _vp]),
    "dg4_poisson_E": (C.c_int, [_vp, _vp, _vp, _vp, _vp]),
    "dg4_ssprk3_run": (C.c_int, [_vp, _vp, _dbl, _i32, _i32, _vp]),
    "dg4_ssprk3_run_host": (C.c_int, [_vp, _vp, _dbl, _i32, _i32]),
    "dg4_get_nodes": (C.c_int, [_vp, _i32, _dp]),
    "dg4_max_stable_dt": (_dbl, [_vp, _dbl]),
    "dg4_set_option": (C.c_int, [_vp, _i32, _i64]),
    "dg4_get_profile": (C.c_int, [_vp, _dp, C.POINTER(_i64), _i32]),
    "dg4_launch_count": (_i64, [_vp]),
    "dg4_last_kernel": (C.c_char_p, [_vp]),
    "dgn_create": (C.c_int, [C.POINTER(GridDescN), C.POINTER(_vp)]),
    "dgn_destroy": (C.c_int, [_vp]),
    "dgn_workspace_bytes": (C.c_size_t, [_vp]),
    "dgn_set_workspace": (C.c_int, [_vp, _vp, C.c_size_t]),
    "dgn_rhs": (C.c_int, [_vp, _vp, _vp, _vp, _vp]),
    "dgn_rk_stage": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _dbl, _dbl, _dbl, _vp]),
    "dgn_density": (C.c_int, [_vp, _vp, _vp, _vp]),
    "dgn_poisson_E": (C.c_int, [_vp, _vp, _vp, _vp]),
    "dgn_ssprk3_run": (C.c_int, [_vp, _vp, _dbl, _i32, _i32, _vp]),
    "dgn_get_nodes": (C.c_int, [_vp, _i32, _dp]),
    "dgn_launch_count": (_i64, [_vp]),
}


def load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2202_13532_b200.build` "
            "(there is no CPU or PyTorch fallback for the DG kernels)")
    lib = C.CDLL(LIB_PATH)
    for name, (res, args) in SIGNATURES.items():
        fn = getattr(lib, name)          # AttributeError if the symbol is not exported
        fn.restype = res
        fn.argtypes = args
    return lib
