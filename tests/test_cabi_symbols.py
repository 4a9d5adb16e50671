"""CPU checks of the boundary: the library builds, loads and exports every symbol the header declares."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = "".join(open(os.path.join(ROOT, "include", h)).read() for h in sorted(os.listdir(os.path.join(ROOT, "include"))))
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dg[4n]?_[A-Za-z0-9_]+)\s*\(", text)))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2202_13532_b200 import build, _lib
    path = build.build()
    lib = ctypes.CDLL(path)
    declared = _declared_symbols()
    assert len(declared) >= 18
    for name in declared:
        assert hasattr(lib, name), name
        assert name in _lib.SIGNATURES, f"binding has no signature for {name}"
    assert set(_lib.SIGNATURES) == set(declared)


def test_binding_loads_without_gpu_and_reports_errors():
    from paper_2202_13532_b200 import _lib
    lib = _lib.load()
    assert b"sm_100a" in lib.dg_version()
    # argument validation happens before any CUDA call
    assert lib.dg_create(None, None) == -1
    assert b"null" in lib.dg_last_error()
    d = _lib.GridDesc()
    d.ndim = 7
    h = ctypes.c_void_p()
    assert lib.dg_create(ctypes.byref(d), ctypes.byref(h)) == -1
    d.ndim = 2
    d.nelem[0], d.nelem[1] = 4, 4
    d.order[0], d.order[1] = 4, 11
    d.hi[0], d.hi[1] = 1.0, 1.0
    assert lib.dg_create(ctypes.byref(d), ctypes.byref(h)) == -2      # DG_ERR_UNSUPPORTED: order > 10


def test_2d2v_argument_validation_without_gpu():
    from paper_2202_13532_b200 import _lib
    lib = _lib.load()
    h = ctypes.c_void_p()
    assert lib.dg4_create(None, ctypes.byref(h)) == -1
    d = _lib.GridDesc4()
    for i in range(4):
        d.nelem[i], d.order[i], d.lo[i], d.hi[i] = 2, 4, 0.0, 1.0
    d.order[3] = 11
    assert lib.dg4_create(ctypes.byref(d), ctypes.byref(h)) == -2      # DG_ERR_UNSUPPORTED: order > 10
    d.order[3] = 4
    d.bc[2] = 2
    assert lib.dg4_create(ctypes.byref(d), ctypes.byref(h)) == -1      # no halo boundary in the 2D2V context
    assert b"bc" in lib.dg_last_error()
    assert lib.dg4_workspace_bytes(None) == 0 and lib.dg4_launch_count(None) == 0
    assert lib.dg4_rhs(None, None, None, None, None, None) == -1


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2202_13532_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".cpp", ".hpp", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in src and "from oracle" not in src and "oracle/" not in src, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith(".py"):
            assert "paper_2202_13532_b200" not in open(os.path.join(ROOT, "oracle", fn)).read().replace(
                "(paper_2202_13532_b200/)", "").replace("paper_2202_13532_b200/ (the CUDA path)", ""), fn
