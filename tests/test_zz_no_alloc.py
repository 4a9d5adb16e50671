"""dg_density_static (include/dgvlasov_noalloc.h): the allocation-free density call.

Some users of the library cannot allocate device memory at the place where they need a density: a diagnostics hook
inside another code's time loop that has already given all of the HBM to its own pool, a latency-critical callback that
cannot take the device-wide stall of a cudaMalloc, a process under a fixed MPS / MIG memory quota.  For them the library
has one call that takes only inputs and the output and keeps its partial sums in a 2 MiB array compiled into the
library.  Because every call on a device shares that array and it is never cleared, the thing to test is two calls in a
row with different data and different shapes: the second must not see anything of the first.

The reference here is the library's existing path (dg_density, partial sums in the caller's workspace), at the tolerance
the density parity tests use (1e-13, max norm, relative); the oracle is checked as a second opinion.

This file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide other tests)."""
import ctypes

import numpy as np
import pytest

import workloads as wl                                                          # noqa: E402

TOL = 1e-13       # tests/test_gpu_parity.py::test_density_matches_oracle


def relerr(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


def _node_weights(ctx, dim, lo, hi):
    """Quadrature weight of every flat node of dimension `dim`: w_b * (Delta / 2), from the library's own LGL weights."""
    _, w, _, _ = ctx.operators(dim)
    N = ctx.nelem[dim]
    return np.tile(w * (0.5 * (hi - lo) / N), N)


# (nelem, order, lo, hi): a ragged 1D2V grid, a smaller one with an odd G_v (scalar-load variant), a 1D1V grid
SHAPES = [
    ((12, 9, 10), (8, 8, 8), (0.0, -8.5, -8.5), (20 * np.pi, 8.5, 8.5)),
    ((5, 4, 3), (4, 6, 5), (0.0, -2.0, -3.0), (3.0, 2.5, 3.0)),
    ((16, 32), (4, 4), (0.0, -6.0), (4 * np.pi, 6.0)),
]


@pytest.mark.gpu
def test_static_density_matches_workspace_path_on_consecutive_calls():
    torch = pytest.importorskip("torch")
    from paper_2202_13532_b200 import api
    from oracle import vlasov as ov
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    # Large first, small second, large again: after call 1 the shared scratch is full of call 1's partial sums, so a
    # call that read a slot it had not written itself would pick them up.
    for k, (nelem, order, lo, hi) in enumerate([SHAPES[0], SHAPES[1], SHAPES[0], SHAPES[2]]):
        bc = (0,) + (1,) * (len(nelem) - 1)
        g = ov.Grid(nelem=nelem, order=order, lo=lo, hi=hi, bc=bc)
        ctx = api.DGContext(nelem, order, lo, hi, bc=bc)
        f = wl.uniform_field(g.flat_shape, 11 + k) - 0.25
        f_d = dev(f)
        wq_u = dev(_node_weights(ctx, 1, lo[1], hi[1]))
        wq_v = dev(_node_weights(ctx, 2, lo[2], hi[2])) if len(nelem) == 3 else None
        want = ctx.density(f_d).cpu().numpy()                        # existing path: partials in the workspace
        out = torch.full((g.flat_shape[0],), float("nan"), dtype=torch.float64, device="cuda")
        got1 = api.density_static(f_d, wq_u, wq_v, out).cpu().numpy().copy()
        out.fill_(float("nan"))
        got2 = api.density_static(f_d, wq_u, wq_v, out).cpu().numpy()        # straight after, same stream
        assert relerr(got1, want) <= TOL, (k, relerr(got1, want))
        assert np.array_equal(got1, got2), k                         # deterministic, nothing left over between calls
        assert relerr(got1, ov.density(g, f)) <= TOL, k
        ctx.close()


@pytest.mark.gpu
def test_static_density_at_the_size_limit_and_beyond():
    torch = pytest.importorskip("torch")
    from paper_2202_13532_b200 import api
    G_x, G_u, G_v = api.STATIC_MAX_GX, 24, 6                        # the most x nodes the built-in scratch serves
    f = torch.from_numpy(wl.uniform_field((G_x, G_u, G_v), 3)).cuda()
    wq_u = torch.linspace(0.5, 1.5, G_u, dtype=torch.float64, device="cuda")
    wq_v = torch.linspace(0.25, 0.75, G_v, dtype=torch.float64, device="cuda")
    out = torch.empty(G_x, dtype=torch.float64, device="cuda")
    api.density_static(f, wq_u, wq_v, out)
    want = torch.einsum("xuv,u,v->x", f, wq_u, wq_v)                 # plain definition of the weighted sum
    assert relerr(out.cpu().numpy(), want.cpu().numpy()) <= TOL
    big = torch.empty((G_x + 1, 1, 2), dtype=torch.float64, device="cuda")
    with pytest.raises(api.DGError, match="DG_STATIC_MAX_GX"):
        api.density_static(big, wq_u[:1], wq_v[:2], torch.empty(G_x + 1, dtype=torch.float64, device="cuda"))


def test_static_density_rejects_bad_arguments_without_a_gpu():
    """Argument checks come before any CUDA call, so they can be exercised on a box without a device."""
    from paper_2202_13532_b200 import _lib
    lib = _lib.load()
    p = ctypes.c_void_p(256)                                          # never dereferenced: the call is refused first
    assert lib.dg_density_static(None, 4, 4, 4, p, p, p, 0, None) == -1
    assert lib.dg_density_static(p, 4, 0, 4, p, p, p, 0, None) == -1
    assert lib.dg_density_static(p, 4, 4, 4, p, None, p, 0, None) == -1      # wq_v may be NULL only for G_v = 1
    assert lib.dg_density_static(p, 16385, 4, 4, p, p, p, 0, None) == -2
    assert b"DG_STATIC_MAX_GX = 16384" in lib.dg_last_error()
