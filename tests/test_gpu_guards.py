"""Out-of-bounds and race evidence without compute-sanitizer (which this GPU pool has closed -- profiles/r2_sanitizers.md):

  * every caller-owned array a kernel writes (out, rho, E, c, the workspace) and reads sits between two guard bands filled with a
    canary bit pattern (a NaN payload no kernel can produce); after the call the bands must be bit-identical -- a store one
    element past either end of any array, or into a neighbouring array, fails the test;
  * outputs are pre-filled with the canary: a node the kernel never wrote keeps it and fails the finiteness check;
  * every call is made twice on fresh output buffers and the two results must be bit-identical -- the kernels are designed
    to be deterministic (fixed-order reductions, no atomics), so an unsynchronised shared-memory hazard or a read of a halo
    that a TMA load had not delivered yet shows up as run-to-run noise.

Sizes are chosen with ragged tile tails (element counts that are not multiples of the tile widths) and every boundary kind."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import workloads as wl  # noqa: E402

CANARY = np.array([0x7FF8DEADBEEFCAFE], dtype=np.uint64).view(np.int64)[0]
GUARD = 512                      # doubles on either side (4 KB): wider than any row or halo the kernels handle
K = 0.1


def api():
    from paper_2202_13532_b200 import api as _api
    return _api


class Guarded:
    """A float64 CUDA array of `shape` between two canary bands, the payload 256-byte aligned."""

    def __init__(self, shape, fill=None):
        n = int(np.prod(shape))
        self.n, self.shape = n, tuple(shape)
        self.raw = torch.empty(n + 2 * GUARD + 32, dtype=torch.int64, device="cuda")
        self.raw.fill_(int(CANARY))
        off = GUARD + ((-(self.raw.data_ptr() // 8 + GUARD)) % 32)
        self.off = off
        self.view = self.raw[off:off + n].view(torch.float64).view(self.shape)
        assert self.view.data_ptr() % 256 == 0
        if fill is not None:
            self.view.copy_(torch.from_numpy(np.ascontiguousarray(fill, dtype=np.float64)).cuda())

    def guards_intact(self):
        lo, hi = self.raw[:self.off], self.raw[self.off + self.n:]
        return bool((lo == int(CANARY)).all().item()) and bool((hi == int(CANARY)).all().item())

    def fully_written(self):
        return bool(torch.isfinite(self.view).all().item())


def check(arrays, what):
    torch.cuda.synchronize()
    for name, a in arrays.items():
        assert a.guards_intact(), f"{what}: guard band of {name} overwritten"


def twice(fn, what):
    """fn() -> dict of Guarded outputs; runs it twice and demands bit-identical, fully written outputs with intact guards."""
    a, b = fn(), fn()
    check(a, what)
    check(b, what)
    for name in a:
        assert a[name].fully_written(), f"{what}: {name} has unwritten or non-finite entries"
        assert torch.equal(a[name].view.view(torch.int64), b[name].view.view(torch.int64)), f"{what}: {name} differs between two runs"


def guarded_workspace(ctx, A, batch=1):
    nbytes = A._L.dg_field_workspace_bytes(ctx._h, batch)
    ws = Guarded(((nbytes + 7) // 8,))
    A._check(A._L.dg_set_workspace(ctx._h, ws.view.data_ptr(), nbytes), "dg_set_workspace")
    return ws


RHS_GRIDS = [
    # nelem, order, bc (ragged v tails for every tile width: KV = 8, 8, 4, 2)
    ((3, 3, 11), (4, 4, 4), (0, 1, 1)),
    ((2, 3, 5), (6, 6, 6), (0, 0, 1)),
    ((3, 2, 7), (8, 8, 8), (0, 1, 1)),
    ((2, 2, 7), (8, 8, 8), (1, 0, 0)),
    ((2, 2, 3), (10, 10, 10), (0, 1, 0)),
    ((3, 2, 4), (3, 5, 4), (0, 1, 1)),          # generic kernel
]


@pytest.mark.parametrize("nelem,order,bc", RHS_GRIDS)
@pytest.mark.parametrize("form", [0, 1])
def test_rhs_and_stage_stay_inside_their_arrays(nelem, order, bc, form):
    A = api()
    lo, hi = (0.0, -4.0, -3.0), (2 * math.pi / K, 4.0, 5.0)
    ctx = A.DGContext(nelem, order, lo, hi, bc=bc, omega_c=0.8, pmax=2, workspace=False)
    ws = guarded_workspace(ctx, A)
    ctx.set_option(A.OPT_FORM, form)
    shape = ctx.flat_shape
    f = Guarded(shape, wl.uniform_field(shape, 7))
    fn = Guarded(shape, wl.uniform_field(shape, 8))
    E = Guarded((shape[0],), 0.7 * wl.normal_E(shape[0], 9))

    def run_rhs():
        out = Guarded(shape)
        ctx.rhs(f.view, E.view, out.view)
        return {"out": out}

    def run_stage():
        out, rho = Guarded(shape), Guarded((shape[0],))
        ctx.rk_stage(f.view, fn.view, E.view, out.view, 0.75, 0.25, 1e-3, rho_out=rho.view)
        return {"out": out, "rho": rho}

    twice(run_rhs, f"dg_rhs {ctx.last_kernel}")
    twice(run_stage, f"dg_rk_stage {ctx.last_kernel}")
    check({"f": f, "fn": fn, "E": E, "workspace": ws}, "inputs / workspace")
    ctx.close()


def test_run_in_place_and_xslab_push_stay_inside():
    A = api()
    from paper_2202_13532_b200 import sharded
    nelem, order = (3, 2, 5), (8, 8, 8)
    lo, hi = (0.0, -8.5, -8.5), (2 * math.pi / K, 8.5, 8.5)
    ctx = A.DGContext(nelem, order, lo, hi, bc=(0, 1, 1), omega_c=1.0, pmax=3, workspace=False)
    ws = guarded_workspace(ctx, A)
    f0 = wl.add_uniform_noise(wl.ring_f0(ctx.nodes(0), ctx.nodes(1), ctx.nodes(2), K), wl.SEED_CFG3_NOISE, 1e-4)

    def run():
        f = Guarded(ctx.flat_shape, f0)
        ctx.ssprk3_run(f.view, 1e-3, 3, True)
        return {"f": f}

    twice(run, "dg_ssprk3_run")
    check({"workspace": ws}, "dg_ssprk3_run")
    ctx.close()

    # x-slab context: exterior planes from a halo buffer, boundary planes of out pushed into two guarded planes
    slab = A.DGContext(nelem, order, lo, hi, bc=(A.BC_HALO, 1, 1), omega_c=1.0, pmax=3, workspace=False)
    ws2 = guarded_workspace(slab, A)
    G = slab.flat_shape
    halo = Guarded((2, G[1], G[2]), wl.uniform_field((2, G[1], G[2]), 21))
    slab.set_xhalo(halo.view)
    fs, fn = Guarded(G, wl.uniform_field(G, 22)), Guarded(G, wl.uniform_field(G, 23))
    E = Guarded((G[0],), 0.3 * wl.normal_E(G[0], 24))

    def run_push():
        out, left, right = Guarded(G), Guarded((G[1], G[2])), Guarded((G[1], G[2]))
        slab.set_xhalo_push(left.view, right.view)
        slab.rk_stage(fs.view, fn.view, E.view, out.view, 1.0 / 3.0, 2.0 / 3.0, 1e-3)
        torch.cuda.synchronize()
        assert torch.equal(left.view, out.view[0]) and torch.equal(right.view, out.view[-1])
        return {"out": out, "left": left, "right": right}

    twice(run_push, "dg_rk_stage with face push")
    check({"halo": halo, "fs": fs, "fn": fn, "E": E, "workspace": ws2}, "x-slab inputs")
    slab.set_xhalo_push(None, None)
    slab.close()
    assert sharded is not None


@pytest.mark.parametrize("N,n,pmax,batch", [(16, 8, 40, 5), (64, 4, 64, 19), (12, 6, 9, 3)])
def test_field_kernels_stay_inside(N, n, pmax, batch):
    A = api()
    ctx = A.DGContext((N,), (n,), (0.0,), (2 * math.pi,), pmax=pmax, workspace=False)
    ws = guarded_workspace(ctx, A, batch)
    x = ctx.nodes(0)
    rho_h, _, _, _ = wl.cosine_sum_density(x, batch, wl.SEED_CFG5, mmax=max(2, N // 4))
    rho = Guarded(rho_h.shape, rho_h)
    kinds = [A.FIELD_SIMPLE, A.FIELD_DMMA, A.FIELD_DFMA] + ([A.FIELD_FFT] if (N & (N - 1)) == 0 and n % 2 == 0 else [])
    for fk in kinds:
        ctx.set_option(A.OPT_FIELD_KERNEL, fk)

        def run():
            E, c, phi = Guarded(rho_h.shape), Guarded((batch, pmax + 1, 2)), Guarded(rho_h.shape)
            ctx.poisson_E(rho.view, E.view)
            ctx.fourier_project(rho.view, c.view)
            ctx.poisson_phi(rho.view, phi.view)
            return {"E": E, "c": c, "phi": phi}

        twice(run, f"field kernel {fk} ({ctx.last_field_kernel})")
    check({"rho": rho, "workspace": ws}, "field inputs / workspace")
    ctx.close()


@pytest.mark.parametrize("nelem,n", [((2, 3, 2, 8), 4), ((3, 2, 2, 6), 4), ((2, 2, 3, 2), 6), ((2, 3, 2, 2), 8), ((2, 2, 2, 3), 5)])
def test_2d2v_kernels_stay_inside(nelem, n):
    A = api()
    lo, hi = (0.0, 0.0, -8.5, -8.5), (2 * math.pi / K, 2 * math.pi / K, 8.5, 8.5)
    ctx = A.DG4Context(nelem, (n,) * 4, lo, hi, bc=(0, 0, 1, 1), omega_c=1.0, workspace=False)
    nbytes = A._L.dg4_workspace_bytes(ctx._h)
    ws = Guarded(((nbytes + 7) // 8,))
    A._check(A._L.dg4_set_workspace(ctx._h, ws.view.data_ptr(), nbytes), "dg4_set_workspace")
    G = ctx.flat_shape
    x, y, u, v = (ctx.nodes(d) for d in range(4))
    f0 = wl.add_uniform_noise(wl.ring2d_f0(x, y, u, v, K, K), wl.SEED_CFG6_NOISE, 1e-4)
    f = Guarded(G, f0)
    fn = Guarded(G, wl.uniform_field(G, 31))
    Ex, Ey = Guarded(G[:2], 0.2 * wl.uniform_field(G[:2], 32) - 0.1), Guarded(G[:2], 0.2 * wl.uniform_field(G[:2], 33) - 0.1)

    def run_rhs():
        out = Guarded(G)
        ctx.rhs(f.view, Ex.view, Ey.view, out.view)
        return {"out": out}

    def run_stage():
        out, rho = Guarded(G), Guarded(G[:2])
        ctx.rk_stage(f.view, fn.view, Ex.view, Ey.view, out.view, 0.75, 0.25, 2e-4, rho_out=rho.view)
        return {"out": out, "rho": rho}

    def run_steps():
        g = Guarded(G, f0)
        ctx.ssprk3_run(g.view, 2e-4, 2)
        return {"f": g}

    twice(run_rhs, f"dg4_rhs {ctx.last_kernel}")
    twice(run_stage, f"dg4_rk_stage {ctx.last_kernel}")
    twice(run_steps, "dg4_ssprk3_run")
    check({"f": f, "fn": fn, "Ex": Ex, "Ey": Ey, "workspace": ws}, "2D2V inputs / workspace")
    ctx.close()


@pytest.mark.parametrize("dx,dv,nelem,order", [(1, 3, (3, 2, 2, 2), (3, 4, 3, 3)), (2, 3, (2, 2, 2, 2, 2), (3, 3, 3, 2, 3)),
                                               (3, 3, (2, 1, 2, 2, 2, 1), (2, 4, 2, 3, 2, 4))])
def test_dimension_generic_kernels_stay_inside(dx, dv, nelem, order):
    A = api()
    nd = dx + dv
    lo = (0.0,) * dx + (-2.0,) * dv
    hi = tuple(1.0 + 0.5 * i for i in range(dx)) + (2.0,) * dv
    ctx = A.DGNContext(dx, dv, nelem, order, lo, hi, omega_c=0.9, pmax=(2,) * dx, workspace=False)
    nbytes = A._L.dgn_workspace_bytes(ctx._h)
    ws = Guarded(((nbytes + 7) // 8,))
    A._check(A._L.dgn_set_workspace(ctx._h, ws.view.data_ptr(), nbytes), "dgn_set_workspace")
    G = ctx.flat_shape
    f0 = 0.5 + wl.uniform_field(G, 51)
    f, fn = Guarded(G, f0), Guarded(G, wl.uniform_field(G, 52))
    E = Guarded((dx,) + G[:dx], 0.4 * wl.uniform_field((dx,) + G[:dx], 53) - 0.2)

    def run():
        out, st, rho, Eo = Guarded(G), Guarded(G), Guarded(G[:dx]), Guarded((dx,) + G[:dx])
        ctx.rhs(f.view, E.view, out.view)
        ctx.rk_stage(f.view, fn.view, E.view, st.view, 0.75, 0.25, 1e-3)
        ctx.density(f.view, rho.view)
        ctx.poisson_E(rho.view, Eo.view)
        g = Guarded(G, f0)
        ctx.ssprk3_run(g.view, 1e-3, 2, True)
        return {"out": out, "stage": st, "rho": rho, "E": Eo, "f": g}

    twice(run, f"dgn_* {dx}D{dv}V")
    check({"f": f, "fn": fn, "E": E, "workspace": ws}, "dgn inputs / workspace")
    assert nd == len(G)
    ctx.close()
