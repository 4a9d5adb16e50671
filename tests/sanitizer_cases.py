"""Small cases for compute-sanitizer (memcheck / racecheck / synccheck), one process, through the C ABI:

    compute-sanitizer --tool memcheck python tests/sanitizer_cases.py [case ...]

Cases: config1 (generic kernel, 1D1V), tiled (2x2x2 elements, n = 8, dg_ssprk3_run with
the one-launch field solve, programmatic launches on and off), xslab (halo context + face push on one device), 2d2v (2x2x2x8
elements, n = 4, one step; 2x2x2x2, n = 8), field (dense DMMA / DFMA / FFT-factorised projection and Poisson solve).
Each case also checks its result against the oracle so that a 'clean' report is about a correct run."""
import math
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import numpy as np                       # noqa: E402
import torch                             # noqa: E402

from oracle import vlasov as ov, vlasov2d2v as o4, fourier as ofr      # noqa: E402
import workloads as wl                   # noqa: E402
from paper_2202_13532_b200 import api, sharded      # noqa: E402

K = 0.1


def relerr(a, b):
    return float(np.max(np.abs(np.asarray(a) - np.asarray(b))) / max(np.max(np.abs(b)), 1e-300))


def case_config1():
    nelem, order, lo, hi = (16, 32), (4, 4), (0.0, -6.0), (4 * math.pi, 6.0)
    ctx = api.DGContext(nelem, order, lo, hi, bc=(0, 1), pmax=16)
    g = ov.Grid(nelem=nelem, order=order, lo=lo, hi=hi, bc=(0, 1), pmax=16)
    f0 = wl.landau_f0(ctx.nodes(0), ctx.nodes(1))
    f = torch.from_numpy(f0).cuda()
    ctx.ssprk3_run(f, 0.01, 2, True)
    fo = ov.ssprk3_step(g, ov.ssprk3_step(g, f0, 0.01), 0.01)
    ctx.close()
    return relerr(f.cpu().numpy(), fo)


def case_tiled():
    nelem, order = (2, 2, 2), (8, 8, 8)
    lo, hi = (0.0, -8.5, -8.5), (2 * math.pi / K, 8.5, 8.5)
    g = ov.Grid(nelem=nelem, order=order, lo=lo, hi=hi, bc=(0, 1, 1), omega_c=1.0, pmax=2)
    worst = 0.0
    for pdl in (1, 0):
        ctx = api.DGContext(nelem, order, lo, hi, bc=(0, 1, 1), omega_c=1.0, pmax=2)
        ctx.set_option(api.OPT_PDL, pdl)
        f0 = wl.add_uniform_noise(wl.ring_f0(ctx.nodes(0), ctx.nodes(1), ctx.nodes(2), K), wl.SEED_CFG3_NOISE, 1e-4)
        f = torch.from_numpy(f0).cuda()
        ctx.ssprk3_run(f, 1e-3, 2, True)
        assert ctx.last_kernel.startswith("rhs_tiled<8,")
        fo = ov.ssprk3_step(g, ov.ssprk3_step(g, f0, 1e-3), 1e-3)
        worst = max(worst, relerr(f.cpu().numpy(), fo))
        assert int(ctx.check_finite(f).item()) == 0
        ctx.close()
    return worst


def case_xslab():
    nelem, order = (2, 2, 2), (8, 8, 8)
    lo, hi = (0.0, -8.5, -8.5), (2 * math.pi / K, 8.5, 8.5)
    g = ov.Grid(nelem=nelem, order=order, lo=lo, hi=hi, bc=(0, 1, 1), omega_c=1.0, pmax=2)
    worst = 0.0
    for push in (False, True):
        st = sharded.XSlabStepper(nelem, order, lo, hi, bc=(0, 1, 1), omega_c=1.0, pmax=2, rank=0, world=1, device=0, push=push)
        f0 = wl.ring_f0(st.be.slab.nodes(0), st.be.slab.nodes(1), st.be.slab.nodes(2), K)
        f = torch.from_numpy(f0).cuda()
        st.run(f, 1e-3, 2, True)
        fo = ov.ssprk3_step(g, ov.ssprk3_step(g, f0, 1e-3), 1e-3)
        worst = max(worst, relerr(f.cpu().numpy(), fo))
        st.close()
    return worst


def case_2d2v():
    worst = 0.0
    for nelem, n in (((2, 2, 2, 8), 4), ((2, 2, 2, 2), 8)):
        lo, hi = (0.0, 0.0, -8.5, -8.5), (2 * math.pi / K, 2 * math.pi / K, 8.5, 8.5)
        ctx = api.DG4Context(nelem, (n,) * 4, lo, hi, bc=(0, 0, 1, 1), omega_c=1.0)
        g = o4.make_grid(nelem, (n,) * 4, lo, hi, omega_c=1.0, pmax=(nelem[0], nelem[1]))
        x, y, u, v = (ctx.nodes(d) for d in range(4))
        f0 = wl.ring2d_f0(x, y, u, v, K, K)
        f = torch.from_numpy(f0).cuda()
        ctx.ssprk3_run(f, 2e-4, 1)
        worst = max(worst, relerr(f.cpu().numpy(), o4.ssprk3_step(g, f0, 2e-4)))
        ctx.close()
    return worst


def case_field():
    N, n, lo, hi, pmax, batch = 16, 8, 0.0, 2 * math.pi, 32, 24
    worst = 0.0
    x = ofr.node_coordinates(lo, hi, N, n)
    rho_h, _, _, _ = wl.cosine_sum_density(x, batch, wl.SEED_CFG5, mmax=8)
    T = ofr.transform_tensor(lo, hi, N, n, pmax)
    Eo = ofr.poisson_E(lo, hi, x, ofr.fourier_project(T, rho_h))
    for fk in (api.FIELD_SIMPLE, api.FIELD_DMMA, api.FIELD_DFMA, api.FIELD_FFT):
        ctx = api.DGContext((N,), (n,), (lo,), (hi,), pmax=pmax, field_batch=batch)
        ctx.set_option(api.OPT_FIELD_KERNEL, fk)
        E = ctx.poisson_E(torch.from_numpy(rho_h).cuda())
        worst = max(worst, relerr(E.cpu().numpy(), Eo))
        ctx.close()
    return worst


CASES = {"config1": case_config1, "tiled": case_tiled, "xslab": case_xslab, "2d2v": case_2d2v, "field": case_field}

if __name__ == "__main__":
    names = sys.argv[1:] or list(CASES)
    for nm in names:
        err = CASES[nm]()
        torch.cuda.synchronize()
        print(f"case {nm}: max relative error vs oracle {err:.3e}", flush=True)
        assert err <= 1e-11, (nm, err)
    print("SANITIZER_CASES_OK", flush=True)
