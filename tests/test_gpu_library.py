"""Library-level behaviour added in round 2: non-finite guard, stage-coefficient table, sign of c1*dt in the tiled kernel,
per-stage profile samples, device guard, FP64 peak probe."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import vlasov as ov          # noqa: E402
import workloads as wl                   # noqa: E402

K = 0.1
LO, HI = (0.0, -8.5, -8.5), (2 * math.pi / K, 8.5, 8.5)


def api():
    from paper_2202_13532_b200 import api as _api
    return _api


def relerr(a, b):
    return float(np.max(np.abs(np.asarray(a) - np.asarray(b))) / max(np.max(np.abs(b)), 1e-300))


def test_stage_coeffs_are_shu_osher():
    """PAPER.md:477 (ref. [38]): (0, 1), (3/4, 1/4), (1/3, 2/3) -- the same table the oracle's ssprk3_step writes out."""
    A = api()
    assert [A.ssprk3_stage_coeffs(s) for s in range(3)] == [(0.0, 1.0), (0.75, 0.25), (1.0 / 3.0, 2.0 / 3.0)]
    with pytest.raises(A.DGError):
        A.ssprk3_stage_coeffs(3)


@pytest.mark.parametrize("shape", [((4, 4, 4), (8, 8, 8)), ((3, 5), (4, 4)), ((2, 3, 3), (5, 3, 3))])
def test_check_finite(shape):
    nelem, order = shape
    nd = len(nelem)
    ctx = api().DGContext(nelem, order, LO[:nd], HI[:nd], bc=(0,) + (1,) * (nd - 1), omega_c=1.0)
    f = torch.rand(ctx.flat_shape, dtype=torch.float64, device="cuda")
    assert int(ctx.check_finite(f).item()) == 0
    for bad in (float("nan"), float("inf"), -float("inf")):
        for pos in (0, f.numel() // 2 + 1, f.numel() - 1):
            g = f.clone()
            g.view(-1)[pos] = bad
            assert int(ctx.check_finite(g).item()) == 1, (bad, pos)
    assert int(ctx.check_finite(f).item()) == 0          # the flag is reset by every call
    ctx.close()


def test_check_finite_catches_the_literal_config2_blowup():
    """Config 2 as literally written (dt = 0.005, omega_c = 1) violates the RK3 limit (reading C22): the run
    diverges and the guard reports it; at the stable dt it does not."""
    nelem, order = (8, 16, 16), (8, 8, 8)
    ctx = api().DGContext(nelem, order, LO, HI, bc=(0, 1, 1), omega_c=1.0, pmax=8)
    f0 = wl.ring_f0(ctx.nodes(0), ctx.nodes(1), ctx.nodes(2), K)
    assert 5e-3 > ctx.max_stable_dt(0.2) > 1e-3
    f = torch.from_numpy(f0).cuda()
    ctx.ssprk3_run(f, 1e-3, 60, True)
    assert int(ctx.check_finite(f).item()) == 0 and float(f.abs().max()) < 0.05
    f = torch.from_numpy(f0).cuda()
    ctx.ssprk3_run(f, 5e-3, 400, True)
    assert int(ctx.check_finite(f).item()) == 1 or float(f.abs().max()) > 1e3
    ctx.close()


@pytest.mark.parametrize("n,N", [(8, (2, 3, 5)), (4, (3, 2, 9)), (6, (2, 2, 5)), (10, (2, 2, 3))])
def test_negative_dt_tiled_matches_generic_and_oracle(n, N):
    """The upwind side of Eq. 23 is chosen by the sign of the speed, not of c1*dt*speed: a stage with
    dt < 0 gives out = c0 f_n + c1 (f_s + dt L(f_s)) with the same L."""
    A = api()
    ctx = A.DGContext(N, (n,) * 3, LO, HI, bc=(0, 1, 0), omega_c=1.0)
    g = ov.Grid(nelem=N, order=(n,) * 3, lo=LO, hi=HI, bc=(0, 1, 0), omega_c=1.0)
    fs = wl.uniform_field(g.flat_shape, wl.SEED_CFG4_F)
    fn = wl.uniform_field(g.flat_shape, wl.SEED_CFG4_F + 1)
    E = wl.normal_E(g.flat_shape[0], wl.SEED_CFG4_E)
    L = ov.rhs(g, fs, E)
    for c0, c1, dt in ((0.75, 0.25, -1e-3), (0.0, 1.0, -2e-3), (1.0 / 3.0, -2.0 / 3.0, 1e-3)):
        ref = c0 * fn + c1 * (fs + dt * L)
        outs = {}
        for kern in (A.KERNEL_TILED, A.KERNEL_GENERIC):
            ctx.set_option(A.OPT_RHS_KERNEL, kern)
            out = torch.empty(g.flat_shape, dtype=torch.float64, device="cuda")
            ctx.rk_stage(torch.from_numpy(fs).cuda(), torch.from_numpy(fn).cuda() if c0 else None, torch.from_numpy(E).cuda(), out,
                         c0, c1, dt)
            outs[kern] = out.cpu().numpy()
            # error relative to the size of the dt*L term, which is what the sign decision changes
            assert np.max(np.abs(outs[kern] - ref)) <= 1e-12 * np.max(np.abs(c1 * dt * L)), (kern, c0, c1, dt)
        assert ctx.last_kernel == "rhs_generic"
    ctx.close()


def test_profile_stage_samples():
    A = api()
    ctx = A.DGContext((4, 4, 8), (8, 8, 8), LO, HI, bc=(0, 1, 1), omega_c=1.0, pmax=4)
    f = torch.from_numpy(wl.ring_f0(ctx.nodes(0), ctx.nodes(1), ctx.nodes(2), K)).cuda()
    ref = f.clone()
    ctx.ssprk3_run(ref, 1e-3, 14, True)
    ctx.set_option(A.OPT_PROFILE, 7)
    ctx.get_profile_stages(reset=True)
    ctx.ssprk3_run(f, 1e-3, 14, True)                 # 42 RHS launches: every 7th bracketed -> 6 samples, 2 per stage
    ms, n = ctx.get_profile_stages(reset=True)
    assert n == [0, 2, 2, 2] and all(m > 0 for m in ms[1:]) and ms[0] == 0
    assert torch.equal(f, ref)                        # sampling does not change the result
    ctx.set_option(A.OPT_PROFILE, 1)
    out = ctx.rhs(f)
    ms, n = ctx.get_profile_stages(reset=True)
    assert n == [1, 0, 0, 0]
    tot, cnt = ctx.get_profile(reset=True)
    assert cnt == 0
    ctx.set_option(A.OPT_PROFILE, 0)
    del out
    ctx.close()


def test_create_restores_the_callers_device_and_two_contexts_coexist():
    A = api()
    cur = torch.cuda.current_device()
    a = A.DGContext((2, 2, 4), (8, 8, 8), LO, HI, omega_c=1.0, device=0)
    b = A.DGContext((2, 2, 4), (8, 8, 8), LO, HI, omega_c=1.0, device=torch.cuda.device_count() - 1)
    assert torch.cuda.current_device() == cur
    fa = torch.rand(a.flat_shape, dtype=torch.float64, device=a.device)
    fb = fa.to(b.device)
    ra, rb = a.rhs(fa), b.rhs(fb)
    assert torch.equal(ra.cpu(), rb.cpu())
    with pytest.raises(A.DGError):
        A.DGContext((2, 2, 4), (8, 8, 8), LO, HI, device=torch.cuda.device_count() + 3)
    a.close(); b.close()


def test_fp64_peak_probe():
    A = api()
    dfma, dmma = A.fp64_peak(0, 0, 4000), A.fp64_peak(0, 1, 4000)
    assert 10.0 < dfma < 80.0 and 10.0 < dmma < 80.0      # nominal 37.2 TFLOP/s at 1.965 GHz
