"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element, on the same
seeded inputs.  Tolerances: max-norm relative error <= 1e-12 per RHS /
density / projection evaluation, <= 1e-10 after 100 RK steps (north_star)."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import vlasov as ov, fourier as ofr, basis as ob, pointwise as opw   # noqa: E402
import workloads as wl                                                          # noqa: E402


def api():
    from paper_2202_13532_b200 import api as _api
    return _api


def relerr(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


def make_pair(nelem, order, lo, hi, bc=None, omega_c=0.0, pmax=0, mass_mode=0, **kw):
    g = ov.Grid(nelem=tuple(nelem), order=tuple(order), lo=tuple(lo), hi=tuple(hi), bc=bc, omega_c=omega_c,
                pmax=pmax, mass_mode=mass_mode)
    ctx = api().DGContext(nelem, order, lo, hi, bc=g.bc, omega_c=omega_c, pmax=pmax, mass_mode=mass_mode, **kw)
    return g, ctx


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


# ---------------------------------------------------------------------------------------------
# setup quantities
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [2, 3, 4, 5, 6, 7, 8, 9, 10])
@pytest.mark.parametrize("mode", [0, 1])
def test_operators_match_oracle(n, mode):
    g, ctx = make_pair((3, 2), (n, n), (0.0, -1.0), (2.0, 1.0), mass_mode=mode, workspace=False)
    xi, w, ups, lift = ctx.operators(0)
    oxi, ow, oups, olift = ob.operators(n, mode)
    assert np.max(np.abs(xi - oxi)) < 1e-15 and np.max(np.abs(w - ow)) < 1e-15
    assert relerr(ups, oups) < 2e-14 and relerr(lift, olift) < 1e-14
    assert np.max(np.abs(ctx.nodes(0) - g.x_nodes())) < 1e-15
    ctx.close()


@pytest.mark.parametrize("N,n,pmax,lo,hi", [(16, 4, 16, 0.0, 4 * math.pi), (32, 8, 32, 0.0, 20 * math.pi),
                                           (7, 6, 30, -1.0, 2.5), (5, 10, 9, 0.0, 1.0), (64, 8, 200, 0.0, 2 * math.pi)])
def test_transform_tensor_matches_oracle(N, n, pmax, lo, hi):
    ctx = api().DGContext((N,), (n,), (lo,), (hi,), pmax=pmax, workspace=False)
    T = ctx.transform()
    To = ofr.transform_tensor(lo, hi, N, n, pmax)
    assert np.max(np.abs(T - To)) < 5e-16 * max(1.0, N * n * np.max(np.abs(To)))
    ctx.close()


# ---------------------------------------------------------------------------------------------
# RHS
# ---------------------------------------------------------------------------------------------
RHS_CASES = [
    # nelem, order, lo, hi, bc, omega_c, mass_mode
    ((16, 32), (4, 4), (0.0, -6.0), (4 * math.pi, 6.0), (0, 1), 0.0, 0),              # config-1 grid
    ((5, 7), (3, 6), (0.0, -2.0), (3.0, 2.5), (0, 0), 0.0, 1),                        # unequal orders, periodic v
    ((4, 6, 8), (8, 8, 8), (0.0, -8.5, -8.5), (20 * math.pi, 8.5, 8.5), (0, 1, 1), 1.0, 0),   # config-2/3 shape, ragged tile tail
    ((3, 4, 5), (8, 8, 8), (0.0, -3.0, -2.0), (2.0, 3.5, 2.5), (0, 0, 0), 0.7, 0),    # all periodic, asymmetric box
    ((3, 4, 5), (8, 8, 8), (0.0, -3.0, -2.0), (2.0, 3.5, 2.5), (1, 1, 0), 0.7, 1),    # lumped, mixed bc
    ((5, 6, 6), (4, 4, 4), (0.0, -4.0, -4.0), (6.0, 4.0, 4.0), (0, 1, 1), 1.0, 0),
    ((4, 4, 5), (6, 6, 6), (0.0, -4.0, -4.0), (6.0, 4.0, 4.0), (0, 1, 1), 1.0, 0),
    ((3, 3, 4), (10, 10, 10), (0.0, -4.0, -4.0), (6.0, 4.0, 4.0), (0, 1, 1), 1.0, 0),
    ((3, 2, 4), (3, 5, 4), (0.0, -1.0, -2.0), (1.5, 1.0, 2.0), (0, 1, 0), 1.3, 0),    # per-dim orders -> generic only
    ((1, 1, 1), (8, 8, 8), (0.0, -1.0, -1.0), (1.0, 1.0, 1.0), (0, 0, 0), 0.5, 0),    # single element, self-periodic
]


@pytest.mark.parametrize("case", RHS_CASES)
@pytest.mark.parametrize("kernel", ["generic", "auto"])
def test_rhs_matches_oracle(case, kernel):
    nelem, order, lo, hi, bc, omega_c, mode = case
    g, ctx = make_pair(nelem, order, lo, hi, bc=bc, omega_c=omega_c, mass_mode=mode)
    ctx.set_option(api().OPT_RHS_KERNEL, api().KERNEL_GENERIC if kernel == "generic" else api().KERNEL_AUTO)
    f = wl.uniform_field(g.flat_shape, wl.SEED_CFG4_F)
    E = wl.normal_E(g.flat_shape[0], wl.SEED_CFG4_E)
    for Ein in (E, None):
        out = ctx.rhs(dev(f), None if Ein is None else dev(Ein)).cpu().numpy()
        ref = ov.rhs(g, f, Ein)
        assert relerr(out, ref) <= 1e-12, (ctx.last_kernel, relerr(out, ref))
    ctx.close()


def test_rhs_zero_speed_nodes_and_sign_changes():
    """Even element counts put a node exactly at v = 0 (a = 0 => zero flux, reading C12) and E makes
    a_u change sign inside elements."""
    g, ctx = make_pair((4, 4, 4), (8, 8, 8), (0.0, -2.0, -2.0), (2.0, 2.0, 2.0), bc=(0, 1, 1), omega_c=1.0)
    f = wl.uniform_field(g.flat_shape, 11)
    E = 1.5 * np.sin(np.arange(g.flat_shape[0]) * 0.7)          # |E| comparable with omega_c |v|
    out = ctx.rhs(dev(f), dev(E)).cpu().numpy()
    assert relerr(out, ov.rhs(g, f, E)) <= 1e-12
    ctx.close()


def test_rhs_errors():
    g, ctx = make_pair((2, 2), (4, 4), (0.0, -1.0), (1.0, 1.0))
    f = dev(np.zeros(g.flat_shape))
    with pytest.raises(api().DGError):
        ctx.rhs(f, None, out=f)                                    # aliasing
    with pytest.raises(api().DGError):
        ctx.rhs(f.float())                                          # wrong dtype is caught by the binding
    ctx.close()
    c1 = api().DGContext((8,), (8,), (0.0,), (1.0,), workspace=False)
    with pytest.raises(api().DGError):
        c1.rhs(f)                                                   # field-only context
    c1.close()


# ---------------------------------------------------------------------------------------------
# density, projection, Poisson
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("case", [RHS_CASES[0], RHS_CASES[1], RHS_CASES[2], RHS_CASES[8]])
def test_density_matches_oracle(case):
    nelem, order, lo, hi, bc, omega_c, mode = case
    g, ctx = make_pair(nelem, order, lo, hi, bc=bc, omega_c=omega_c, mass_mode=mode)
    f = wl.uniform_field(g.flat_shape, 5) - 0.25
    rho = ctx.density(dev(f)).cpu().numpy()
    assert relerr(rho, ov.density(g, f)) <= 1e-13
    rho2 = ctx.density(dev(f)).cpu().numpy()
    assert np.array_equal(rho, rho2)                                # deterministic
    ctx.close()


@pytest.mark.parametrize("N,n,pmax,batch,kernel", [(16, 4, 16, 1, 0), (32, 8, 32, 3, 1), (64, 8, 100, 40, 2),
                                                  (37, 6, 51, 33, 2), (64, 8, 64, 1, 2), (9, 5, 7, 130, 0),
                                                  (64, 8, 100, 40, 3), (9, 5, 7, 130, 2), (40, 8, 150, 200, 2),
                                                  (41, 6, 163, 300, 2), (40, 8, 150, 200, 3)])
def test_project_and_poisson_match_oracle(N, n, pmax, batch, kernel):
    lo, hi = 0.0, 2 * math.pi
    ctx = api().DGContext((N,), (n,), (lo,), (hi,), pmax=pmax, field_batch=batch)
    ctx.set_option(api().OPT_FIELD_KERNEL, kernel)
    x = ofr.node_coordinates(lo, hi, N, n)
    rho, A, M, PH = wl.cosine_sum_density(x, batch, wl.SEED_CFG5, mmax=max(1, min(1024, pmax // 2)))
    To = ofr.transform_tensor(lo, hi, N, n, pmax)
    c = ctx.fourier_project(dev(rho)).cpu().numpy()
    co = ofr.fourier_project(To, rho)
    assert relerr(c[..., 0] + 1j * c[..., 1], co) <= 1e-12
    E = ctx.poisson_E(dev(rho)).cpu().numpy()
    Eo = ofr.poisson_E(lo, hi, x, co)
    assert relerr(E, Eo) <= 1e-12
    ctx.close()


def test_poisson_single_cosine_closed_form():
    """Closed form E = -(A/k) sin(kx + phi) on the config-5 grid (2048 x 8), modes <= 1024."""
    N, n, lo, hi = 2048, 8, 0.0, 2 * math.pi
    ctx = api().DGContext((N,), (n,), (lo,), (hi,), pmax=2048, field_batch=4)
    x = ctx.nodes(0)
    ms, A, ph = np.array([1, 16, 333, 1024]), 0.05, 0.4
    rho = 1 + A * np.cos(ms[:, None] * x[None, :] + ph)
    E = ctx.poisson_E(dev(rho)).cpu().numpy()
    Eex = -(A / ms[:, None]) * np.sin(ms[:, None] * x[None, :] + ph)
    for i in range(4):
        assert relerr(E[i], Eex[i]) < (1e-11 if ms[i] < 1024 else 1e-8), (ms[i], relerr(E[i], Eex[i]))   # m = 1024: 2 elements per wavelength
    c = ctx.fourier_project(dev(rho)).cpu().numpy()
    for i, m in enumerate(ms):
        assert abs(c[i, m, 0] + 1j * c[i, m, 1] - 0.5 * A * np.exp(1j * ph)) < (1e-13 if m < 1024 else 1e-9)
        assert abs(c[i, 0, 0] - 1) < 1e-13
    ctx.close()


# ---------------------------------------------------------------------------------------------
# SSP-RK3
# ---------------------------------------------------------------------------------------------
def test_config1_landau_10_steps():
    g, ctx = make_pair((16, 32), (4, 4), (0.0, -6.0), (4 * math.pi, 6.0), bc=(0, 1), pmax=16)
    x, v = ctx.nodes(0), ctx.nodes(1)
    f0 = wl.landau_f0(x, v)
    fo = f0.copy()
    for _ in range(10):
        fo = ov.ssprk3_step(g, fo, 0.01)
    fd = dev(f0)
    for _ in range(10):
        ctx.ssprk3_step(fd, 0.01, True)
    assert relerr(fd.cpu().numpy(), fo) <= 1e-10
    fd2 = dev(f0)
    ctx.ssprk3_run(fd2, 0.01, 10, True)
    assert relerr(fd2.cpu().numpy(), fo) <= 1e-10
    fh = f0.copy()
    ctx.ssprk3_run_host(fh, 0.01, 10, True)
    assert relerr(fh, fo) <= 1e-10
    assert abs(ctx.max_stable_dt(0.02) - 1.0 / (6.0 / (0.1301 * 4 * math.pi / 16) + 0.02 / (0.1301 * 12 / 32))) < 2e-3 * ctx.max_stable_dt(0.02)
    ctx.close()


@pytest.mark.parametrize("kernel", ["generic", "auto"])
@pytest.mark.parametrize("self_consistent", [True, False])
def test_small_1d2v_ring_steps(kernel, self_consistent):
    """Config-2 physics on an 8x8x8-element replica: ring x (1 + 0.01 sin kx), omega_c = 1, zero-inflow v."""
    k = 0.1
    g, ctx = make_pair((8, 8, 8), (8, 8, 8), (0.0, -8.5, -8.5), (2 * math.pi / k, 8.5, 8.5), bc=(0, 1, 1),
                       omega_c=1.0, pmax=8)
    ctx.set_option(api().OPT_RHS_KERNEL, api().KERNEL_GENERIC if kernel == "generic" else api().KERNEL_AUTO)
    f0 = wl.ring_f0(ctx.nodes(0), ctx.nodes(1), ctx.nodes(2), k)
    dt, steps = 0.004, 6
    fo = f0.copy()
    for _ in range(steps):
        fo = ov.ssprk3_step(g, fo, dt, self_consistent=self_consistent)
    fd = dev(f0)
    ctx.ssprk3_run(fd, dt, steps, self_consistent)
    assert relerr(fd.cpu().numpy(), fo) <= 1e-11
    assert ctx.launch_count > 0
    ctx.close()
