"""GPU parity of the 2D2V path (include/dgvlasov2d2v.h) against oracle/vlasov2d2v.py on the same seeded inputs.
Tolerances as for the 1D2V path: max-norm relative error <= 1e-12 per RHS / density / field
evaluation, <= 1e-11 after a few RK steps."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import vlasov2d2v as o4      # noqa: E402
import workloads as wl                   # noqa: E402

LO, HI = (0.0, -1.0, -6.0, -5.5), (2.0 * math.pi, 2.0, 6.0, 5.5)


def api():
    from paper_2202_13532_b200 import api as _api
    return _api


def relerr(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def make_pair(N, n, bc=(0, 0, 1, 1), omega_c=0.8, pmax=(0, 0), mass_mode=0, lo=LO, hi=HI):
    g = o4.make_grid(N, n, lo, hi, bc=bc, omega_c=omega_c, pmax=pmax, mass_mode=mass_mode)
    ctx = api().DG4Context(N, n, lo, hi, bc=bc, omega_c=omega_c, pmax=pmax, mass_mode=mass_mode)
    return g, ctx


def seeded_inputs(g):
    dof = int(np.prod(g.flat_shape))
    f = wl.counter_uniform_chunked(wl.SEED_CFG6_NOISE, dof).reshape(g.flat_shape)
    gxy = g.flat_shape[0] * g.flat_shape[1]
    E = 0.5 * wl.counter_normal(wl.SEED_CFG6_E, 0, 2 * gxy)
    return f, E[:gxy].reshape(g.flat_shape[:2]), E[gxy:].reshape(g.flat_shape[:2])


# (N, n): generic kernel for mixed orders, tiled kernel <2>, <4>, <8> for n = 4 (several tiles + zero-inflow / periodic edges)
SHAPES = [((3, 2, 3, 4), (3, 4, 5, 2)), ((2, 3, 2, 3), (4, 4, 4, 4)), ((3, 2, 3, 2), (4, 4, 4, 4)), ((2, 3, 3, 4), (4, 4, 4, 4)),
          ((3, 2, 2, 8), (4, 4, 4, 4)), ((2, 2, 3, 16), (4, 4, 4, 4)), ((2, 2, 2, 2), (6, 6, 6, 6)), ((3, 2, 3, 2), (6, 6, 6, 6)),
          ((2, 3, 1, 2), (8, 8, 8, 8)), ((1, 1, 2, 3), (8, 8, 8, 8)), ((2, 2, 2, 2), (5, 5, 5, 5))]


@pytest.mark.parametrize("N,n", SHAPES)
@pytest.mark.parametrize("bc", [(0, 0, 1, 1), (0, 0, 0, 0), (1, 1, 1, 1)])
@pytest.mark.parametrize("mode", [0, 1])
def test_rhs_matches_oracle(N, n, bc, mode):
    g, ctx = make_pair(N, n, bc=bc, mass_mode=mode)
    f, Ex, Ey = seeded_inputs(g)
    r = ctx.rhs(dev(f), dev(Ex), dev(Ey)).cpu().numpy()
    ro = o4.rhs(g, f, Ex, Ey)
    assert relerr(r, ro) < 1e-12, ctx.last_kernel
    if all(k == 4 for k in n) and N[3] % 2 == 0:
        expect = "rhs4_tile"
    elif n == (8, 8, 8, 8):
        expect = "rhs4_line"
    elif n == (6, 6, 6, 6):
        expect = "rhs4_elem"
    else:
        expect = "rhs4_generic"
    assert ctx.last_kernel.startswith(expect), ctx.last_kernel
    ctx.close()


def test_tiled_equals_generic_kernel():
    g, ctx = make_pair((10, 3, 3, 8), (4, 4, 4, 4))
    f, Ex, Ey = seeded_inputs(g)
    fd, exd, eyd = dev(f), dev(Ex), dev(Ey)
    a = ctx.rhs(fd, exd, eyd).cpu().numpy()
    assert ctx.last_kernel == "rhs4_tile<8>"
    ctx.set_option(api().OPT4_RHS_KERNEL, 1)
    b = ctx.rhs(fd, exd, eyd).cpu().numpy()
    assert ctx.last_kernel == "rhs4_generic"
    assert relerr(a, b) < 1e-13
    assert relerr(a, o4.rhs(g, f, Ex, Ey)) < 1e-12
    ctx.close()


@pytest.mark.parametrize("N,n", [((3, 2, 3, 3), (4, 4, 4, 4)), ((2, 2, 2, 8), (4, 4, 4, 4)), ((2, 2, 3, 2), (6, 6, 6, 6)), ((2, 1, 2, 2), (8, 8, 8, 8))])
@pytest.mark.parametrize("bc", [(0, 0, 1, 1), (1, 1, 0, 0)])
def test_element_kernel_stage_and_density(N, n, bc):
    """rhs4_elem_kernel forced (DG4_OPT_RHS_KERNEL = 3): one Shu-Osher stage with f_n and the epilogue density, and the RHS
    against the generic kernel on the device."""
    g, ctx = make_pair(N, n, bc=bc)
    ctx.set_option(api().OPT4_RHS_KERNEL, 3)
    f, Ex, Ey = seeded_inputs(g)
    fn = 0.5 + wl.counter_uniform_chunked(wl.SEED_CFG6_E, f.size).reshape(f.shape)
    fd, fnd, exd, eyd = dev(f), dev(fn), dev(Ex), dev(Ey)
    out, rho = torch.empty_like(fd), torch.empty(g.flat_shape[:2], dtype=torch.float64, device="cuda")
    ctx.rk_stage(fd, fnd, exd, eyd, out, 1.0 / 3.0, 2.0 / 3.0, 1e-3, rho_out=rho)
    assert ctx.last_kernel.startswith("rhs4_elem")
    ro = o4.rhs(g, f, Ex, Ey)
    oo = (1.0 / 3.0) * fn + (2.0 / 3.0) * (f + 1e-3 * ro)
    assert relerr(out.cpu().numpy(), oo) < 1e-13
    assert relerr(rho.cpu().numpy(), o4.density(g, oo)) < 1e-13
    a = ctx.rhs(fd, exd, eyd).cpu().numpy()
    ctx.set_option(api().OPT4_RHS_KERNEL, 1)
    b = ctx.rhs(fd, exd, eyd).cpu().numpy()
    assert relerr(a, ro) < 1e-12 and relerr(a, b) < 1e-13
    ctx.close()


@pytest.mark.parametrize("N", [(2, 1, 2, 2), (1, 2, 3, 2), (3, 2, 1, 1), (4, 2, 2, 3)])
@pytest.mark.parametrize("bc", [(0, 0, 1, 1), (1, 1, 0, 0), (0, 0, 0, 0)])
@pytest.mark.parametrize("mode", [0, 1])
def test_line_kernel_stage_and_density(N, bc, mode):
    """rhs4_line_kernel (n = 8, TMA): what `auto` takes at the paper's order.  One Shu-Osher stage with f_n and the epilogue
    density, a stage without f_n, the plain RHS against the oracle and against the generic and element kernels on the device
    (the mirrored u lines of the odd-jy threads and the x-rasterisation groups are both exercised by N_x = 4, N_y = 2)."""
    n = (8, 8, 8, 8)
    g, ctx = make_pair(N, n, bc=bc, mass_mode=mode)
    f, Ex, Ey = seeded_inputs(g)
    fn = 0.5 + wl.counter_uniform_chunked(wl.SEED_CFG6_E, f.size).reshape(f.shape)
    fd, fnd, exd, eyd = dev(f), dev(fn), dev(Ex), dev(Ey)
    out, rho = torch.empty_like(fd), torch.empty(g.flat_shape[:2], dtype=torch.float64, device="cuda")
    ctx.rk_stage(fd, fnd, exd, eyd, out, 1.0 / 3.0, 2.0 / 3.0, 1e-3, rho_out=rho)
    assert ctx.last_kernel == "rhs4_line<8>"
    ro = o4.rhs(g, f, Ex, Ey)
    oo = (1.0 / 3.0) * fn + (2.0 / 3.0) * (f + 1e-3 * ro)
    assert relerr(out.cpu().numpy(), oo) < 1e-13
    assert relerr(rho.cpu().numpy(), o4.density(g, oo)) < 1e-13
    # in place on f_n (stage 3 of dg4_ssprk3_run) and without f_n (stage 1), negative dt (upwind side from the unscaled speed)
    inpl = fnd.clone()
    ctx.rk_stage(fd, inpl, exd, eyd, inpl, 1.0 / 3.0, 2.0 / 3.0, 1e-3)
    assert torch.equal(inpl, out)
    ctx.rk_stage(fd, None, exd, eyd, out, 0.0, 1.0, -2e-3)
    assert np.max(np.abs(out.cpu().numpy() - (f - 2e-3 * ro))) <= 1e-12 * 2e-3 * np.max(np.abs(ro))
    a = ctx.rhs(fd, exd, eyd).cpu().numpy()
    assert ctx.last_kernel == "rhs4_line<8>"
    ctx.set_option(api().OPT4_RHS_KERNEL, 1)
    b = ctx.rhs(fd, exd, eyd).cpu().numpy()
    ctx.set_option(api().OPT4_RHS_KERNEL, 3)
    c = ctx.rhs(fd, exd, eyd).cpu().numpy()
    assert ctx.last_kernel.startswith("rhs4_elem")
    assert relerr(a, ro) < 1e-12 and relerr(a, b) < 1e-13 and relerr(a, c) < 1e-13
    # E = NULL
    ctx.set_option(api().OPT4_RHS_KERNEL, 0)
    assert relerr(ctx.rhs(fd).cpu().numpy(), o4.rhs(g, f)) < 1e-12
    ctx.close()


def test_rhs_without_field_and_zero_speed_nodes():
    """E = NULL; an even number of velocity elements puts nodes at u = 0, v = 0 (zero flux there, Eq. 23)."""
    g, ctx = make_pair((2, 2, 4, 8), (4, 4, 4, 4), omega_c=0.0, lo=(0, 0, -2, -2), hi=(1, 1, 2, 2))
    f, _, _ = seeded_inputs(g)
    r = ctx.rhs(dev(f)).cpu().numpy()
    assert relerr(r, o4.rhs(g, f)) < 1e-12
    ctx.close()


@pytest.mark.parametrize("N,n", [((3, 2, 3, 4), (3, 4, 5, 2)), ((2, 3, 3, 8), (4, 4, 4, 4)), ((2, 2, 5, 3), (4, 4, 4, 5))])
def test_density_matches_oracle(N, n):
    g, ctx = make_pair(N, n)
    f, _, _ = seeded_inputs(g)
    rho = ctx.density(dev(f)).cpu().numpy()
    assert relerr(rho, o4.density(g, f)) < 1e-13
    ctx.close()


@pytest.mark.parametrize("N,n,pmax", [((8, 6, 1, 1), (8, 8, 2, 2), (5, 4)), ((5, 7, 1, 1), (4, 6, 2, 2), (0, 0)), ((16, 16, 1, 1), (4, 4, 2, 2), (16, 16))])
def test_projection_and_field_match_oracle(N, n, pmax):
    g, ctx = make_pair(N, n, pmax=pmax, lo=(0.0, 1.0, -1, -1), hi=(2 * math.pi, 4.0, 1, 1))
    x, y = g.coords[0].reshape(-1), g.coords[1].reshape(-1)
    rng_u = wl.counter_uniform(wl.SEED_CFG6_E, 0, 64)
    rho = np.ones((x.size, y.size))
    for i in range(8):                                     # seeded sum of plane waves + noise
        p, q = 1 + int(rng_u[4 * i] * 3), int(rng_u[4 * i + 1] * 7) - 3
        rho += 0.05 * rng_u[4 * i + 2] * np.cos(p * x[:, None] + 2 * math.pi * q / 3.0 * y[None, :] + 6.28 * rng_u[4 * i + 3])
    rho += 1e-3 * wl.counter_normal(wl.SEED_CFG6_NOISE, 0, rho.size).reshape(rho.shape)
    c = ctx.fourier_project(dev(rho)).cpu().numpy()
    co = o4.fourier_project(g, rho)
    assert relerr(c[..., 0] + 1j * c[..., 1], co) < 1e-12
    Ex, Ey = ctx.poisson_E(dev(rho))
    Exo, Eyo = o4.poisson_E(g, co)
    scale = max(np.max(np.abs(Exo)), np.max(np.abs(Eyo)))
    assert np.max(np.abs(Ex.cpu().numpy() - Exo)) < 1e-12 * scale + 1e-14      # reading C26: rho carries the mean 1
    assert np.max(np.abs(Ey.cpu().numpy() - Eyo)) < 1e-12 * scale + 1e-14
    ctx.close()


def test_plane_wave_field_closed_form():
    g, ctx = make_pair((8, 8, 1, 1), (8, 8, 2, 2), pmax=(3, 3), lo=(0.0, 0.0, -1, -1), hi=(2 * math.pi, 3.0, 1, 1))
    x, y = ctx.nodes(0), ctx.nodes(1)
    kx, ky = 2.0, -2 * math.pi / 3.0
    arg = kx * x[:, None] + ky * y[None, :] + 0.3
    Ex, Ey = ctx.poisson_E(dev(1.0 + 0.05 * np.cos(arg)))
    k2 = kx * kx + ky * ky
    assert np.max(np.abs(Ex.cpu().numpy() + 0.05 * kx / k2 * np.sin(arg))) < 1e-11
    assert np.max(np.abs(Ey.cpu().numpy() + 0.05 * ky / k2 * np.sin(arg))) < 1e-11
    ctx.close()


@pytest.mark.parametrize("N,n", [((3, 2, 3, 8), (4, 4, 4, 4)), ((2, 2, 3, 2), (3, 4, 4, 3)), ((2, 2, 2, 3), (6, 6, 6, 6)), ((1, 2, 2, 2), (8, 8, 8, 8))])
def test_self_consistent_steps_match_oracle(N, n):
    """Ring workload, three SSP-RK3 steps with the 2-D Poisson solve at every stage (density partials from the tile epilogue)."""
    g, ctx = make_pair(N, n, omega_c=1.0, lo=(0.0, 0.0, -8.5, -8.5), hi=(20 * math.pi, 10 * math.pi, 8.5, 8.5))
    x, y, u, v = [c.reshape(-1) for c in g.coords]
    f = wl.ring2d_f0(x, y, u, v, 0.1, 0.2)
    f = wl.add_uniform_noise(f, wl.SEED_CFG6_NOISE, 1e-4)
    dt = 2e-3
    fo = f.copy()
    for _ in range(3):
        fo = o4.ssprk3_step(g, fo, dt)
    fd = ctx.ssprk3_run(dev(f), dt, 3).cpu().numpy()
    assert relerr(fd, fo) < 1e-11
    fh = f.copy()
    ctx.ssprk3_run_host(fh, dt, 3)
    assert np.array_equal(fh, fd)
    ctx.close()


def test_rk_stage_density_output():
    g, ctx = make_pair((2, 2, 3, 8), (4, 4, 4, 4), bc=(0, 0, 0, 0))
    f, Ex, Ey = seeded_inputs(g)
    fd = dev(f)
    out, rho = torch.empty_like(fd), torch.empty(g.flat_shape[:2], dtype=torch.float64, device="cuda")
    ctx.rk_stage(fd, fd, dev(Ex), dev(Ey), out, 0.75, 0.25, 1e-3, rho_out=rho)
    oo = 0.75 * f + 0.25 * (f + 1e-3 * o4.rhs(g, f, Ex, Ey))
    assert relerr(out.cpu().numpy(), oo) < 1e-13
    assert relerr(rho.cpu().numpy(), o4.density(g, oo)) < 1e-13
    ctx.close()


def test_errors():
    a = api()
    with pytest.raises(a.DGError):
        a.DG4Context((2, 2, 2, 2), (4, 4, 4, 11), LO, HI)
    ctx = a.DG4Context((2, 2, 2, 3), (4, 4, 4, 4), LO, HI)
    ctx.set_option(a.OPT4_RHS_KERNEL, 2)
    f = torch.zeros(ctx.flat_shape, dtype=torch.float64, device="cuda")
    with pytest.raises(a.DGError):
        ctx.rhs(f)                     # odd N_v: no tiled kernel
    ctx.close()


def test_bench_size_64_full_array_stage_against_oracle():
    """config6_2d2v_64^4 (16.7 M DOF, the launch configuration bench.py times: rhs4_tile<8>, 8192 tiles): one Shu-Osher stage
    with a seeded field, the whole output array and the epilogue density against the oracle."""
    N = (16, 16, 16, 16)
    lo, hi = (0.0, 0.0, -8.5, -8.5), (20 * math.pi, 20 * math.pi, 8.5, 8.5)
    g, ctx = make_pair(N, (4, 4, 4, 4), omega_c=1.0, lo=lo, hi=hi)
    x, y, u, v = [c.reshape(-1) for c in g.coords]
    f = wl.add_uniform_noise(wl.ring2d_f0(x, y, u, v, 0.1, 0.1), wl.SEED_CFG6_NOISE, 1e-4)
    gxy = g.flat_shape[0] * g.flat_shape[1]
    E = 0.1 * wl.counter_normal(wl.SEED_CFG6_E, 0, 2 * gxy)
    Ex, Ey = E[:gxy].reshape(g.flat_shape[:2]), E[gxy:].reshape(g.flat_shape[:2])
    fd = dev(f)
    out, rho = torch.empty_like(fd), torch.empty(g.flat_shape[:2], dtype=torch.float64, device="cuda")
    ctx.rk_stage(fd, fd, dev(Ex), dev(Ey), out, 0.75, 0.25, 2e-4, rho_out=rho)
    assert ctx.last_kernel == "rhs4_tile<8>"
    ro = o4.rhs(g, f, Ex, Ey)
    oo = 0.75 * f + 0.25 * (f + 2e-4 * ro)
    assert relerr(out.cpu().numpy(), oo) < 1e-13
    assert relerr(rho.cpu().numpy(), o4.density(g, oo)) < 1e-13
    r = ctx.rhs(fd, dev(Ex), dev(Ey)).cpu().numpy()
    assert relerr(r, ro) < 1e-12
    ctx.close()


def test_bench_size_128_sampled_against_oracle():
    """config6_2d2v_128^4 (268 M DOF, 2.1 GB per array): dg4_rhs on the full grid, 400 seeded sample nodes (tile corners, box
    faces and interior) against the oracle's node-by-node loops, and the full-grid density against its plain definition."""
    N = (32, 32, 32, 32)
    lo, hi = (0.0, 0.0, -8.5, -8.5), (20 * math.pi, 20 * math.pi, 8.5, 8.5)
    g, ctx = make_pair(N, (4, 4, 4, 4), omega_c=1.0, lo=lo, hi=hi)
    x, y, u, v = [c.reshape(-1) for c in g.coords]
    f = wl.add_uniform_noise(wl.ring2d_f0(x, y, u, v, 0.1, 0.1), wl.SEED_CFG6_NOISE, 1e-4)
    gxy = g.flat_shape[0] * g.flat_shape[1]
    E = 0.1 * wl.counter_normal(wl.SEED_CFG6_E, 0, 2 * gxy)
    Ex, Ey = E[:gxy].reshape(g.flat_shape[:2]), E[gxy:].reshape(g.flat_shape[:2])
    fd = dev(f)
    r = ctx.rhs(fd, dev(Ex), dev(Ey))
    assert ctx.last_kernel == "rhs4_tile<8>"
    G = g.flat_shape[0]
    pick = (wl.counter_uniform(wl.SEED_CFG6_E, 1 << 20, 4 * 400) * G).astype(np.int64).reshape(400, 4)
    edge = np.array([0, 3, 4, 31, 32, 63, 64, 127, G - 4, G - 1])
    pick[:120] = edge[(pick[:120] % edge.size)]                      # element / tile / box boundaries in every dimension
    idx = torch.from_numpy(pick).cuda()
    got = r[idx[:, 0], idx[:, 1], idx[:, 2], idx[:, 3]].cpu().numpy()
    scale = float(r.abs().max().item())
    for k in range(pick.shape[0]):
        want = o4.rhs_at(g, f, Ex, Ey, tuple(int(i) for i in pick[k]))
        assert abs(got[k] - want) < 1e-12 * scale, (pick[k], got[k], want)
    rho = ctx.density(fd).cpu().numpy()
    wu, wv = np.tile(g.w[2] / g.J[2], g.nelem[2]), np.tile(g.w[3] / g.J[3], g.nelem[3])
    for gx, gy in [(0, 0), (5, 77), (127, 64), (64, 127)]:
        assert abs(rho[gx, gy] - wu @ f[gx, gy] @ wv) < 1e-13 * abs(rho[gx, gy])
    ctx.close()


# ---------------------------------------------------------------------------------------------
# physics on the GPU path: signs and coupling of the second space dimension, end to end
# ---------------------------------------------------------------------------------------------
def _landau_rate(ctx, f, dt, per, nsamp):
    amp = []
    for _ in range(nsamp):
        ctx.ssprk3_run(f, dt, per, True)
        Ex, Ey = ctx.poisson_E(ctx.density(f))
        amp.append(float(torch.sqrt(Ex * Ex + Ey * Ey).max()))
    amp = np.array(amp); t = dt * per * (np.arange(nsamp) + 1)
    pk = [i for i in range(1, nsamp - 1) if amp[i] > amp[i - 1] and amp[i] > amp[i + 1]]
    assert len(pk) >= 6
    return np.polyfit(t[pk], np.log(amp[pk]), 1)[0], float(np.mean(np.diff(t[pk])))


@pytest.mark.parametrize("direction", ["y", "oblique"])
def test_landau_damping_2d2v(direction):
    """Unmagnetised Maxwellian with a 1 % density wave of |k| = 0.5 along y, or along the diagonal of a square box: the field
    decays at the textbook Landau rate -0.1533 with omega_r = 1.4156 (as config 1; a wrong sign of E_y or of a_v grows
    instead), and E(0) = -(A/|k|^2) k sin(k.x) (closed form)."""
    if direction == "y":
        N, kx, ky = (2, 16, 8, 32), 0.0, 0.5
        hi_xy = (4 * math.pi, 4 * math.pi)
    else:
        N, kx, ky = (16, 16, 32, 32), 0.5 / math.sqrt(2.0), 0.5 / math.sqrt(2.0)
        hi_xy = (2 * math.pi / kx, 2 * math.pi / ky)
    ctx = api().DG4Context(N, (4, 4, 4, 4), (0.0, 0.0, -6.0, -6.0), hi_xy + (6.0, 6.0), bc=(0, 0, 1, 1), omega_c=0.0, pmax=(4, 4))
    x, y, u, v = (ctx.nodes(d) for d in range(4))
    arg = kx * x[:, None] + ky * y[None, :]
    maxw = np.exp(-0.5 * (u[:, None] ** 2 + v[None, :] ** 2)) / (2 * math.pi)
    f = torch.from_numpy((1.0 + 0.01 * np.cos(arg))[:, :, None, None] * maxw[None, None]).cuda()
    Ex, Ey = ctx.poisson_E(ctx.density(f))
    k2 = kx * kx + ky * ky
    assert np.max(np.abs(Ex.cpu().numpy() + 0.01 * kx / k2 * np.sin(arg))) < 2e-6
    assert np.max(np.abs(Ey.cpu().numpy() + 0.01 * ky / k2 * np.sin(arg))) < 2e-6
    assert 0.008 < ctx.max_stable_dt(0.05) < 0.02             # sum_d |a_d| dt / Delta_d against the n = 4 RK3 limit 0.13
    rate, period = _landau_rate(ctx, f, 0.008, 6, 420)
    assert -0.165 < rate < -0.143, rate
    assert abs(period - math.pi / 1.4156) < 0.08
    assert ctx.last_kernel == "rhs4_tile<8>"
    ctx.close()


def test_cyclotron_rotation_2d2v():
    """E = 0, uniform in x and y: f(u, v, t) = f0(u cos th + v sin th, -u sin th + v cos th), th = omega_c t (counter-clockwise,
    reading C15): a blob at (u, v) = (1.5, 0) is at (0, 1.5) after a quarter gyration."""
    ctx = api().DG4Context((1, 1, 16, 16), (4, 4, 4, 4), (0.0, 0.0, -6.0, -6.0), (1.0, 1.0, 6.0, 6.0), bc=(0, 0, 1, 1), omega_c=1.0)
    u, v = ctx.nodes(2), ctx.nodes(3)
    blob = lambda a, b: np.exp(-((a - 1.5) ** 2 + b ** 2) / (2 * 0.6 ** 2))
    f0 = np.broadcast_to(blob(u[:, None], v[None, :]), ctx.flat_shape).copy()
    steps = 400
    dt = 0.5 * math.pi / steps
    f = ctx.ssprk3_run(torch.from_numpy(f0).cuda(), dt, steps, False).cpu().numpy()
    th = 0.5 * math.pi
    U, V = u[:, None], v[None, :]
    ccw = blob(U * math.cos(th) + V * math.sin(th), -U * math.sin(th) + V * math.cos(th))
    cw = blob(U * math.cos(th) - V * math.sin(th), U * math.sin(th) + V * math.cos(th))
    assert np.max(np.abs(f - ccw[None, None])) < 0.02
    assert np.max(np.abs(f - cw[None, None])) > 0.5
    ctx.close()


def test_density_with_more_than_65535_space_nodes():
    """G_x G_y = 66 564 (x, y) pairs: the density kernels run in slices of the launch grid; sampled against the definition."""
    N, n = (43, 43, 1, 2), (6, 6, 2, 4)
    g, ctx = make_pair(N, n)
    dof = int(np.prod(g.flat_shape))
    f = wl.counter_uniform_chunked(wl.SEED_CFG6_NOISE, dof).reshape(g.flat_shape)
    rho = ctx.density(dev(f)).cpu().numpy()
    assert relerr(rho, o4.density(g, f)) < 1e-13
    ctx.close()



# ---------------------------------------------------------------------------------------------
# x-slab halo boundary (DG_BC_HALO, dg4_set_xhalo): two slabs on one GPU against the UNSHARDED oracle
# ---------------------------------------------------------------------------------------------
XSLAB_CASES = [
    # N, n, bc0 of the global grid, x-elements of slab 0, expected kernel
    ((5, 2, 2, 3), (3, 4, 5, 2), 0, 2, "rhs4_generic"),
    ((4, 3, 2, 8), (4, 4, 4, 4), 0, 1, "rhs4_tile"),
    ((4, 2, 3, 4), (4, 4, 4, 4), 1, 3, "rhs4_tile"),
    ((3, 2, 2, 2), (6, 6, 6, 6), 0, 1, "rhs4_elem"),
    ((3, 2, 1, 2), (8, 8, 8, 8), 0, 2, "rhs4_line"),
    ((2, 1, 2, 2), (8, 8, 8, 8), 1, 1, "rhs4_line"),
]


def _slab(A, N, n, lo, hi, bc, omega_c, e0, e1):
    dx = (hi[0] - lo[0]) / N[0]
    return A.DG4Context((e1 - e0,) + tuple(N[1:]), n, (lo[0] + e0 * dx,) + tuple(lo[1:]), (lo[0] + e1 * dx,) + tuple(hi[1:]),
                        bc=(A.BC_HALO,) + tuple(bc[1:]), omega_c=omega_c)


def _fill_halos(halos, parts, bc0):
    """halos[s][0] <- last x plane of the slab below, halos[s][1] <- first plane of the slab above (periodic wrap, or
    zeros at the outer faces for zero inflow): device copies in stream order."""
    S = len(parts)
    for s in range(S):
        below, above = parts[(s - 1) % S], parts[(s + 1) % S]
        if s > 0 or bc0 == 0:
            halos[s][0].copy_(below[-1])
        else:
            halos[s][0].zero_()
        if s < S - 1 or bc0 == 0:
            halos[s][1].copy_(above[0])
        else:
            halos[s][1].zero_()


@pytest.mark.parametrize("N,n,bc0,split,kernel", XSLAB_CASES)
def test_xslab_halo_stage_matches_unsharded_oracle(N, n, bc0, split, kernel):
    """dg4_rk_stage on two x-slabs (exterior x planes from dg4_set_xhalo) = the stage on the whole grid (oracle)."""
    A = api()
    bc = (bc0, 0, 1, 1)
    g = o4.make_grid(N, n, LO, HI, bc=bc, omega_c=0.8)
    f, Ex, Ey = seeded_inputs(g)
    fn = wl.counter_uniform_chunked(wl.SEED_CFG6_NOISE + 1, f.size).reshape(f.shape)
    c0, c1, dt = 0.75, 0.25, 1e-3
    ref = c0 * fn + c1 * (f + dt * o4.rhs(g, f, Ex, Ey))
    cuts = [(0, split), (split, N[0])]
    ctxs = [_slab(A, N, n, LO, HI, bc, 0.8, a, b) for a, b in cuts]
    fs = [dev(f[a * n[0]:b * n[0]]) for a, b in cuts]
    halos = [torch.empty((2,) + tuple(f.shape[1:]), dtype=torch.float64, device="cuda") for _ in cuts]
    _fill_halos(halos, fs, bc0)
    for (a, b), ctx, fsl, h in zip(cuts, ctxs, fs, halos):
        with pytest.raises(A.DGError):
            ctx.rhs(fsl, None, None)                        # halo context without a halo buffer
        ctx.set_xhalo(h)
        sl = slice(a * n[0], b * n[0])
        rho = torch.empty(fsl.shape[:2], dtype=torch.float64, device="cuda")
        out = ctx.rk_stage(fsl, dev(fn[sl]), dev(Ex[sl]), dev(Ey[sl]), torch.empty_like(fsl), c0, c1, dt, rho_out=rho)
        assert ctx.last_kernel.startswith(kernel), ctx.last_kernel
        assert relerr(out.cpu().numpy(), ref[sl]) < 1e-12 * max(1.0, np.abs(ref).max() / np.abs(ref[sl]).max())
        assert relerr(rho.cpu().numpy(), o4.density(g, ref)[sl]) < 1e-12
        r = ctx.rhs(fsl, dev(Ex[sl]), dev(Ey[sl])).cpu().numpy()
        assert relerr(r, o4.rhs(g, f, Ex, Ey)[sl]) < 1e-12
        ctx.close()


def test_xslab_two_slabs_self_consistent_steps():
    """Two SSP-RK3 steps with the 2-D Poisson solve at every stage, the phase space cut into two x-slabs: per stage the
    slab densities are joined, the GLOBAL field is solved on an (x, y)-only context, the face planes are exchanged and each
    slab runs dg4_rk_stage -- against oracle.vlasov2d2v.ssprk3_step on the whole grid."""
    A = api()
    N, n, k = (4, 2, 2, 8), (4, 4, 4, 4), 0.1
    lo, hi = (0.0, 0.0, -8.5, -8.5), (2 * math.pi / k, 2 * math.pi / k, 8.5, 8.5)
    bc = (0, 0, 1, 1)
    g = o4.make_grid(N, n, lo, hi, bc=bc, omega_c=1.0, pmax=(3, 2))
    x, y, u, v = [c.reshape(-1) for c in g.coords]
    f0 = wl.add_uniform_noise(wl.ring2d_f0(x, y, u, v, k, k), wl.SEED_CFG6_NOISE, 1e-3)
    dt, nsteps = 1e-3, 2
    fo = f0
    for _ in range(nsteps):
        fo = o4.ssprk3_step(g, fo, dt)
    cuts = [(0, 1), (1, 4)]
    ctxs = [_slab(A, N, n, lo, hi, bc, 1.0, a, b) for a, b in cuts]
    field = A.DG4Context((N[0], N[1], 1, 1), (n[0], n[1], 2, 2), lo, hi, bc=(0, 0, 1, 1), omega_c=1.0, pmax=(3, 2))
    mk = lambda: [torch.empty((b - a) * n[0], *f0.shape[1:], dtype=torch.float64, device="cuda") for a, b in cuts]
    fs, u1, u2 = [dev(f0[a * n[0]:b * n[0]]) for a, b in cuts], mk(), mk()
    halos = [torch.empty((2,) + tuple(f0.shape[1:]), dtype=torch.float64, device="cuda") for _ in cuts]
    rho = torch.empty(f0.shape[:2], dtype=torch.float64, device="cuda")
    rho_parts = [rho[a * n[0]:b * n[0]] for a, b in cuts]
    for ctx, h in zip(ctxs, halos):
        ctx.set_xhalo(h)

    def stage(src, fn, dst, stage_no, rho_known):
        c0, c1 = A.ssprk3_stage_coeffs(stage_no)
        if not rho_known:
            for ctx, s, r in zip(ctxs, src, rho_parts):
                ctx.density(s, r)
        Ex, Ey = field.poisson_E(rho)
        _fill_halos(halos, src, 0)
        for (a, b), ctx, s, fnn, d, r in zip(cuts, ctxs, src, fn, dst, rho_parts):
            sl = slice(a * n[0], b * n[0])
            ctx.rk_stage(s, fnn if c0 != 0.0 else None, Ex[sl].contiguous(), Ey[sl].contiguous(), d, c0, c1, dt, rho_out=r)

    for i in range(nsteps):
        stage(fs, fs, u1, 0, i > 0)
        stage(u1, fs, u2, 1, True)
        stage(u2, fs, fs, 2, True)
    got = np.concatenate([t.cpu().numpy() for t in fs], axis=0)
    assert relerr(got, fo) < 1e-11
    for c in ctxs + [field]:
        c.close()


def test_xslab_halo_argument_checks():
    A = api()
    ctx = A.DG4Context((2, 2, 2, 2), (4,) * 4, LO, HI, bc=(0, 0, 1, 1))
    with pytest.raises(A.DGError):
        ctx.set_xhalo(torch.zeros((2, 8, 8, 8), dtype=torch.float64, device="cuda"))      # not a halo context
    ctx.close()
    with pytest.raises(A.DGError):
        A.DG4Context((2, 2, 2, 2), (4,) * 4, LO, HI, bc=(0, A.BC_HALO, 1, 1))             # only x can be a slab
    slab = A.DG4Context((2, 2, 2, 2), (4,) * 4, LO, HI, bc=(A.BC_HALO, 0, 1, 1))
    f = torch.zeros(slab.flat_shape, dtype=torch.float64, device="cuda")
    with pytest.raises(A.DGError):
        slab.ssprk3_run(f, 1e-3, 1, True)                                                  # the Poisson solve is global
    slab.set_xhalo(torch.zeros((2,) + tuple(f.shape[1:]), dtype=torch.float64, device="cuda"))
    with pytest.raises(A.DGError, match="stage by stage"):
        slab.ssprk3_run(f, 1e-3, 1, False)          # one halo buffer cannot serve three stage inputs: dg4_rk_stage only
    slab.close()
