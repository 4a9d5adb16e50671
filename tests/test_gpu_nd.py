"""GPU parity of the dimension-generic path (include/dgvlasov_nd.h, dgn_*) against oracle/vlasov_nd.py on the same seeded
inputs, for every (d_x, d_v) with 1 <= d_x <= d_v <= 3, and against the dedicated 1D2V / 2D2V entry points on their shapes.
Tolerances as for the other paths."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import vlasov_nd as on       # noqa: E402
import workloads as wl                   # noqa: E402


def api():
    from paper_2202_13532_b200 import api as _api
    return _api


def relerr(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rnd(shape, seed):
    return wl.counter_uniform_chunked(seed, int(np.prod(shape))).reshape(shape)


# dx, dv, nelem, order, lo, hi, bc, omega_c, pmax
CASES = [
    (1, 1, (5, 6), (4, 3), (0.0, -3.0), (4 * math.pi, 3.0), (0, 1), 0.0, (4,)),
    (1, 2, (3, 2, 3), (4, 3, 5), (0.0, -2.0, -2.5), (2.0, 2.0, 2.5), (0, 1, 0), 0.8, (3,)),
    (1, 3, (3, 2, 2, 2), (3, 4, 3, 3), (0.0, -2.0, -2.0, -1.0), (3.0, 2.0, 2.0, 1.0), (0, 1, 1, 0), 1.1, (3,)),
    (2, 2, (2, 3, 2, 2), (3, 2, 4, 3), (0.0, -1.0, -2.0, -2.5), (2.0, 2.0, 2.0, 2.5), (0, 0, 1, 1), 0.6, (2, 3)),
    (2, 3, (2, 2, 2, 2, 2), (3, 3, 3, 2, 3), (0.0, 0.0, -2.0, -2.0, -1.5), (2.0, 3.0, 2.0, 2.0, 1.5), (0, 0, 1, 1, 1), 0.9, (2, 2)),
    (3, 3, (2, 2, 2, 2, 2, 2), (3, 2, 3, 2, 3, 2), (0.0, 0.0, 0.0, -1.0, -1.5, -2.0), (1.0, 2.0, 1.5, 1.0, 1.5, 2.0), (0, 0, 0, 1, 1, 1), 0.7, (2, 2, 1)),
    (3, 3, (2, 1, 2, 2, 2, 1), (2, 4, 2, 3, 2, 4), (0.0, 0.0, 0.0, -1.0, -1.5, -2.0), (1.0, 2.0, 1.5, 1.0, 1.5, 2.0), (0, 0, 0, 0, 0, 0), 0.7, (1, 1, 2)),
]


def make_pair(case, mass_mode=0):
    dx, dv, nelem, order, lo, hi, bc, wc, pmax = case
    g = on.make_grid(dx, dv, nelem, order, lo, hi, bc=bc, omega_c=wc, pmax=pmax, mass_mode=mass_mode)
    ctx = api().DGNContext(dx, dv, nelem, order, lo, hi, bc=bc, omega_c=wc, pmax=pmax, mass_mode=mass_mode)
    return g, ctx


@pytest.mark.parametrize("case", CASES)
@pytest.mark.parametrize("mass_mode", [0, 1])
def test_rhs_density_field_match_oracle(case, mass_mode):
    g, ctx = make_pair(case, mass_mode)
    dx = case[0]
    for d in range(g.ndim):
        assert np.max(np.abs(ctx.nodes(d) - g.coords[d].reshape(-1))) < 1e-14
    f = rnd(g.flat_shape, 101)
    E = np.stack([0.6 * rnd(g.flat_shape[:dx], 102 + i) - 0.3 for i in range(dx)])
    r = ctx.rhs(dev(f), dev(E)).cpu().numpy()
    assert relerr(r, on.rhs(g, f, list(E))) < 1e-12
    r0 = ctx.rhs(dev(f), None).cpu().numpy()
    assert relerr(r0, on.rhs(g, f, None)) < 1e-12
    rho = ctx.density(dev(f)).cpu().numpy()
    rho_o = on.density(g, f)
    assert relerr(rho, rho_o) < 1e-13
    Eg = ctx.poisson_E(dev(rho_o)).cpu().numpy()
    Eo = on.poisson_E(g, on.fourier_project(g, rho_o))
    scale = max(np.max(np.abs(e)) for e in Eo)
    for i in range(dx):
        assert np.max(np.abs(Eg[i] - Eo[i])) < 1e-12 * scale, i
    fn = rnd(g.flat_shape, 103)
    out = ctx.rk_stage(dev(f), dev(fn), dev(E), torch.empty_like(dev(f)), 0.75, 0.25, 1e-3).cpu().numpy()
    assert relerr(out, 0.75 * fn + 0.25 * (f + 1e-3 * on.rhs(g, f, list(E)))) < 1e-13
    ctx.close()


@pytest.mark.parametrize("case", [CASES[2], CASES[4], CASES[5]])
def test_self_consistent_steps_match_oracle(case):
    """Two SSP-RK3 steps with the d_x-dimensional Poisson solve at every stage."""
    g, ctx = make_pair(case)
    f0 = 0.5 + rnd(g.flat_shape, 111)
    fd = dev(f0)
    ctx.ssprk3_run(fd, 1e-3, 2, True)
    fo = f0
    for _ in range(2):
        fo = on.ssprk3_step(g, fo, 1e-3)
    assert relerr(fd.cpu().numpy(), fo) < 1e-12
    ctx.close()


def test_agrees_with_the_dedicated_1d2v_and_2d2v_paths():
    """The same grids through dg_* (tiled kernel), dg4_* (tiled kernel) and dgn_*: three code paths, one result."""
    A = api()
    nelem, order, lo, hi = (3, 2, 4), (8, 8, 8), (0.0, -4.0, -4.0), (2 * math.pi, 4.0, 4.0)
    c3 = A.DGContext(nelem, order, lo, hi, bc=(0, 1, 1), omega_c=1.0, pmax=3)
    cn = A.DGNContext(1, 2, nelem, order, lo, hi, bc=(0, 1, 1), omega_c=1.0, pmax=(3,))
    f0 = 0.5 + rnd(c3.flat_shape, 121)
    a, b = dev(f0), dev(f0)
    c3.ssprk3_run(a, 1e-3, 2, True)
    cn.ssprk3_run(b, 1e-3, 2, True)
    assert c3.last_kernel.startswith("rhs_tiled")
    assert relerr(b.cpu().numpy(), a.cpu().numpy()) < 1e-12
    c3.close(); cn.close()
    N4, n4, lo4, hi4 = (2, 2, 2, 4), (4, 4, 4, 4), (0.0, 0.0, -4.0, -4.0), (2 * math.pi, 3.0, 4.0, 4.0)
    c4 = A.DG4Context(N4, n4, lo4, hi4, bc=(0, 0, 1, 1), omega_c=1.0, pmax=(2, 2))
    cn = A.DGNContext(2, 2, N4, n4, lo4, hi4, bc=(0, 0, 1, 1), omega_c=1.0, pmax=(2, 2))
    f0 = 0.5 + rnd(c4.flat_shape, 122)
    a, b = dev(f0), dev(f0)
    c4.ssprk3_run(a, 1e-3, 2)
    cn.ssprk3_run(b, 1e-3, 2, True)
    assert c4.last_kernel.startswith("rhs4_tile")
    assert relerr(b.cpu().numpy(), a.cpu().numpy()) < 1e-12
    c4.close(); cn.close()


def test_argument_checks():
    A = api()
    with pytest.raises(A.DGError):
        A.DGNContext(2, 1, (2, 2, 2), (3, 3, 3), (0, 0, -1), (1, 1, 1))                      # dv < dx
    with pytest.raises(A.DGError):
        A.DGNContext(1, 1, (2, 2), (3, 11), (0, -1), (1, 1))                                 # order above DG_MAX_ORDER
    ctx = A.DGNContext(1, 2, (2, 2, 2), (3, 3, 3), (0, -1, -1), (1, 1, 1), bc=(1, 1, 1), workspace=False)
    f = torch.zeros(ctx.flat_shape, dtype=torch.float64, device="cuda")
    with pytest.raises(A.DGError):
        ctx.ssprk3_run(f, 1e-3, 1, True)                                                     # no workspace
    with pytest.raises(A.DGError):
        ctx.rhs(f, None, f)                                                                  # dfdt aliases f
    ctx.close()
    ctx = A.DGNContext(1, 2, (2, 2, 2), (3, 3, 3), (0, -1, -1), (1, 1, 1), bc=(1, 1, 1))
    with pytest.raises(A.DGError):
        ctx.ssprk3_run(f, 1e-3, 1, True)                                                     # Poisson needs periodic x
    ctx.ssprk3_run(f, 1e-3, 1, False)
    ctx.close()


def test_landau_damping_2d3v_along_y():
    """End-to-end signs of the d-dimensional path: an unmagnetised Maxwellian in three velocity dimensions with a 1 % density
    wave of k = 0.5 along y (the SECOND space dimension: E_2 and a_{v_2} = -E_2 carry it).  E(0) has the closed form
    -(A/k) sin(k y), and the field decays at the textbook Landau rate -0.1533 with omega_r = 1.4156 (a wrong sign of E_2 or of
    a_{v_2} grows instead)."""
    A = api()
    ky = 0.5
    ctx = A.DGNContext(2, 3, (1, 16, 8, 32, 8), (2, 4, 3, 4, 3), (0.0, 0.0, -6.0, -6.0, -6.0), (10.0, 2 * math.pi / ky, 6.0, 6.0, 6.0),
                       bc=(0, 0, 1, 1, 1), omega_c=0.0, pmax=(1, 4))
    x, y, u, v, w = (ctx.nodes(d) for d in range(5))
    m = lambda s: np.exp(-0.5 * s * s) / math.sqrt(2 * math.pi)
    f0 = (1.0 + 0.01 * np.cos(ky * y))[None, :, None, None, None] * m(u)[None, None, :, None, None] * m(v)[None, None, None, :, None] \
        * m(w)[None, None, None, None, :] * np.ones((x.size, 1, 1, 1, 1))
    f = dev(f0)
    E = ctx.poisson_E(ctx.density(f)).cpu().numpy()
    # 5e-4 of the amplitude 0.02: the quadrature error of the Maxwellian on the coarse u and w grids (8 x 3 nodes over +-6)
    assert np.max(np.abs(E[1] + (0.01 / ky) * np.sin(ky * y)[None, :])) < 1e-5
    assert np.max(np.abs(E[0])) < 1e-12
    dt, per, nsamp = 0.008, 6, 400
    amp = []
    for _ in range(nsamp):
        ctx.ssprk3_run(f, dt, per, True)
        amp.append(float(ctx.poisson_E(ctx.density(f))[1].abs().max()))
    amp = np.array(amp); t = dt * per * (np.arange(nsamp) + 1)
    pk = [i for i in range(1, nsamp - 1) if amp[i] > amp[i - 1] and amp[i] > amp[i + 1]]
    assert len(pk) >= 6
    rate = np.polyfit(t[pk], np.log(amp[pk]), 1)[0]
    period = float(np.mean(np.diff(t[pk])))
    assert -0.165 < rate < -0.143, rate
    assert abs(period - math.pi / 1.4156) < 0.08
    ctx.close()


def test_landau_damping_3d3v_along_z():
    """The same run with the wave along z in the full 3D3V phase space: E_3 and a_{v_3} = -E_3 carry it (pinned on the oracle
    side by tests/test_oracle_nd.py's pair-swap and z-only reductions).  Closed-form E(0), textbook rate -0.1533 and
    omega_r = 1.4156; a wrong sign of E_3 or of a_{v_3} grows instead of damping."""
    A = api()
    kz = 0.5
    ctx = A.DGNContext(3, 3, (1, 1, 16, 8, 8, 32), (2, 2, 4, 3, 3, 4), (0.0, 0.0, 0.0, -6.0, -6.0, -6.0),
                       (10.0, 7.0, 2 * math.pi / kz, 6.0, 6.0, 6.0), bc=(0, 0, 0, 1, 1, 1), omega_c=0.0, pmax=(1, 1, 4))
    x, y, z, u, v, w = (ctx.nodes(d) for d in range(6))
    m = lambda s: np.exp(-0.5 * s * s) / math.sqrt(2 * math.pi)
    f0 = np.einsum("a,b,c,d,e,f->abcdef", np.ones(x.size), np.ones(y.size), 1.0 + 0.01 * np.cos(kz * z), m(u), m(v), m(w))
    f = dev(f0)
    E = ctx.poisson_E(ctx.density(f)).cpu().numpy()
    assert np.max(np.abs(E[2] + (0.01 / kz) * np.sin(kz * z)[None, None, :])) < 1e-5
    assert max(np.max(np.abs(E[0])), np.max(np.abs(E[1]))) < 1e-12
    dt, per, nsamp = 0.008, 6, 400
    amp = []
    for _ in range(nsamp):
        ctx.ssprk3_run(f, dt, per, True)
        amp.append(float(ctx.poisson_E(ctx.density(f))[2].abs().max()))
    amp = np.array(amp); t = dt * per * (np.arange(nsamp) + 1)
    pk = [i for i in range(1, nsamp - 1) if amp[i] > amp[i - 1] and amp[i] > amp[i + 1]]
    assert len(pk) >= 6
    rate = np.polyfit(t[pk], np.log(amp[pk]), 1)[0]
    period = float(np.mean(np.diff(t[pk])))
    assert -0.165 < rate < -0.143, rate
    assert abs(period - math.pi / 1.4156) < 0.08
    ctx.close()
