"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times: sampled outputs
against the pointwise oracle, plus whole-array properties (mass conservation, density, field)."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import vlasov as ov, pointwise as opw, fourier as ofr   # noqa: E402
import workloads as wl                                               # noqa: E402

K = 0.1


def api():
    from paper_2202_13532_b200 import api as _api
    return _api


def relerr(a, b):
    return float(np.max(np.abs(np.asarray(a) - np.asarray(b))) / max(np.max(np.abs(b)), 1e-300))


def sample_nodes(shape, count, seed):
    """Random nodes plus every kind of boundary node (first/last element and node of each dimension)."""
    rng = np.random.default_rng(seed)
    pts = [tuple(int(rng.integers(0, s)) for s in shape) for _ in range(count)]
    edge = [0, 1, 7, 8]
    for d in range(len(shape)):
        for e in edge + [shape[d] - 1 - q for q in edge]:
            p = [int(rng.integers(0, s)) for s in shape]
            p[d] = e % shape[d]
            pts.append(tuple(p))
    return pts


def test_config3_full_grid_rhs_density_field():
    """512^3 production grid (config 3): tiled kernel, one RHS with the self-consistent E."""
    nelem, order = (64, 64, 64), (8, 8, 8)
    lo, hi = (0.0, -8.5, -8.5), (2 * math.pi / K, 8.5, 8.5)
    ctx = api().DGContext(nelem, order, lo, hi, bc=(0, 1, 1), omega_c=1.0, pmax=64)
    g = ov.Grid(nelem=nelem, order=order, lo=lo, hi=hi, bc=(0, 1, 1), omega_c=1.0, pmax=64)
    f0 = wl.add_uniform_noise(wl.ring_f0(ctx.nodes(0), ctx.nodes(1), ctx.nodes(2), K), wl.SEED_CFG3_NOISE, 1e-4)
    fd = torch.from_numpy(f0).cuda()
    # density: whole array against the oracle
    rho = ctx.density(fd).cpu().numpy()
    rho_o = ov.density(g, f0)
    assert relerr(rho, rho_o) <= 1e-13
    E = ctx.poisson_E(torch.from_numpy(rho_o).cuda()).cpu().numpy()
    E_o = ofr.poisson_E(lo[0], hi[0], g.x_nodes(), ofr.fourier_project(g.T, rho_o))
    assert relerr(E, E_o) <= 1e-12
    out = ctx.rhs(fd, torch.from_numpy(E_o).cuda())
    assert ctx.last_kernel.startswith("rhs_tiled<8,")
    out_h = out.cpu().numpy()
    scale = np.max(np.abs(out_h))
    for p in sample_nodes(g.flat_shape, 150, 3):
        ref = opw.rhs_at(g, f0, E_o, p)
        assert abs(out_h[p] - ref) <= 1e-12 * scale, (p, out_h[p], ref)
    # property that holds at any size: d(mass)/dt = - outflow through the zero-inflow velocity boundaries
    W = [np.tile(g.w[d] / g.J[d], g.nelem[d]) for d in range(3)]
    dm = np.einsum("i,j,k,ijk->", W[0], W[1], W[2], out_h)
    u, v = g.coords[1].reshape(-1), g.coords[2].reshape(-1)
    au = -E_o[:, None] - g.omega_c * v[None, :]          # [gx, gv]
    av = g.omega_c * u                                    # [gu]
    outflow = (np.einsum("i,k,ik,ik->", W[0], W[2], np.maximum(au, 0), f0[:, -1, :])
               + np.einsum("i,k,ik,ik->", W[0], W[2], np.maximum(-au, 0), f0[:, 0, :])
               + np.einsum("i,j,ij->", W[0], W[1] * np.maximum(av, 0), f0[:, :, -1])
               + np.einsum("i,j,ij->", W[0], W[1] * np.maximum(-av, 0), f0[:, :, 0]))
    assert abs(dm + outflow) < 1e-9 * max(abs(outflow), 1e-12), (dm, outflow)
    # the 1000-step production run of config 3 (dt = 5e-4, Poisson at every stage): mass, finiteness and field monitored
    # (the oracle cannot follow 1000 steps at this size; the 128^3 replica below carries the parity claim)
    Wx = torch.from_numpy(W[0]).cuda()
    mass0 = float((ctx.density(fd) * Wx).sum())
    l0 = ctx.launch_count
    for _ in range(10):
        ctx.ssprk3_run(fd, 5e-4, 100, True)
        assert bool(torch.isfinite(fd).all())
    assert ctx.launch_count - l0 == 10 * (1 + 100 * 6)      # per call: one density pass, then field + RHS per stage
    rho1 = ctx.density(fd)
    mass1 = float((rho1 * Wx).sum())
    # the seeded noise (1e-4, zero mean) reaches the zero-inflow velocity boundary: what leaves is a sum of ~1e6 terms of
    # random sign, each <= a dt w f ~ 1e-9 of the mass -- relative drift ~1e-6, not round-off
    assert abs(mass1 - mass0) < 5e-6 * mass0
    assert abs(float(rho1.mean()) - 1.0) < 1e-3 and float(ctx.poisson_E(rho1).abs().max()) < 0.2
    # stays within the initial range (ring peak 0.03566 x 1.01, noise +-1e-4) up to grid-scale over/undershoots of the noise
    # (upwind DG is not monotone: the element-scale noise over/undershoots by a few times its amplitude)
    assert float(fd.min()) > -1e-3 and float(fd.max()) < 0.03566 * 1.01 + 1e-3
    ctx.close()


@pytest.mark.parametrize("n,N", [(8, 50), (4, 100), (6, 67), (10, 40)])
def test_config4_full_size_rhs_whole_array(n, N):
    """GL-order sweep (config 4) at ~64M DOF: U(0,1) f, N(0,0.1^2) E.  The whole array against the array oracle (every tile,
    the ragged tile tails of N = 50 / 67 / 100 included), and sampled nodes against the scalar-loop oracle as a second opinion."""
    nelem, order = (N, N, N), (n, n, n)
    lo, hi = (0.0, -8.5, -8.5), (2 * math.pi / K, 8.5, 8.5)
    ctx = api().DGContext(nelem, order, lo, hi, bc=(0, 1, 1), omega_c=1.0, workspace=False)
    g = ov.Grid(nelem=nelem, order=order, lo=lo, hi=hi, bc=(0, 1, 1), omega_c=1.0, pmax=2)
    f = wl.uniform_field(g.flat_shape, wl.SEED_CFG4_F)
    E = wl.normal_E(g.flat_shape[0], wl.SEED_CFG4_E)
    out = ctx.rhs(torch.from_numpy(f).cuda(), torch.from_numpy(E).cuda())
    assert ctx.last_kernel.startswith("rhs_tiled<%d," % n)
    out_h = out.cpu().numpy()
    scale = np.max(np.abs(out_h))
    for p in sample_nodes(g.flat_shape, 80, n):
        ref = opw.rhs_at(g, f, E, p)
        assert abs(out_h[p] - ref) <= 1e-12 * scale, (p, out_h[p], ref)
    ctx.close()
    del out
    ref = ov.rhs(g, f, E)
    ref -= out_h
    assert float(np.max(np.abs(ref))) <= 1e-12 * scale


def test_config2_grid_one_full_step():
    """256^3 (config 2 grid): one self-consistent SSP-RK3 step, whole array against the oracle."""
    nelem, order = (32, 32, 32), (8, 8, 8)
    lo, hi = (0.0, -8.5, -8.5), (2 * math.pi / K, 8.5, 8.5)
    ctx = api().DGContext(nelem, order, lo, hi, bc=(0, 1, 1), omega_c=1.0, pmax=32)
    g = ov.Grid(nelem=nelem, order=order, lo=lo, hi=hi, bc=(0, 1, 1), omega_c=1.0, pmax=32)
    f0 = wl.ring_f0(ctx.nodes(0), ctx.nodes(1), ctx.nodes(2), K)
    fd = torch.from_numpy(f0).cuda()
    ctx.ssprk3_run(fd, 1e-3, 1, True)
    fo = ov.ssprk3_step(g, f0, 1e-3)
    assert relerr(fd.cpu().numpy(), fo) <= 1e-12
    # literal config-2 time step (dt = 0.005, unstable over 100 steps, C22): 1 step is still a parity case
    fd = torch.from_numpy(f0).cuda()
    ctx.ssprk3_run(fd, 5e-3, 1, True)
    assert relerr(fd.cpu().numpy(), ov.ssprk3_step(g, f0, 5e-3)) <= 1e-12
    ctx.close()


def test_config2_replica_100_steps():
    """north_star: <= 1e-10 after 100 RK steps. Config-2 physics on a 16^3-element (128^3 DOF) replica."""
    nelem, order = (16, 16, 16), (8, 8, 8)
    lo, hi = (0.0, -8.5, -8.5), (2 * math.pi / K, 8.5, 8.5)
    ctx = api().DGContext(nelem, order, lo, hi, bc=(0, 1, 1), omega_c=1.0, pmax=16)
    g = ov.Grid(nelem=nelem, order=order, lo=lo, hi=hi, bc=(0, 1, 1), omega_c=1.0, pmax=16)
    f0 = wl.ring_f0(ctx.nodes(0), ctx.nodes(1), ctx.nodes(2), K)
    dt = 2e-3
    assert dt < ctx.max_stable_dt(0.2)
    fd = torch.from_numpy(f0).cuda()
    ctx.ssprk3_run(fd, dt, 100, True)
    fo = f0.copy()
    for _ in range(100):
        fo = ov.ssprk3_step(g, fo, dt)
    assert np.isfinite(fo).all()
    assert relerr(fd.cpu().numpy(), fo) <= 1e-10
    ctx.close()


def test_config5_full_batch_sampled_against_oracle():
    """Config 5 at full size in the launch configuration bench.py times (auto -> field_fft_kernel, 4096 vectors x 16 384
    nodes, modes <= 8192, persistent grid): c_p for every p and E at every node of sampled vectors (first, last, two
    interior) against the oracle's dense definition, walked in slices of 512 modes (the full T is 2 GB)."""
    A = api()
    N, n, lo, hi, pmax, batch = 2048, 8, 0.0, 2 * math.pi, 8192, 4096
    ctx = A.DGContext((N,), (n,), (lo,), (hi,), pmax=pmax, field_batch=batch, workspace=False)
    x = ctx.nodes(0)
    assert np.array_equal(x, ofr.node_coordinates(lo, hi, N, n)) or relerr(x, ofr.node_coordinates(lo, hi, N, n)) < 1e-15
    sample = [0, 1777, 2048, batch - 1]
    rows = {b: wl.cosine_sum_density(x, 1, wl.SEED_CFG5, b0=b)[0][0] for b in sample}
    # the rest of the batch: the same recipe evaluated on the device would need the generator there; the parity claim is
    # on the sampled vectors, the others only have to be finite and independent of their position in the batch
    filler = wl.cosine_sum_density(x, 8, wl.SEED_CFG5, b0=5000)[0]
    rho = torch.from_numpy(np.tile(filler, (batch // 8, 1))).cuda()
    for b, r in rows.items():
        rho[b] = torch.from_numpy(r).cuda()
    c = ctx.fourier_project(rho)
    E = ctx.poisson_E(rho)
    torch.cuda.synchronize()
    assert ctx.last_field_kernel == "field_fft_kernel"          # what `auto` takes on this grid
    cs = c[sample].cpu().numpy(); cs = cs[..., 0] + 1j * cs[..., 1]
    Es = E[sample].cpu().numpy()
    R = np.stack([rows[b] for b in sample])
    co = np.empty((len(sample), pmax + 1), dtype=np.complex128)
    for p0 in range(0, pmax + 1, 512):
        p1 = min(pmax, p0 + 511)
        co[:, p0:p1 + 1] = ofr.fourier_project(ofr.transform_tensor(lo, hi, N, n, p1, p_first=p0), R)
    assert relerr(cs, co) <= 1e-12
    # conditioned bound (reading C26): |E| ~ 1e-3 here while round-off enters at eps |rho| with |rho| ~ 1
    Eo = ofr.poisson_E(lo, hi, x, co)
    assert np.max(np.abs(Es - Eo)) <= 1e-12 * np.max(np.abs(Eo)) + 1e-14 * np.max(np.abs(R)) * (hi - lo) / (2 * math.pi)
    # position independence: the filler rows repeat every 8 vectors
    Eall = E.reshape(batch // 8, 8, -1)
    keep = [i for i in range(batch // 8) if not any(8 * i <= b < 8 * i + 8 for b in sample)]
    assert torch.equal(Eall[keep[0]], Eall[keep[-1]]) and torch.equal(Eall[keep[0]], Eall[keep[len(keep) // 2]])
    assert bool(torch.isfinite(E).all()) and bool(torch.isfinite(c).all())
    ctx.close()


def test_config5_full_batch_survey_slices():
    """Config 5 at full size with the REAL batch (all 4096 vectors from the recipe, no filler), compared on the two slices
    SURVEY 8(d) prescribes (the dense oracle for the whole batch is 2.2e12 flop per contraction): (i) 64 vectors spread over
    the batch on all 8193 modes (c_p; E at every node for 16 of them -- the oracle's synthesis is a loop over the modes),
    (ii) all 4096 vectors on a 256-mode slice of c_p, taken across the m <= 1024 band edge of the recipe.
    Last: the FFT-factorised kernel against the dense DMMA kernel over the whole batch -- a kernel-vs-kernel cross-check
    (both are the product's; it shows that the 4032 vectors the oracle did not visit get the same treatment), NOT parity."""
    A = api()
    N, n, lo, hi, pmax, batch = 2048, 8, 0.0, 2 * math.pi, 8192, 4096
    ctx = A.DGContext((N,), (n,), (lo,), (hi,), pmax=pmax, field_batch=batch)
    x = ctx.nodes(0)
    R = wl.cosine_sum_density(x, batch, wl.SEED_CFG5)[0]
    rho = torch.from_numpy(R).cuda()
    c = ctx.fourier_project(rho)
    E = ctx.poisson_E(rho)
    torch.cuda.synchronize()
    assert ctx.last_field_kernel == "field_fft_kernel"
    # (i) 64 vectors, every mode
    sample = list(range(0, batch, 65))[:63] + [batch - 1]
    assert len(sample) == 64
    cs = c[sample].cpu().numpy(); cs = cs[..., 0] + 1j * cs[..., 1]
    co = np.empty((64, pmax + 1), dtype=np.complex128)
    for p0 in range(0, pmax + 1, 512):
        p1 = min(pmax, p0 + 511)
        co[:, p0:p1 + 1] = ofr.fourier_project(ofr.transform_tensor(lo, hi, N, n, p1, p_first=p0), R[sample])
    assert relerr(cs, co) <= 1e-12
    sub = sample[::4]
    Eo = ofr.poisson_E(lo, hi, x, co[::4])
    Es = E[sub].cpu().numpy()
    # conditioned bound (reading C26), as in the sampled test above
    bound = 1e-12 * np.max(np.abs(Eo)) + 1e-14 * np.max(np.abs(R)) * (hi - lo) / (2 * math.pi)
    assert np.max(np.abs(Es - Eo)) <= bound
    # (ii) every vector, modes 896..1151
    p0, p1 = 896, 1151
    ca = c[:, p0:p1 + 1].cpu().numpy(); ca = ca[..., 0] + 1j * ca[..., 1]
    cao = ofr.fourier_project(ofr.transform_tensor(lo, hi, N, n, p1, p_first=p0), R)
    assert relerr(ca, cao) <= 1e-12
    # kernel-vs-kernel cross-check over the whole batch (not parity): dense DMMA contraction against the FFT factorisation
    ctx.set_option(A.OPT_FIELD_KERNEL, A.FIELD_DMMA)
    c2 = ctx.fourier_project(rho)
    assert ctx.last_field_kernel == "field_gemm_dmma_kernel"
    cscale = float(torch.sqrt(c2[..., 0] ** 2 + c2[..., 1] ** 2).max())
    assert float((c2 - c).abs().max()) <= 2e-12 * cscale
    del c2
    E2 = ctx.poisson_E(rho)
    assert float((E2 - E).abs().max()) <= 2 * bound
    ctx.close()
