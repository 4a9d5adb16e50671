"""GPU parity of the FFT-factorised field solve (DG_OPT_FIELD_KERNEL = 4, dg_kernels_fft.cuh) and of dg_poisson_phi
against the oracle's dense definition (Eq. 63 / 70 / 71): c_p, E and Phi element by element,
max-norm relative error <= 1e-12."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import fourier as ofr        # noqa: E402
import workloads as wl                    # noqa: E402


def api():
    from paper_2202_13532_b200 import api as _api
    return _api


def relerr(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


# (N elements, order n, pmax, batch, lo): every radix-pass split (log2 N = 1..8), every even order, pmax below N/2,
# between N/2 and N, and several times N (modes folded onto the N bins), a shifted interval (phase e^{i k lo})
FFT_CASES = [
    (2, 4, 1, 3, 0.0), (4, 2, 9, 5, 0.0), (8, 8, 8, 2, -1.5), (16, 4, 16, 1, 0.0), (16, 6, 5, 7, 0.3),
    (32, 8, 32, 3, 0.0), (32, 10, 100, 4, 2.0), (64, 8, 64, 40, 0.0), (64, 8, 257, 9, -0.7), (128, 6, 128, 300, 0.0),
    (256, 8, 1024, 5, 0.0), (256, 4, 100, 150, 1.0), (512, 8, 700, 3, 0.0), (1024, 10, 1024, 2, 0.0),
]


@pytest.mark.parametrize("N,n,pmax,batch,lo", FFT_CASES)
def test_fft_field_matches_dense_oracle(N, n, pmax, batch, lo):
    A = api()
    hi = lo + 2 * math.pi
    ctx = A.DGContext((N,), (n,), (lo,), (hi,), pmax=pmax, field_batch=batch)
    ctx.set_option(A.OPT_FIELD_KERNEL, A.FIELD_FFT)
    x = ofr.node_coordinates(lo, hi, N, n)
    rho, _, _, _ = wl.cosine_sum_density(x, batch, wl.SEED_CFG5, mmax=max(1, min(1024, pmax // 2)))
    To = ofr.transform_tensor(lo, hi, N, n, pmax)
    co = ofr.fourier_project(To, rho)
    c = ctx.fourier_project(dev(rho)).cpu().numpy()
    assert relerr(c[..., 0] + 1j * c[..., 1], co) <= 1e-12
    E = ctx.poisson_E(dev(rho)).cpu().numpy()
    assert relerr(E, ofr.poisson_E(lo, hi, x, co)) <= 1e-12
    Phi = ctx.poisson_phi(dev(rho)).cpu().numpy()
    # Phi is the ill-conditioned output: |Phi| ~ |rho - 1| / k^2 while round-off enters at eps |rho| (the mean density 1
    # is carried through both transforms), so the bound has an absolute part eps-scaled by |rho| / k_1^2
    Phio = ofr.poisson_phi(lo, hi, x, co)
    assert np.max(np.abs(Phi - Phio)) <= 1e-12 * np.max(np.abs(Phio)) + 1e-14 * np.max(np.abs(rho)) * ((hi - lo) / (2 * math.pi)) ** 2
    assert np.array_equal(E, ctx.poisson_E(dev(rho)).cpu().numpy())          # deterministic
    ctx.close()


@pytest.mark.parametrize("kernel", [1, 2, 3])
def test_phi_dense_paths_match_oracle(kernel):
    """dg_poisson_phi through the dense kernels (simple, DMMA, DFMA): c_p (i/k_p) fed to the synthesis of Eq. 71."""
    A = api()
    N, n, pmax, batch, lo, hi = 40, 8, 60, 48, 0.0, 2 * math.pi
    ctx = A.DGContext((N,), (n,), (lo,), (hi,), pmax=pmax, field_batch=batch)
    ctx.set_option(A.OPT_FIELD_KERNEL, kernel)
    x = ofr.node_coordinates(lo, hi, N, n)
    rho, _, _, _ = wl.cosine_sum_density(x, batch, 11, mmax=20)
    co = ofr.fourier_project(ofr.transform_tensor(lo, hi, N, n, pmax), rho)
    assert relerr(ctx.poisson_phi(dev(rho)).cpu().numpy(), ofr.poisson_phi(lo, hi, x, co)) <= 1e-12
    ctx.close()


def test_fft_unsupported_shapes_fail_loudly():
    A = api()
    for N, n in [(37, 6), (64, 5)]:                       # not a power of two; odd order
        ctx = A.DGContext((N,), (n,), (0.0,), (2 * math.pi,), pmax=8, field_batch=2)
        ctx.set_option(A.OPT_FIELD_KERNEL, A.FIELD_FFT)
        rho = torch.ones((2, N * n), dtype=torch.float64, device="cuda")
        with pytest.raises(A.DGError):
            ctx.poisson_E(rho)
        ctx.close()


def test_fft_config5_grid_closed_form_and_sampled_oracle():
    """Config-5 grid (2048 x 8, modes <= 8192) through the FFT kernel: single cosines against the closed forms
    E = -(A/m) sin(mx + ph), Phi = -(A/m^2) cos(mx + ph), c_m = (A/2) e^{i ph}; seeded cosine sums against the
    oracle's dense contraction on a slice of modes and on a few vectors."""
    A = api()
    N, n, lo, hi, pmax = 2048, 8, 0.0, 2 * math.pi, 8192
    ctx = A.DGContext((N,), (n,), (lo,), (hi,), pmax=pmax, field_batch=4, workspace=False)
    ctx.set_option(A.OPT_FIELD_KERNEL, A.FIELD_FFT)
    x = ctx.nodes(0)
    ms, amp, ph = np.array([1, 16, 333, 700]), 0.05, 0.4
    rho = 1 + amp * np.cos(ms[:, None] * x[None, :] + ph)
    c = ctx.fourier_project(dev(rho)).cpu().numpy()
    for i, m in enumerate(ms):
        assert abs(c[i, m, 0] + 1j * c[i, m, 1] - 0.5 * amp * np.exp(1j * ph)) < 5e-13
        assert abs(c[i, 0, 0] - 1) < 1e-13
    ctx.close()
    # with the modes of a physical setting (pmax = N: PAPER.md:429) the closed forms hold to round-off
    ctx = A.DGContext((N,), (n,), (lo,), (hi,), pmax=N, field_batch=4, workspace=False)
    ctx.set_option(A.OPT_FIELD_KERNEL, A.FIELD_FFT)
    E = ctx.poisson_E(dev(rho)).cpu().numpy()
    Phi = ctx.poisson_phi(dev(rho)).cpu().numpy()
    for i, m in enumerate(ms):
        tol = 1e-11 if m <= 333 else 1e-9        # m = 700: 2.9 elements per wavelength, discretisation error of Eq. 63
        assert relerr(E[i], -(amp / m) * np.sin(m * x + ph)) < tol
        # conditioned bound as above: |Phi| = amp / m^2 against round-off eps |rho| / k_1^2
        assert np.max(np.abs(Phi[i] + (amp / m ** 2) * np.cos(m * x + ph))) < tol * amp / m ** 2 + 1e-14
    ctx.close()
    # seeded batch against the oracle on a mode slice (the full dense T of config 5 is 2 GB: the oracle builds 96 rows)
    ctx = A.DGContext((N,), (n,), (lo,), (hi,), pmax=pmax, field_batch=4, workspace=False)
    ctx.set_option(A.OPT_FIELD_KERNEL, A.FIELD_FFT)
    rho, _, _, _ = wl.cosine_sum_density(x, 6, wl.SEED_CFG5, mmax=1024)
    c = ctx.fourier_project(dev(rho)).cpu().numpy()
    cz = c[..., 0] + 1j * c[..., 1]
    To = ofr.transform_tensor(lo, hi, N, n, 95)
    assert relerr(cz[:, :96], ofr.fourier_project(To, rho)) <= 1e-12
    ctx.close()


@pytest.mark.parametrize("N,n,batch", [(10, 3, 1), (25, 8, 4), (64, 8, 40), (300, 5, 7), (2048, 8, 3)])
def test_field_energy_matches_oracle(N, n, batch):
    """dg_field_energy (Fig. 10; mass matrix of Eq. 50) against the oracle; the P_{n-1} closed form
    L / (2 (2n - 1)) that a lumped quadrature gets wrong; deterministic."""
    A = api()
    lo, hi = -0.5, 2.0
    ctx = A.DGContext((N,), (n,), (lo,), (hi,), pmax=4, workspace=False)
    E = wl.uniform_field((batch, N * n), 41) - 0.5
    W = ctx.field_energy(dev(E)).cpu().numpy()
    assert relerr(W, ofr.field_energy(lo, hi, N, n, E)) <= 1e-13
    assert np.array_equal(W, ctx.field_energy(dev(E)).cpu().numpy())
    xi = ctx.operators(0)[0]
    Pn1 = np.tile(np.polynomial.legendre.legval(xi, [0.0] * (n - 1) + [1.0]), N)
    assert abs(float(ctx.field_energy(dev(Pn1))[0]) - (hi - lo) / (2.0 * (2 * n - 1))) < 1e-13 * (hi - lo)
    ctx.close()


@pytest.mark.parametrize("N,n,batch", [(10, 3, 1), (25, 8, 4), (64, 8, 40), (300, 5, 7), (2048, 8, 3)])
def test_broken_l2_matches_oracle(N, n, batch):
    """dg_broken_l2 (Eq. 72 with the LGL mass matrix of Eq. 50) against the oracle, with and without v."""
    A = api()
    lo, hi = -0.5, 2.0
    ctx = A.DGContext((N,), (n,), (lo,), (hi,), pmax=4, workspace=False)
    u = wl.uniform_field((batch, N * n), 31) - 0.5
    v = wl.uniform_field((batch, N * n), 32) - 0.5
    e = ctx.broken_l2(dev(u), dev(v)).cpu().numpy()
    assert relerr(e, ofr.broken_l2(lo, hi, N, n, u, v)) <= 1e-13
    e0 = ctx.broken_l2(dev(u)).cpu().numpy()
    assert relerr(e0, ofr.broken_l2(lo, hi, N, n, u)) <= 1e-13
    assert np.array_equal(e, ctx.broken_l2(dev(u), dev(v)).cpu().numpy())
    ctx.close()


@pytest.mark.parametrize("n", [3, 4, 5, 6, 8])
def test_poisson_hp_convergence_fig4_on_gpu(n):
    """Fig. 4: Phi'' = sin(2 pi x) on [0, 1], N = 10, 15, 20, 25, pmax = N, through dg_poisson_phi and
    dg_broken_l2: every error equals the oracle's (same chain on the CPU), and for n <= 6 (above round-off) the
    h-convergence is at least the paper's O(dx^{n+1/2}).  dg_broken_l2 measures the NODAL error (interpolant of
    Phi - Phi_exact at the LGL nodes), which superconverges (n = 4: rate 6.5); the rate of the continuous error that
    Fig. 4 plots is pinned on the oracle in tests/test_oracle_fourier.py::test_poisson_convergence_fig4."""
    A = api()
    lo, hi = 0.0, 1.0
    errs, Ns = [], [10, 15, 20, 25]
    for N in Ns:
        ctx = A.DGContext((N,), (n,), (lo,), (hi,), pmax=N, workspace=True)
        x = ctx.nodes(0)
        src = np.sin(2 * np.pi * x)
        exact = -src / (4 * np.pi ** 2)
        Phi = ctx.poisson_phi(dev(src))
        eps = float(ctx.broken_l2(Phi, dev(exact)).cpu().numpy()[0])
        co = ofr.fourier_project(ofr.transform_tensor(lo, hi, N, n, N), src)
        eps_o = float(ofr.broken_l2(lo, hi, N, n, ofr.poisson_phi(lo, hi, ofr.node_coordinates(lo, hi, N, n), co), exact))
        assert abs(eps - eps_o) <= 1e-9 * eps_o + 1e-16, (N, eps, eps_o)
        errs.append(eps)
        ctx.close()
    if n <= 6:
        slope = np.polyfit(np.log(1.0 / np.array(Ns)), np.log(errs), 1)[0]
        assert slope > n - 0.2, (slope, errs)


@pytest.mark.parametrize("n,N,pmax,batch,kernel", [(8, 24, 30, 1, 0), (6, 37, 50, 40, 2), (5, 9, 12, 70, 3), (4, 64, 64, 5, 1)])
def test_nonuniform_element_widths_match_oracle(n, N, pmax, batch, kernel):
    """dg_create_field_nonuniform: Eq. 63 with per-element widths.  T, nodes, c_p, E, Phi and the broken l2 norm against the
    oracle on a graded grid (widths varying 4x); the FFT kernel must refuse (it needs equal widths)."""
    A = api()
    w = 1.0 + 0.6 * np.sin(np.arange(N) * 0.7)
    edges = -0.3 + np.concatenate([[0.0], np.cumsum(w)]) * (2 * math.pi / w.sum())
    ctx = A.DGContext.field_nonuniform(edges, n, pmax=pmax, field_batch=batch)
    x = ofr.node_coordinates_edges(edges, n)
    assert np.max(np.abs(ctx.nodes(0) - x)) < 1e-15 * 8
    To = ofr.transform_tensor_edges(edges, n, pmax)
    assert np.max(np.abs(ctx.transform() - To)) <= 5e-16 * N * n
    ctx.set_option(A.OPT_FIELD_KERNEL, kernel)
    rho, _, _, _ = wl.cosine_sum_density(x, batch, 77, mmax=max(1, pmax // 3))
    co = ofr.fourier_project(To, rho)
    c = ctx.fourier_project(dev(rho)).cpu().numpy()
    assert relerr(c[..., 0] + 1j * c[..., 1], co) <= 1e-12
    assert relerr(ctx.poisson_E(dev(rho)).cpu().numpy(), ofr.poisson_E(edges[0], edges[-1], x, co)) <= 1e-12
    Phio = ofr.poisson_phi(edges[0], edges[-1], x, co)
    assert np.max(np.abs(ctx.poisson_phi(dev(rho)).cpu().numpy() - Phio)) <= 1e-12 * np.max(np.abs(Phio)) + 1e-14 * np.max(np.abs(rho))
    u, v = wl.uniform_field((batch, N * n), 5), wl.uniform_field((batch, N * n), 6)
    assert relerr(ctx.broken_l2(dev(u), dev(v)).cpu().numpy(), ofr.broken_l2(0, 0, N, n, u, v, edges=edges)) <= 1e-13
    assert relerr(ctx.field_energy(dev(u)).cpu().numpy(), ofr.field_energy(0, 0, N, n, u, edges=edges)) <= 1e-13
    ctx.set_option(A.OPT_FIELD_KERNEL, A.FIELD_FFT)
    with pytest.raises(A.DGError):
        ctx.poisson_E(dev(rho))
    ctx.close()
