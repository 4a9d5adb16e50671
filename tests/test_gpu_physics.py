"""End-to-end physics on the GPU path: the cyclotron-harmonic instability of the paper's Section 6.1 on a scaled grid.

Simulation A: ring distribution j = 6 (Eq. 31), omega_p/omega_c = 10 (B_ext = 0.1), perturbed by the
eigenmode of Eq. 35-36 at (k, omega) = (0.886 / r_L, 0.349i omega_c), domain length 2 pi / k, velocity box +-8.5.  Linear
theory (Eq. 30 / 34) and Fig. 10a of the paper: the field energy grows as exp(2 * 0.349 omega_c t).  Here: (16, 32, 32)
elements x 8^3 nodes instead of (25, 50, 50) (a few seconds of GPU time), self-consistent SSP-RK3 through dg_ssprk3_run,
field energy from dg_density + dg_poisson_E."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import workloads as wl     # noqa: E402


def _run(k_larmor, omega, t_end, t_diag, nelem, amp=2e-4, sense=-1):
    from paper_2202_13532_b200 import api
    wc, j, n = 0.1, 6, 8
    k_sim = k_larmor * wc                      # 1/r_L -> 1/lambda_D: r_L = (omega_p/omega_c) lambda_D
    L = 2 * math.pi / k_sim
    ctx = api.DGContext(nelem, (n, n, n), (0.0, -8.5, -8.5), (L, 8.5, 8.5), bc=(0, 1, 1), omega_c=wc, pmax=nelem[0])
    x, u, v = ctx.nodes(0), ctx.nodes(1), ctx.nodes(2)
    f1 = wl.eigenmode_perturbation(x, u, v, k_sim, k_larmor, omega, j, sense=sense)
    rho1 = ctx.density(torch.from_numpy(f1).cuda()).cpu().numpy()
    f = torch.from_numpy(wl.ring_distribution(u, v, j)[None] + (amp / np.max(np.abs(rho1))) * f1).cuda()
    wx = np.tile(ctx.operators(0)[1] * 0.5 * L / nelem[0], nelem[0])          # LGL quadrature weights in x

    def energy():
        return float(ctx.field_energy(ctx.poisson_E(ctx.density(f)))[0])      # dg_field_energy: Fig. 10's diagnostic on the device

    mass0 = float(np.sum(wx * ctx.density(f).cpu().numpy()))
    steps = max(1, math.ceil(t_diag / (0.9 * ctx.max_stable_dt(0.3))))
    dt = t_diag / steps
    ts, W = [0.0], [energy()]
    while ts[-1] < t_end - 1e-9:
        ctx.ssprk3_run(f, dt, steps, True)
        ts.append(ts[-1] + t_diag); W.append(energy())
    mass1 = float(np.sum(wx * ctx.density(f).cpu().numpy()))
    assert bool(torch.isfinite(f).all())
    ctx.close()
    return np.array(ts), np.array(W), (mass1 - mass0) / mass0, wc


def test_simulation_A_growth_rate():
    """Purely growing mode: energy growth rate 2 * 0.349 omega_c (Fig. 10a) from t = 0, within 2 %."""
    ts, W, dmass, wc = _run(0.886, 0.349j, 60.0, 2.0, (16, 32, 32))
    m = ts >= 10.0
    gamma = np.polyfit(ts[m], np.log(W[m]), 1)[0] / 2.0 / wc
    assert abs(gamma / 0.349 - 1.0) < 0.02, gamma
    assert np.all(np.diff(W) > 0)                                # a clean eigenmode: monotone from the first sample
    resid = np.log(W[m]) - np.polyval(np.polyfit(ts[m], np.log(W[m]), 1), ts[m])
    assert np.max(np.abs(resid)) < 0.02                          # exponential to 2 % over 3.5 e-foldings of the energy
    assert abs(dmass) < 1e-8                                     # zero-inflow velocity boundaries at 8.5 v_th


def test_eq36_as_printed_is_the_other_handedness():
    """DESIGN.md reading C24: Eq. 36 literally (sense = +1) is the eigenmode of the opposite gyration; under Eq. 28 it is a
    mixture of stable cyclotron harmonics and the energy does not grow over the first cyclotron period."""
    ts, W, _, _ = _run(0.886, 0.349j, 40.0, 4.0, (16, 32, 32), sense=+1)
    assert W[-1] < 2.0 * W[0]                                    # the true eigenmode gains a factor 16 by t = 40


def test_simulation_B_growth_rate_and_frequency():
    """Mode with a real frequency: (k, omega) = (1.4, 1.182 + 0.131i); field energy ~ exp(2 * 0.131 omega_c t)
    (Fig. 10b).  The energy of a travelling eigenmode grows without oscillating; tolerance 5 % (three-digit root, and
    the slower mode is contaminated longer by the stable harmonics the truncated series leaves behind)."""
    ts, W, dmass, wc = _run(1.4, 1.182 + 0.131j, 150.0, 5.0, (16, 32, 32))
    m = ts >= 30.0
    gamma = np.polyfit(ts[m], np.log(W[m]), 1)[0] / 2.0 / wc
    assert abs(gamma / 0.131 - 1.0) < 0.05, gamma
    assert abs(dmass) < 1e-8


def test_landau_damping_rate_config1():
    """Config 1 (1D1V, 16 x 32 elements, n = 4, generic kernel) run to t = 20 through dg_ssprk3_run: the k = 0.5 field mode
    decays at the textbook Landau rate -0.1533 with omega_r = 1.4156 (the closed-form pin of the oracle; a
    wrong sign of E or of the v-speed grows instead), and E(0) = -0.02 sin(0.5 x) to the n = 4 discretisation error."""
    from paper_2202_13532_b200 import api
    ctx = api.DGContext((16, 32), (4, 4), (0.0, -6.0), (4 * math.pi, 6.0), bc=(0, 1), pmax=16)
    x, v = ctx.nodes(0), ctx.nodes(1)
    f = torch.from_numpy(wl.landau_f0(x, v)).cuda()
    E0 = ctx.poisson_E(ctx.density(f)).cpu().numpy()
    assert np.max(np.abs(E0 + 0.02 * np.sin(0.5 * x))) < 1e-6
    dt, per, nsamp = 0.01, 5, 400
    amp = []
    for _ in range(nsamp):
        ctx.ssprk3_run(f, dt, per, True)
        amp.append(float(ctx.poisson_E(ctx.density(f)).abs().max()))
    amp = np.array(amp); t = dt * per * (np.arange(nsamp) + 1)
    pk = [i for i in range(1, nsamp - 1) if amp[i] > amp[i - 1] and amp[i] > amp[i + 1]]
    assert len(pk) >= 6
    rate = np.polyfit(t[pk], np.log(amp[pk]), 1)[0]
    assert -0.165 < rate < -0.143, rate
    assert abs(np.mean(np.diff(t[pk])) - math.pi / 1.4156) < 0.08
    assert ctx.last_kernel == "rhs_generic"
    ctx.close()
