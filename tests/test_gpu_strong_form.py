"""GPU parity of the strong-form variant (DG_OPT_FORM = 1, Eq. 15) against the oracle's rhs_strong, on
both RHS kernels, and of D (Eq. 55) against the oracle and against exactness on polynomials."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import vlasov as ov, basis as ob      # noqa: E402
import workloads as wl                             # noqa: E402


def api():
    from paper_2202_13532_b200 import api as _api
    return _api


def relerr(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("n", [2, 3, 4, 5, 6, 7, 8, 9, 10])
def test_dmatrix_matches_oracle_and_is_exact_on_polynomials(n):
    A = api()
    ctx = A.DGContext((2, 2), (n, n), (0.0, -1.0), (1.0, 1.0), workspace=False)
    D = ctx.dmatrix(0)
    assert np.max(np.abs(D - ob.lagrange_derivative_matrix(n))) <= 2e-13 * np.max(np.abs(D))
    xi = ctx.operators(0)[0]
    for m in range(n):                                   # d/dxi xi^m = m xi^(m-1), degree <= n-1 (north_star)
        exact = m * xi ** (m - 1) if m > 0 else np.zeros(n)
        assert np.max(np.abs(D @ xi ** m - exact)) < 1e-12 * max(1.0, n * n)
    ctx.close()


# (nelem, order, lo, hi, bc, omega_c, mass_mode, kernel)
K = 0.1
BOX3 = ((0.0, -8.5, -8.5), (2 * math.pi / K, 8.5, 8.5))
CASES = [
    ((16, 32), (4, 4), (0.0, -6.0), (4 * math.pi, 6.0), (0, 1), 0.0, 0, "auto"),          # 1D1V: generic kernel
    ((5, 6), (7, 3), (0.0, -5.0), (3.0, 5.0), (0, 0), 0.0, 1, "auto"),                    # mixed orders, lumped
    ((3, 5, 9), (8, 8, 8), BOX3[0], BOX3[1], (0, 1, 1), 1.0, 0, "auto"),                  # tiled <8,4>, ragged v tile
    ((3, 5, 9), (8, 8, 8), BOX3[0], BOX3[1], (0, 1, 1), 1.0, 0, "generic"),
    ((4, 3, 17), (4, 4, 4), BOX3[0], BOX3[1], (0, 0, 0), 0.7, 0, "auto"),                 # tiled <4,8>, all periodic
    ((3, 4, 5), (6, 6, 6), BOX3[0], BOX3[1], (0, 1, 1), 1.0, 1, "auto"),                  # tiled <6,8>, lumped mass
    ((2, 3, 4), (10, 10, 10), BOX3[0], BOX3[1], (0, 1, 0), -0.5, 0, "auto"),              # tiled <10,3>
]


@pytest.mark.parametrize("case", CASES)
def test_strong_form_rhs_and_stage_match_oracle(case):
    nelem, order, lo, hi, bc, omega_c, mode, kernel = case
    A = api()
    g = ov.Grid(nelem=nelem, order=order, lo=lo, hi=hi, bc=bc, omega_c=omega_c, mass_mode=mode)
    ctx = A.DGContext(nelem, order, lo, hi, bc=bc, omega_c=omega_c, mass_mode=mode)
    ctx.set_option(A.OPT_RHS_KERNEL, A.KERNEL_GENERIC if kernel == "generic" else A.KERNEL_AUTO)
    f = wl.uniform_field(g.flat_shape, 41) - 0.3
    E = wl.normal_E(g.flat_shape[0], 42)
    weak = ctx.rhs(dev(f), dev(E)).cpu().numpy()
    ctx.set_option(A.OPT_FORM, A.FORM_STRONG)
    strong = ctx.rhs(dev(f), dev(E)).cpu().numpy()
    so = ov.rhs_strong(g, f, E)
    assert relerr(strong, so) <= 1e-12
    assert relerr(strong, weak) <= 1e-11 and not np.array_equal(strong, weak)     # same scheme, different rounding
    assert relerr(ctx.rhs(dev(f), None).cpu().numpy(), ov.rhs_strong(g, f, None)) <= 1e-12
    if len(nelem) == 3:
        fn = wl.uniform_field(g.flat_shape, 43)
        out = torch.empty_like(dev(f))
        ctx.rk_stage(dev(f), dev(fn), dev(E), out, 0.75, 0.25, 1e-3)
        assert relerr(out.cpu().numpy(), 0.75 * fn + 0.25 * (f + 1e-3 * so)) <= 1e-13
    ctx.close()


@pytest.mark.parametrize("kernel", ["generic", "auto"])
def test_strong_form_steps_match_oracle(kernel):
    """Config-2 physics on a small replica, 3 self-consistent SSP-RK3 steps in the strong form."""
    A = api()
    nelem, order = (4, 4, 8), (8, 8, 8)
    g = ov.Grid(nelem=nelem, order=order, lo=BOX3[0], hi=BOX3[1], bc=(0, 1, 1), omega_c=1.0, pmax=4)
    ctx = A.DGContext(nelem, order, BOX3[0], BOX3[1], bc=(0, 1, 1), omega_c=1.0, pmax=4)
    ctx.set_option(A.OPT_RHS_KERNEL, A.KERNEL_GENERIC if kernel == "generic" else A.KERNEL_AUTO)
    ctx.set_option(A.OPT_FORM, A.FORM_STRONG)
    f0 = wl.add_uniform_noise(wl.ring_f0(ctx.nodes(0), ctx.nodes(1), ctx.nodes(2), K), 9, 1e-4)
    fo = f0.copy()
    for _ in range(3):
        fo = ov.ssprk3_step(g, fo, 5e-4, strong=True)
    fd = dev(f0)
    ctx.ssprk3_run(fd, 5e-4, 3, True)
    assert relerr(fd.cpu().numpy(), fo) <= 1e-12
    ctx.close()
