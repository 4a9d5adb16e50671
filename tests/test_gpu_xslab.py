"""GPU parity of the x-slab (DG_BC_HALO) path: dg_set_xhalo / dg_rk_stage and the sharded stepper on ONE GPU.
Two slabs are advanced one after the other by the same process (plain stream order: no kernel waits on another),
with the face planes exchanged by device copies; the reference is the UNSHARDED oracle on the global grid."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import vlasov as ov      # noqa: E402
import workloads as wl               # noqa: E402


def api():
    from paper_2202_13532_b200 import api as _api
    return _api


def relerr(a, b):
    return float(np.max(np.abs(np.asarray(a) - np.asarray(b))) / max(np.max(np.abs(b)), 1e-300))


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


CASES = [
    # nelem, order, lo, hi, bc, omega_c, split (x-elements of slab 0), kernel
    ((4, 4, 8), (8, 8, 8), (0.0, -8.5, -8.5), (20 * math.pi, 8.5, 8.5), (0, 1, 1), 1.0, 1, "auto"),      # tiled <8,4>
    ((4, 4, 8), (8, 8, 8), (0.0, -8.5, -8.5), (20 * math.pi, 8.5, 8.5), (0, 1, 1), 1.0, 2, "generic"),
    ((5, 6, 6), (4, 4, 4), (0.0, -4.0, -4.0), (6.0, 4.0, 4.0), (0, 1, 1), 1.0, 2, "auto"),               # tiled <4,8>
    ((3, 3, 4), (10, 10, 10), (0.0, -4.0, -4.0), (6.0, 4.0, 4.0), (1, 1, 0), 0.7, 1, "auto"),            # zero inflow in x
    ((6, 9), (4, 5), (0.0, -5.0), (4 * math.pi, 5.0), (0, 1), 0.0, 4, "auto"),                           # 1D1V, generic
]


def _slab_ctx(nelem, order, lo, hi, bc, omega_c, e0, e1, kernel):
    A = api()
    dx = (hi[0] - lo[0]) / nelem[0]
    ctx = A.DGContext((e1 - e0,) + tuple(nelem[1:]), order, (lo[0] + e0 * dx,) + tuple(lo[1:]), (lo[0] + e1 * dx,) + tuple(hi[1:]),
                      bc=(A.BC_HALO,) + tuple(bc[1:]), omega_c=omega_c, pmax=1)
    ctx.set_option(A.OPT_RHS_KERNEL, A.KERNEL_GENERIC if kernel == "generic" else A.KERNEL_AUTO)
    return ctx


@pytest.mark.parametrize("case", CASES)
def test_two_slabs_rhs_and_stage_match_unsharded_oracle(case):
    nelem, order, lo, hi, bc, omega_c, split, kernel = case
    g = ov.Grid(nelem=nelem, order=order, lo=lo, hi=hi, bc=bc, omega_c=omega_c)
    n = order[0]
    f = wl.uniform_field(g.flat_shape, 21) - 0.3
    fn = wl.uniform_field(g.flat_shape, 22)
    E = wl.normal_E(g.flat_shape[0], 23)
    ro = ov.rhs(g, f, E)
    parts = [(0, split), (split, nelem[0])]
    periodic = bc[0] == 0
    for r, (e0, e1) in enumerate(parts):
        ctx = _slab_ctx(nelem, order, lo, hi, bc, omega_c, e0, e1, kernel)
        fs, fns, Es = dev(f[e0 * n:e1 * n]), dev(fn[e0 * n:e1 * n]), dev(E[e0 * n:e1 * n])
        halo = torch.zeros((2,) + fs.shape[1:], dtype=torch.float64, device="cuda")
        with pytest.raises(api().DGError):
            ctx.rhs(fs, Es)                                   # no halo set yet: must fail loudly
        left_plane = f[e0 * n - 1] if e0 > 0 else (f[-1] if periodic else None)
        right_plane = f[e1 * n] if e1 < nelem[0] else (f[0] if periodic else None)
        if left_plane is not None:
            halo[0].copy_(dev(left_plane))
        if right_plane is not None:
            halo[1].copy_(dev(right_plane))
        ctx.set_xhalo(halo)
        out = ctx.rhs(fs, Es).cpu().numpy()
        assert float(np.max(np.abs(out - ro[e0 * n:e1 * n])) / np.max(np.abs(ro))) <= 1e-12
        o2 = torch.empty_like(fs)
        ctx.rk_stage(fs, fns, Es, o2, 0.75, 0.25, 1e-3)
        ref = 0.75 * fn[e0 * n:e1 * n] + 0.25 * (f[e0 * n:e1 * n] + 1e-3 * ro[e0 * n:e1 * n])
        assert relerr(o2.cpu().numpy(), ref) <= 1e-13
        rho_out = torch.empty(fs.shape[0], dtype=torch.float64, device="cuda")
        o3 = torch.empty_like(fs)
        ctx.rk_stage(fs, fns, Es, o3, 0.75, 0.25, 1e-3, rho_out)   # density of `out` from the epilogue partials (S10)
        assert torch.equal(o3, o2)
        gs = ov.Grid(nelem=(e1 - e0,) + tuple(nelem[1:]), order=order, lo=lo, hi=hi, bc=bc, omega_c=omega_c)
        assert relerr(rho_out.cpu().numpy(), ov.density(gs, ref)) <= 1e-13
        ctx.rk_stage(fs, None, None, o2, 0.0, 1.0, 1e-3)      # E = 0, no f_n
        ref0 = f[e0 * n:e1 * n] + 1e-3 * ov.rhs(g, f, None)[e0 * n:e1 * n]
        assert relerr(o2.cpu().numpy(), ref0) <= 1e-13
        with pytest.raises(api().DGError):
            ctx.rk_stage(fs, None, None, o2, 0.5, 0.5, 1e-3)  # c0 != 0 needs f_n
        ctx.close()


@pytest.mark.parametrize("kernel_n", [8, 4])
@pytest.mark.parametrize("push", [False, True])
def test_sharded_stepper_world1_matches_oracle(kernel_n, push):
    """XSlabStepper with the CUDA backend, world = 1: the periodic wrap goes through the halo planes and the Poisson
    solve through the x-only global context; 3 self-consistent steps against the oracle."""
    from paper_2202_13532_b200 import sharded
    k = 0.1
    n = kernel_n
    nelem, order = (4, 4, 8) if n == 8 else (6, 6, 8), (n, n, n)
    lo, hi = (0.0, -8.5, -8.5), (2 * math.pi / k, 8.5, 8.5)
    g = ov.Grid(nelem=nelem, order=order, lo=lo, hi=hi, bc=(0, 1, 1), omega_c=1.0, pmax=4)
    f0 = wl.add_uniform_noise(wl.ring_f0(g.coords[0].reshape(-1), g.coords[1].reshape(-1), g.coords[2].reshape(-1), k), 5, 1e-4)
    st = sharded.XSlabStepper(nelem, order, lo, hi, bc=(0, 1, 1), omega_c=1.0, pmax=4, rank=0, world=1, device=0, push=push)
    f = dev(f0)
    st.run(f, 5e-4, 3, True)
    fo = f0.copy()
    for _ in range(3):
        fo = ov.ssprk3_step(g, fo, 5e-4)
    assert relerr(f.cpu().numpy(), fo) <= 1e-12
    # without the field solve (no all-gather between the stages), and single steps (halos primed by a plain exchange)
    f = dev(f0)
    st.run(f, 5e-4, 2, False)
    st.step(f, 5e-4, False)
    fo = f0.copy()
    for _ in range(3):
        fo = ov.ssprk3_step(g, fo, 5e-4, self_consistent=False)
    assert relerr(f.cpu().numpy(), fo) <= 1e-12
    st.close()


@pytest.mark.parametrize("case", [((3, 5, 9), (8, 8, 8), "auto"), ((3, 5, 9), (8, 8, 8), "generic"), ((2, 3, 17), (4, 4, 4), "auto"),
                                  ((2, 3, 5), (6, 6, 6), "auto"), ((2, 2, 3), (10, 10, 10), "auto")])
def test_rk_stage_pushes_boundary_planes(case):
    """dg_set_xhalo_push: the first / last x plane of `out` lands in the given planes bit for bit (swizzled and row-major
    tiles, ragged last v tile, generic kernel), `out` itself is unchanged, and NULL disables a side."""
    nelem, order, kernel = case
    A = api()
    lo, hi = (0.0, -8.5, -8.5), (2 * math.pi / 0.1, 8.5, 8.5)
    ctx = A.DGContext(nelem, order, lo, hi, bc=(A.BC_HALO, 1, 1), omega_c=1.0, pmax=1)
    ctx.set_option(A.OPT_RHS_KERNEL, A.KERNEL_GENERIC if kernel == "generic" else A.KERNEL_AUTO)
    shape = ctx.flat_shape
    fs, fn = dev(wl.uniform_field(shape, 51) - 0.3), dev(wl.uniform_field(shape, 52))
    E = dev(wl.normal_E(shape[0], 53))
    halo = dev(wl.uniform_field((2,) + shape[1:], 54))
    ctx.set_xhalo(halo)
    ref = torch.empty_like(fs)
    ctx.rk_stage(fs, fn, E, ref, 0.75, 0.25, 1e-3)
    dst = torch.full((2, 2) + shape[1:], 7.0, dtype=torch.float64, device="cuda")
    ctx.set_xhalo_push(dst[1][1], dst[0][0])
    out = torch.empty_like(fs)
    ctx.rk_stage(fs, fn, E, out, 0.75, 0.25, 1e-3)
    assert torch.equal(out, ref)
    assert torch.equal(dst[1][1], ref[0]) and torch.equal(dst[0][0], ref[-1])
    assert bool((dst[0][1] == 7.0).all()) and bool((dst[1][0] == 7.0).all())
    dst.fill_(7.0)
    ctx.set_xhalo_push(None, dst[0][0])
    ctx.rk_stage(fs, fn, E, out, 0.75, 0.25, 1e-3)
    assert torch.equal(dst[0][0], ref[-1]) and bool((dst[1] == 7.0).all())
    dst.fill_(7.0)
    ctx.rhs(fs, E, out)                                   # the plain RHS never pushes
    assert bool((dst == 7.0).all())
    ctx.close()


@pytest.mark.parametrize("push", [False, True])
def test_two_slab_emulation_steps_match_unsharded_oracle(push):
    """Two slabs of unequal size stepped on one GPU, exchange by device copies (or, push = True, by the RHS kernels storing
    their boundary planes into the other slab's ping-pong halo buffers), rho gathered by concatenation: the data path
    of a 2-rank run, kernel for kernel, against 2 unsharded oracle steps."""
    from paper_2202_13532_b200 import sharded
    A = api()
    k = 0.1
    nelem, order = (5, 4, 8), (8, 8, 8)
    lo, hi = (0.0, -8.5, -8.5), (2 * math.pi / k, 8.5, 8.5)
    g = ov.Grid(nelem=nelem, order=order, lo=lo, hi=hi, bc=(0, 1, 1), omega_c=1.0, pmax=5)
    f0 = wl.add_uniform_noise(wl.ring_f0(g.coords[0].reshape(-1), g.coords[1].reshape(-1), g.coords[2].reshape(-1), k), 6, 1e-4)
    parts = sharded.slab_partition(nelem[0], 2)
    assert parts == [(0, 2), (2, 5)]
    n = 8
    bes = [sharded.CudaBackend(nelem, order, lo, hi, (0, 1, 1), 1.0, 5, 0, e0, e1, 0) for e0, e1 in parts]
    fs = [dev(f0[e0 * n:e1 * n]) for e0, e1 in parts]
    u1 = [torch.empty_like(x) for x in fs]
    u2 = [torch.empty_like(x) for x in fs]
    halos = [torch.zeros((2,) + x.shape[1:], dtype=torch.float64, device="cuda") for x in fs]
    H = [torch.zeros((2, 2) + x.shape[1:], dtype=torch.float64, device="cuda") for x in fs]      # [parity][side] per slab
    for be, h in zip(bes, halos):
        be.set_halo(h)
    sidx = [0]
    rho, E = torch.empty(g.flat_shape[0], dtype=torch.float64, device="cuda"), torch.empty(g.flat_shape[0], dtype=torch.float64, device="cuda")

    def stage(src, fn, dst, c0, c1, dt):
        for r, (e0, e1) in enumerate(parts):
            bes[r].density(src[r], rho[e0 * n:e1 * n])
        bes[0].poisson_E(rho, E)
        if push:
            cur, nxt = sidx[0] % 2, (sidx[0] + 1) % 2
            if sidx[0] == 0:                               # prime the first parity by a plain exchange
                for r in range(2):
                    H[r][0][0].copy_(src[(r - 1) % 2][-1]); H[r][0][1].copy_(src[(r + 1) % 2][0])
            for r in range(2):
                bes[r].set_halo(H[r][cur])
                bes[r].set_push(H[(r - 1) % 2][nxt][1], H[(r + 1) % 2][nxt][0])
            sidx[0] += 1
        else:
            for r in range(2):
                halos[r][0].copy_(src[(r - 1) % 2][-1]); halos[r][1].copy_(src[(r + 1) % 2][0])
        for r, (e0, e1) in enumerate(parts):
            bes[r].rk_stage(src[r], fn[r] if c0 else None, E[e0 * n:e1 * n].contiguous(), dst[r], c0, c1, dt)

    dt = 5e-4
    for _ in range(2):
        stage(fs, fs, u1, 0.0, 1.0, dt)
        stage(u1, fs, u2, 0.75, 0.25, dt)
        stage(u2, fs, fs, 1.0 / 3.0, 2.0 / 3.0, dt)
    fo = f0.copy()
    for _ in range(2):
        fo = ov.ssprk3_step(g, fo, dt)
    got = torch.cat(fs, 0).cpu().numpy()
    assert relerr(got, fo) <= 1e-12
    for be in bes:
        be.close()


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two GPUs: the x-slab exchange over NCCL / peer memory has only been run on one device (DESIGN.md section 9)")
@pytest.mark.parametrize("mode", ["sendrecv", "push"])
def test_two_gpu_xslab_matches_unsharded_oracle(mode):
    """World-size-2 run of the sharded step (one rank per GPU, torchrun): plain NCCL send/recv of the face planes, and
    the fused push of the faces into the neighbours' symmetric-memory halo buffers; against the unsharded oracle."""
    import json
    import os
    import socket
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(root, "tests", "_xslab_gpu_worker.py"), mode]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=root)
    assert res.returncode == 0, res.stderr[-3000:]
    out = json.loads([l for l in res.stdout.splitlines() if l.startswith("{")][-1])
    assert out["world"] == 2
    for k, v in out.items():
        if k.startswith("err_"):
            assert v <= 1e-11, (k, v)


def test_two_processes_one_gpu_xslab_host_staged():
    """Two RANKS AS TWO PROCESSES sharing cuda:0 (torchrun, gloo, sharded.HostStagedComm: faces and densities travel through
    host memory), uneven slabs (2 + 3 x-elements), XSlabStepper + CudaBackend: three self-consistent steps with the global
    Poisson solve and three without (periodic and zero-inflow x), against the UNSHARDED oracle.  The cross-process ordering
    of the sharded step through the library's kernels on the one GPU there is; the NCCL / peer-memory transports stay
    unmeasured across devices."""
    import json
    import os
    import socket
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(root, "tests", "_xslab_gpu_worker.py"), "hoststaged"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=root)
    assert res.returncode == 0, res.stderr[-3000:]
    out = json.loads([l for l in res.stdout.splitlines() if l.startswith("{")][-1])
    assert out["world"] == 2 and out["staged"] and len(set(out["pids"])) == 2
    assert out["slab_sc1_bc0"] == [0, 2]                       # rank 0 of the uneven 2 + 3 split
    errs = {k: v for k, v in out.items() if k.startswith("err_")}
    assert set(errs) == {"err_sc1_bc0", "err_sc0_bc0", "err_sc0_bc1"}
    for k, v in errs.items():
        assert v <= 1e-11, (k, v)
