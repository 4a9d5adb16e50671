"""SSP-RK3 steps of BASELINE.json's configs 2 and 3 against the oracle on the WHOLE array (north_star:
<= 1e-12 per evaluation, <= 1e-10 after 100 RK steps):

  * config 3 on its own 512^3 grid (ring + seeded noise, dt 5e-4, Poisson at every stage): 3 steps, compared after each;
  * config 3's recipe on the 16^3-element (128^3 DOF) replica for all 1000 steps, compared at steps 100 and 1000;
  * config 2 on its own 256^3 grid, dt 1e-3 (reading C22), 100 steps, compared at steps 10 and 100.

The oracle needs ~6 min for the 1000-step and ~5 min for the 100-step trajectory on the GPU box's host cores; both run in
worker processes (tests/_oracle_traj_worker.py: oracle + workloads only) started when this module's first test begins, so they
overlap each other and the 512^3 test.  The error bound for K steps is derived in DESIGN.md section 6 (linear accumulation of the
per-step rounding difference, 1000 x ~2e-15)."""
import math
import os
import subprocess
import sys
import time

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import vlasov as ov          # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, os.path.join(ROOT, "tests"))
from _oracle_traj_worker import make_grid, initial_state      # noqa: E402  (the workers' own grid and input recipe)

K = 0.1
LO, HI = (0.0, -8.5, -8.5), (2 * math.pi / K, 8.5, 8.5)

# name: (elements per dim, order, dt, noise amplitude, steps, checkpoints)
TRAJ = {
    "config3_replica_128": ((16, 16, 16), 8, 5e-4, 1e-4, 1000, (100, 1000)),
    "config2_256": ((32, 32, 32), 8, 1e-3, 0.0, 100, (10, 100)),
}


def api():
    from paper_2202_13532_b200 import api as _api
    return _api


def relerr(a, b):
    return float(np.max(np.abs(np.asarray(a) - np.asarray(b))) / max(np.max(np.abs(b)), 1e-300))


@pytest.fixture(scope="module")
def oracle_workers(tmp_path_factory):
    out = str(tmp_path_factory.mktemp("oracle_traj"))
    ncpu = os.cpu_count() or 1
    env = dict(os.environ)
    for v in ("OMP_NUM_THREADS", "OPENBLAS_NUM_THREADS", "MKL_NUM_THREADS"):
        env[v] = str(max(1, ncpu // 3))
    procs = {}
    for name, (nelem, order, dt, noise, steps, cps) in TRAJ.items():
        cmd = [sys.executable, os.path.join(ROOT, "tests", "_oracle_traj_worker.py"), out, name] + [str(n) for n in nelem] + \
              [str(order), repr(dt), repr(noise), str(steps), ",".join(str(c) for c in cps)]
        procs[name] = subprocess.Popen(cmd, env=env, cwd=ROOT, stdout=subprocess.DEVNULL, stderr=subprocess.PIPE, text=True)
    yield out, procs
    for p in procs.values():
        if p.poll() is None:
            p.kill()


def wait_checkpoint(workers, name, step, timeout=2400.0):
    out, procs = workers
    path = os.path.join(out, f"{name}_{step}.npy")
    t0 = time.time()
    while not os.path.exists(path):
        rc = procs[name].poll()
        if rc is not None and rc != 0:
            raise RuntimeError(f"oracle worker {name} failed ({rc}): {procs[name].stderr.read()[-2000:]}")
        if time.time() - t0 > timeout:
            raise TimeoutError(f"oracle worker {name} did not reach step {step} within {timeout} s")
        time.sleep(0.5)
    return np.load(path)


def same_state(ctx, nelem, order, noise):
    """The state the worker starts from (seeded recipe on the oracle's node coordinates, which the library's match to an ulp):
    both sides get the identical array."""
    g = make_grid(nelem, order)
    for d in range(3):
        assert relerr(ctx.nodes(d), g.coords[d].reshape(-1)) < 1e-15
    return g, initial_state(g, noise)


def test_config3_512_three_steps_whole_array(oracle_workers):
    """Config 3 on its own grid: three self-consistent SSP-RK3 steps (dg_ssprk3_run, tiled kernel, the launch configuration
    bench.py times), every node compared with oracle.vlasov.ssprk3_step after each step."""
    nelem, order = (64, 64, 64), (8, 8, 8)
    ctx = api().DGContext(nelem, order, LO, HI, bc=(0, 1, 1), omega_c=1.0, pmax=64)
    g, f0 = same_state(ctx, nelem, 8, 1e-4)
    fd = torch.from_numpy(f0).cuda()
    # two steps in one call (stage k+1 takes its density from stage k's epilogue partials across the step boundary), then one
    fo = f0
    fo = ov.ssprk3_step(g, fo, 5e-4)
    ctx.ssprk3_run(fd, 5e-4, 1, True)
    assert ctx.last_kernel.startswith("rhs_tiled<8,")
    e1 = relerr(fd.cpu().numpy(), fo)
    assert e1 <= 1e-12, e1
    fo = ov.ssprk3_step(g, fo, 5e-4)
    fo = ov.ssprk3_step(g, fo, 5e-4)
    ctx.ssprk3_run(fd, 5e-4, 2, True)
    e3 = relerr(fd.cpu().numpy(), fo)
    assert e3 <= 1e-12, e3
    # and the three steps in ONE call from the initial state, bit-identical to 1 + 2 (same kernels, same order)
    fd2 = torch.from_numpy(f0).cuda()
    ctx.ssprk3_run(fd2, 5e-4, 3, True)
    assert relerr(fd2.cpu().numpy(), fo) <= 1e-12
    ctx.close()


def test_config3_replica_1000_steps(oracle_workers):
    """Config 3's recipe (ring + SEED_CFG3_NOISE, dt 5e-4, Poisson at every stage) on the 128^3 replica, all 1000 steps."""
    nelem, order, dt, noise, steps, cps = TRAJ["config3_replica_128"]
    ctx = api().DGContext(nelem, (order,) * 3, LO, HI, bc=(0, 1, 1), omega_c=1.0, pmax=nelem[0])
    assert dt < ctx.max_stable_dt(0.2)
    fd = torch.from_numpy(same_state(ctx, nelem, order, noise)[1]).cuda()
    done = 0
    for cp in cps:
        ctx.ssprk3_run(fd, dt, cp - done, True)
        done = cp
        fo = wait_checkpoint(oracle_workers, "config3_replica_128", cp)
        assert np.isfinite(fo).all()
        err = relerr(fd.cpu().numpy(), fo)
        assert err <= 1e-10, (cp, err)
    assert ctx.last_kernel.startswith("rhs_tiled<8,")
    ctx.close()


def test_config2_256_100_steps(oracle_workers):
    """Config 2 on its own 256^3 grid, dt = 1e-3 (the literal 5e-3 violates the RK3 limit, reading C22), 100 steps."""
    nelem, order, dt, noise, steps, cps = TRAJ["config2_256"]
    ctx = api().DGContext(nelem, (order,) * 3, LO, HI, bc=(0, 1, 1), omega_c=1.0, pmax=nelem[0])
    assert dt < ctx.max_stable_dt(0.2)
    fd = torch.from_numpy(same_state(ctx, nelem, order, noise)[1]).cuda()
    done = 0
    for cp in cps:
        ctx.ssprk3_run(fd, dt, cp - done, True)
        done = cp
        fo = wait_checkpoint(oracle_workers, "config2_256", cp)
        assert np.isfinite(fo).all()
        err = relerr(fd.cpu().numpy(), fo)
        assert err <= 1e-10, (cp, err)
    ctx.close()
