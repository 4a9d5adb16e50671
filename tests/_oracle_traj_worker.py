"""Worker process of tests/test_gpu_config_steps.py: advances the ORACLE (oracle.vlasov.ssprk3_step, nothing else) over a
config's time steps and saves the state at the requested checkpoints as .npy files.  Runs beside the GPU tests so that the
long oracle trajectories (1000 steps at 128^3, 100 steps at 256^3) overlap each other and the other GPU tests.

    python tests/_oracle_traj_worker.py <outdir> <name> <Nx> <Nu> <Nv> <order> <dt> <noise> <steps> <checkpoint,...>

The state comes from workloads.py (the seeded input recipe) on the oracle's own node coordinates.  Imports no product code."""
import math
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import numpy as np                       # noqa: E402

from oracle import vlasov as ov          # noqa: E402
import workloads as wl                   # noqa: E402

K = 0.1


def make_grid(nelem, order):
    return ov.Grid(nelem=tuple(nelem), order=(order,) * 3, lo=(0.0, -8.5, -8.5), hi=(2 * math.pi / K, 8.5, 8.5), bc=(0, 1, 1),
                   omega_c=1.0, pmax=nelem[0])


def initial_state(g, noise):
    f0 = wl.ring_f0(g.coords[0].reshape(-1), g.coords[1].reshape(-1), g.coords[2].reshape(-1), K)
    if noise:
        f0 = wl.add_uniform_noise(f0, wl.SEED_CFG3_NOISE, noise)
    return np.ascontiguousarray(f0)


def main():
    outdir, name = sys.argv[1], sys.argv[2]
    nelem = [int(a) for a in sys.argv[3:6]]
    order, dt, noise, steps = int(sys.argv[6]), float(sys.argv[7]), float(sys.argv[8]), int(sys.argv[9])
    checkpoints = sorted(int(c) for c in sys.argv[10].split(","))
    g = make_grid(nelem, order)
    f = initial_state(g, noise)
    for s in range(1, steps + 1):
        f = ov.ssprk3_step(g, f, dt)
        if s in checkpoints:
            tmp = os.path.join(outdir, f"{name}_{s}.tmp.npy")
            np.save(tmp, f)
            os.replace(tmp, os.path.join(outdir, f"{name}_{s}.npy"))      # atomic: the reader never sees a partial file
    open(os.path.join(outdir, f"{name}.done"), "w").write("ok\n")


if __name__ == "__main__":
    main()
