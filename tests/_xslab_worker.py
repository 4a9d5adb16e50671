"""Worker for tests/test_distributed_cpu.py: world_size-2 gloo run of the x-slab sharded SSP-RK3 plumbing
(paper_2202_13532_b200/sharded.py) with the ORACLE as the arithmetic backend, checked against the unsharded oracle.
Also importable: OracleSlabBackend is used in-process for the world = 1 case."""
import json
import math
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from oracle import fourier as ofr          # noqa: E402
from oracle import vlasov as ov            # noqa: E402
from paper_2202_13532_b200 import sharded  # noqa: E402
import workloads as wl                     # noqa: E402


class OracleSlabBackend:
    """CPU arithmetic for the plumbing tests.  The slab's exterior x states are imposed by padding one element on each
    side whose nodes all carry the halo plane (the upwind flux of Eq. 23 only reads the neighbour's face node) and
    running the oracle RHS with zero inflow in x on the padded grid; the padded elements' own results are dropped."""

    def __init__(self, nelem, order, lo, hi, bc, omega_c, pmax, e0, e1):
        self.n = order[0]
        self.lo, self.hi, self.N, self.pmax = lo[0], hi[0], nelem[0], pmax if pmax > 0 else nelem[0]
        lo_s, hi_s = sharded.slab_bounds(lo[0], hi[0], nelem[0], e0, e1)
        dx = (hi[0] - lo[0]) / nelem[0]
        nloc = e1 - e0
        self.slab = ov.Grid(nelem=(nloc,) + tuple(nelem[1:]), order=order, lo=(lo_s,) + tuple(lo[1:]), hi=(hi_s,) + tuple(hi[1:]),
                            bc=(1,) + tuple(bc[1:]), omega_c=omega_c, pmax=1)
        self.pad = ov.Grid(nelem=(nloc + 2,) + tuple(nelem[1:]), order=order, lo=(lo_s - dx,) + tuple(lo[1:]),
                           hi=(hi_s + dx,) + tuple(hi[1:]), bc=(1,) + tuple(bc[1:]), omega_c=omega_c, pmax=1)
        self.flat_shape = self.slab.flat_shape
        self.T = ofr.transform_tensor(self.lo, self.hi, self.N, self.n, self.pmax)
        self.x = ofr.node_coordinates(self.lo, self.hi, self.N, self.n)
        self.halo = None

    def empty(self, shape):
        return torch.zeros(shape, dtype=torch.float64)

    def density(self, f, out):
        out.copy_(torch.from_numpy(ov.density(self.slab, f.numpy())))
        return out

    def poisson_E(self, rho, out):
        c = ofr.fourier_project(self.T, rho.numpy())
        out.copy_(torch.from_numpy(ofr.poisson_E(self.lo, self.hi, self.x, c)))
        return out

    def set_halo(self, halo):
        self.halo = halo

    def stage_coeffs(self, stage):
        """Shu-Osher table as oracle.vlasov.ssprk3_step writes it out (reading C3)."""
        return ((0.0, 1.0), (0.75, 0.25), (1.0 / 3.0, 2.0 / 3.0))[stage]

    def rk_stage(self, f_s, f_n, E_loc, out, c0, c1, dt, rho_out=None):
        n = self.n
        fs = f_s.numpy()
        h = self.halo.numpy()
        left = np.broadcast_to(h[0][None], (n,) + h[0].shape)
        right = np.broadcast_to(h[1][None], (n,) + h[1].shape)
        fpad = np.concatenate([left, fs, right], axis=0)
        Epad = None if E_loc is None else np.concatenate([np.zeros(n), E_loc.numpy(), np.zeros(n)])
        r = ov.rhs(self.pad, fpad, Epad)[n:-n]
        res = c1 * (fs + dt * r)
        if f_n is not None and c0 != 0.0:
            res = c0 * f_n.numpy() + res
        out.copy_(torch.from_numpy(res))
        if rho_out is not None:
            rho_out.copy_(torch.from_numpy(ov.density(self.slab, res)))
        return out


CASE = dict(nelem=(5, 3, 3), order=(4, 4, 4), lo=(0.0, -6.0, -6.0), hi=(2 * math.pi / 0.3, 6.0, 6.0), bc=(0, 1, 1), omega_c=1.0, pmax=5)
K_WAVE, DT, NSTEPS = 0.3, 2e-3, 2


def initial_state(grid):
    f0 = wl.ring_f0(grid.coords[0].reshape(-1), grid.coords[1].reshape(-1), grid.coords[2].reshape(-1), K_WAVE)
    return wl.add_uniform_noise(f0, 77, 1e-3)


def run_sharded(rank, world, comm=None, self_consistent=True, bc0=0):
    case = dict(CASE); case["bc"] = (bc0,) + CASE["bc"][1:]
    g = ov.Grid(**case)
    f0 = initial_state(g)
    e0, e1 = sharded.slab_partition(case["nelem"][0], world)[rank]
    be = OracleSlabBackend(case["nelem"], case["order"], case["lo"], case["hi"], case["bc"], case["omega_c"], case["pmax"], e0, e1)
    st = sharded.XSlabStepper(case["nelem"], case["order"], case["lo"], case["hi"], bc=case["bc"], omega_c=case["omega_c"],
                              pmax=case["pmax"], rank=rank, world=world, backend=be, comm=comm)
    n = case["order"][0]
    f = torch.from_numpy(f0[e0 * n:e1 * n].copy())
    st.run(f, DT, NSTEPS, self_consistent)
    fo = f0.copy()
    for _ in range(NSTEPS):
        fo = ov.ssprk3_step(g, fo, DT, self_consistent=self_consistent)
    err = float(np.max(np.abs(f.numpy() - fo[e0 * n:e1 * n])) / np.max(np.abs(fo)))
    return err, (e0, e1)


if __name__ == "__main__":
    import torch.distributed as dist
    from paper_2202_13532_b200 import dist_util as du
    world, rank = du.init("gloo")
    out = {}
    staged = len(sys.argv) > 1 and sys.argv[1] == "hoststaged"      # the host-staged transport (sharded.HostStagedComm)
    for sc in (True, False):
        for bc0 in ((0, 1) if not sc else (0,)):
            err, part = run_sharded(rank, world, comm=sharded.HostStagedComm(rank, world) if staged else None,
                                    self_consistent=sc, bc0=bc0)
            err = du.max_over_ranks(err)
            out[f"err_sc{int(sc)}_bc{bc0}"] = err
    du.barrier()
    if rank == 0:
        out["world"] = world
        out["parts"] = sharded.slab_partition(CASE["nelem"][0], world)
        print(json.dumps(out), flush=True)
    du.finalize()
