"""Worker for tests/test_gpu_xslab.py::test_two_gpu_xslab_matches_unsharded_oracle: one rank per GPU (torchrun, NCCL),
the x-slab sharded SSP-RK3 step of paper_2202_13532_b200/sharded.py through the library's kernels (CudaBackend), checked
against the UNSHARDED oracle.  argv[1] = "push" selects the fused face push into the neighbours' halo buffers
(symmetric memory); "hoststaged" puts EVERY rank on cuda:0 with a gloo group and sharded.HostStagedComm (concurrent
processes on the one GPU of a single-GPU box); anything else the plain send/recv exchange.  Prints one JSON line on rank 0."""
import json
import math
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from oracle import vlasov as ov                         # noqa: E402
from paper_2202_13532_b200 import dist_util as du       # noqa: E402
from paper_2202_13532_b200 import sharded               # noqa: E402
import workloads as wl                                  # noqa: E402

K_WAVE, DT, NSTEPS = 0.1, 1e-3, 3
CASE = dict(nelem=(5, 2, 5), order=(8, 8, 8), lo=(0.0, -8.5, -8.5), hi=(2 * math.pi / K_WAVE, 8.5, 8.5), bc=(0, 1, 1), omega_c=1.0, pmax=5)


def main():
    push = len(sys.argv) > 1 and sys.argv[1] == "push"
    staged = len(sys.argv) > 1 and sys.argv[1] == "hoststaged"
    _, _, local = du.env_world()
    if staged:
        local = 0
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    world, rank = du.init("gloo") if staged else du.init("nccl", dev)
    out = {"world": world, "push": push, "staged": staged, "pid": os.getpid()}
    for sc in (True, False):
        for bc0 in ((0,) if sc else (0, 1)):
            case = dict(CASE); case["bc"] = (bc0,) + CASE["bc"][1:]
            g = ov.Grid(**case)
            f0 = wl.add_uniform_noise(wl.ring_f0(g.coords[0].reshape(-1), g.coords[1].reshape(-1), g.coords[2].reshape(-1), K_WAVE), 77, 1e-3)
            st = sharded.XSlabStepper(case["nelem"], case["order"], case["lo"], case["hi"], bc=case["bc"], omega_c=case["omega_c"],
                                      pmax=case["pmax"], rank=rank, world=world, device=local, push=push,
                                      comm=sharded.HostStagedComm(rank, world) if staged else None)
            n = case["order"][0]
            f = torch.from_numpy(f0[st.e0 * n:st.e1 * n].copy()).to(dev)
            st.run(f, DT, NSTEPS, sc)
            fo = f0.copy()
            for _ in range(NSTEPS):
                fo = ov.ssprk3_step(g, fo, DT, self_consistent=sc)
            err = float(np.max(np.abs(f.cpu().numpy() - fo[st.e0 * n:st.e1 * n])) / np.max(np.abs(fo)))
            out[f"err_sc{int(sc)}_bc{bc0}"] = du.max_over_ranks(err, None if staged else dev)
            out[f"slab_sc{int(sc)}_bc{bc0}"] = [st.e0, st.e1]
            st.close()
    du.barrier(dev)
    if staged:
        pids = [None] * world
        torch.distributed.all_gather_object(pids, os.getpid())
        out["pids"] = pids
    if rank == 0:
        print(json.dumps(out), flush=True)
    du.finalize()


if __name__ == "__main__":
    main()
