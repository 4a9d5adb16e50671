"""Multi-rank plumbing for bench.py: one process per GPU, replicas of the workload.

The data path has no collective in round 1 (each rank advances its own replica); torch.distributed carries only
the barrier and the max-over-ranks of the device time.  Backend "nccl" on GPUs, "gloo" in the CPU tests."""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def env_world():
    return (int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")))


def init(backend: str, device=None, log_nccl: bool = False):
    """log_nccl (bench.py passes it; off for every other caller): send NCCL's communicator lines to a per-process file and
    have rank 0 echo its "Init COMPLETE" line to stderr after the first collective, so that a reader of the bench log can
    see the N ranks.  Without it the caller's environment is left alone and no file is written."""
    world, rank, _ = env_world()
    if world > 1 and not dist.is_initialized():
        kw = {}
        log = None
        if backend == "nccl" and device is not None:
            kw["device_id"] = device
            if log_nccl:
                os.environ.setdefault("NCCL_DEBUG", "INFO")
                os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
                log = os.environ.setdefault("NCCL_DEBUG_FILE", "/tmp/dg_nccl_%h_%p.log")
        dist.init_process_group(backend, **kw)
        if log is not None:
            dist.barrier()
            _echo_nccl_init(log, rank)
    return world, rank


def _echo_nccl_init(pattern: str, rank: int):
    import socket
    import sys
    path = pattern.replace("%h", socket.gethostname()).replace("%p", str(os.getpid()))
    try:
        with open(path) as fh:
            lines = [l.rstrip() for l in fh if "Init COMPLETE" in l or "nranks" in l]
    except OSError:
        return
    if rank == 0:
        for l in lines[-2:]:
            print("[nccl] " + l, file=sys.stderr, flush=True)


def barrier(device=None):
    if dist.is_initialized():
        dist.barrier()
    if device is not None and device.type == "cuda":
        torch.cuda.synchronize(device)


def max_over_ranks(value: float, device=None) -> float:
    """Slowest rank's time: every multi-GPU number is the max over ranks, never a wall clock."""
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def all_ranks_true(flag: bool, device=None) -> bool:
    if not dist.is_initialized():
        return bool(flag)
    t = torch.tensor([1.0 if flag else 0.0], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MIN)
    return bool(t.item() > 0.5)


def replica_throughput(dof_per_rank: int, stages_per_step: int, steps: int, ms_max: float, world: int) -> float:
    """Whole-job DOF-updates/s per RK stage of `world` replicas that all finished within ms_max."""
    return world * dof_per_rank * float(stages_per_step) * steps / (ms_max * 1e-3)


def finalize():
    if dist.is_initialized():
        dist.destroy_process_group()
