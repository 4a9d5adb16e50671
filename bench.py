#!/usr/bin/env python
"""bench.py -- DOF-updates/s per RK stage of the fused DG RHS + SSP-RK3 step (with the Poisson
solve every stage) on the 1D2V production grid, through the C ABI (libdgvlasov.so).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A step = one SSP-RK3 step = 3 x (density -> c_p -> E -> fused RHS + stage combine) over the whole
grid.  Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "FP64 phase-space DOF-updates/s per RK stage"
UNIT = "DOF-updates/s"
K_WAVE = 0.1

WORKLOADS = {
    # BASELINE.json configs[2]: the production grid the north_star's 70 % target is quoted on
    "config3_1d2v_512^3": dict(nelem=(64, 64, 64), order=(8, 8, 8), dt=5e-4, noise=1e-4),
    # BASELINE.json configs[1]
    "config2_1d2v_256^3": dict(nelem=(32, 32, 32), order=(8, 8, 8), dt=1e-3, noise=0.0),
    # small replica for quick checks
    "small_1d2v_128^3": dict(nelem=(16, 16, 16), order=(8, 8, 8), dt=1e-3, noise=1e-4),
}
BYTES_PER_DOF_PER_STAGE = 64.0 / 3.0     # stage 1 reads f, writes u1 (16 B); stages 2,3 read f_s, f_n, write out (24 B)


def grid_args(w):
    return dict(nelem=w["nelem"], order=w["order"], lo=(0.0, -8.5, -8.5), hi=(2 * math.pi / K_WAVE, 8.5, 8.5),
                bc=(0, 1, 1), omega_c=1.0, pmax=w["nelem"][0])


def make_f0(x, vx, vy, w):
    import workloads as wl
    f0 = wl.ring_f0(x, vx, vy, K_WAVE)
    if w["noise"]:
        f0 = wl.add_uniform_noise(f0, wl.SEED_CFG3_NOISE, w["noise"])
    return np.ascontiguousarray(f0)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None
        self.t0 = self.t1 = None

    def wait_ready(self, timeout=5.0):
        """nvidia-smi takes a few hundred ms to print its first line: block until it has (so that a short timed region
        is not over before the first sample)."""
        t = time.perf_counter()
        while self.proc is not None and not self.lines and time.perf_counter() - t < timeout:
            time.sleep(0.01)

    def mark_begin(self):
        self.t0 = time.perf_counter()

    def mark_end(self):
        self.t1 = time.perf_counter()

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        # samples taken inside the timed region [mark_begin, mark_end] (+ one sampling period of slack on both sides);
        # all samples of the run if no marks were set
        lines = [(t, l) for t, l in self.lines
                 if self.t0 is None or self.t1 is None or (self.t0 - 0.05 <= t <= self.t1 + 0.05)]
        sm, mx, reasons = [], [], set()
        for _, l in lines:
            p = [s.strip() for s in l.split(",")]
            if len(p) < 8:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), p[4:8]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def measured_peak_hbm():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


# -----------------------------------------------------------------------------------------------
# reference arm: the oracle on the host cores, bounded sample of the same workload
# -----------------------------------------------------------------------------------------------
def oracle_sample(w, steps, warmup, x_elems=2):
    """One SSP-RK3 step of the oracle on an x-slab (x_elems of the N_x elements, full velocity grid,
    periodic in x within the slab) of the workload.  Returns (DOF-updates/s per stage, cores, description)."""
    from oracle import vlasov as ov
    import workloads as wl
    try:
        from threadpoolctl import threadpool_info
        cores = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        cores = os.cpu_count() or 1
    ga = grid_args(w)
    nelem = (x_elems,) + tuple(ga["nelem"][1:])
    hi = (ga["hi"][0] * x_elems / ga["nelem"][0],) + tuple(ga["hi"][1:])
    g = ov.Grid(nelem=nelem, order=ga["order"], lo=ga["lo"], hi=hi, bc=ga["bc"], omega_c=ga["omega_c"], pmax=x_elems)
    f = make_f0(g.coords[0].reshape(-1), g.coords[1].reshape(-1), g.coords[2].reshape(-1), w)
    for _ in range(warmup):
        ov.ssprk3_step(g, f, w["dt"])
    t0 = time.perf_counter()
    for _ in range(steps):
        f = ov.ssprk3_step(g, f, w["dt"])
    dt_wall = time.perf_counter() - t0
    dof = f.size
    value = dof * 3.0 * steps / dt_wall
    desc = (f"oracle.vlasov.ssprk3_step (NumPy), x-slab of {x_elems}/{ga['nelem'][0]} x-elements x full velocity grid "
            f"= {dof} DOF, {steps} step(s)")
    return value, cores, desc, dt_wall / max(steps, 1)


def run_reference(args, w, name):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    steps = max(1, min(args.steps, 3))
    value, cores, desc, sec_per_step = oracle_sample(w, steps, min(args.warmup, 1))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": min(args.warmup, 1), "ms_per_step": 1e3 * sec_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "note": "CPU oracle on a bounded x-slab sample of the workload"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# -----------------------------------------------------------------------------------------------
# our arm
# -----------------------------------------------------------------------------------------------
NCU_TRAFFIC_BYTES_PER_LAUNCH = {("config3_1d2v_512^3", "rhs_tiled<8,4>"): (2.110807e9 + 3.199168e9 + 3.185062e9) / 3.0}


def run_ours(args, w, name):
    import torch
    from paper_2202_13532_b200 import api, dist_util as du

    _, _, local = du.env_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the DG kernels have no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    world, rank = du.init("nccl", dev)

    def barrier():
        du.barrier(dev)

    def max_over_ranks(v):
        return du.max_over_ranks(v, dev)

    if args.parallelism in ("xslab", "xslab-push"):
        return run_xslab(args, w, name, world, rank, local, dev, barrier, max_over_ranks)
    ga = grid_args(w)
    ctx = api.DGContext(device=local, **ga)
    f0 = make_f0(ctx.nodes(0), ctx.nodes(1), ctx.nodes(2), w)
    dof = f0.size
    dt = w["dt"]
    f = torch.from_numpy(f0).to(dev)

    # warm-up, then K timed steps, device-timed, barrier + synchronize on both sides
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        sampler.wait_ready()
    ctx.ssprk3_run(f, dt, args.warmup, True)
    barrier()
    l0 = ctx.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.mark_begin()
    e0.record()
    ctx.ssprk3_run(f, dt, args.steps, True)
    e1.record()
    barrier()
    sampler.mark_end()
    ms = max_over_ranks(e0.elapsed_time(e1))
    clocks = sampler.stop() if rank == 0 else None
    launches = ctx.launch_count - l0
    finite = du.all_ranks_true(bool(torch.isfinite(f).all().item()), dev)
    value = du.replica_throughput(dof, 3, args.steps, ms, world)

    # roofline of the dominant kernel (fused RHS + stage): per-launch events inside the library
    ctx.set_option(api.OPT_PROFILE, 1)
    ctx.get_profile(reset=True)
    psteps = max(1, min(args.steps, 10))
    ctx.ssprk3_run(f, dt, psteps, True)
    rhs_ms, rhs_n = ctx.get_profile(reset=True)
    ctx.set_option(api.OPT_PROFILE, 0)
    kernel = ctx.last_kernel
    peak, peak_src = measured_peak_hbm()
    avg_launch_s = rhs_ms * 1e-3 / max(rhs_n, 1)
    achieved = BYTES_PER_DOF_PER_STAGE * dof / avg_launch_s / 1e9
    # dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full capture of this kernel on
    # this workload (profiles/r1_kernels.md: 2.111, 3.199, 3.185 GB for the three stages of a step); null elsewhere
    traffic = NCU_TRAFFIC_BYTES_PER_LAUNCH.get((name, kernel))
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_source": "profiles/r1_kernels.md (ncu --set full)" if traffic else None, "kernel": kernel, "avg_launch_ms": avg_launch_s * 1e3, "launches_timed": rhs_n,
                "algorithmic_bytes_per_launch": BYTES_PER_DOF_PER_STAGE * dof, "peak_source": peak_src,
                "rhs_share_of_step": (rhs_ms / psteps) / (ms / args.steps)}

    # end to end through the host-buffer entry point: H2D of f, K steps of 1, D2H of f, every step
    e2e_steps = max(1, min(args.steps, 3))
    fh = torch.from_numpy(f0.copy()).pin_memory()
    ctx.ssprk3_run_host(fh, dt, 1, True)          # warm-up (allocates the staging array)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        ctx.ssprk3_run_host(fh, dt, 1, True)
    barrier()
    e2e_s = max_over_ranks(time.perf_counter() - t0)
    e2e = {"value": world * dof * 3.0 * e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": dof * 8,
           "d2h_bytes_per_step": dof * 8, "steps": e2e_steps, "api": "dg_ssprk3_run_host (pinned host buffer)"}

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, cores, desc, _ = oracle_sample(w, 1, 0)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "grid": "x".join(str(n * o) for n, o in zip(w["nelem"], w["order"])), "dof": dof,
                       "dt": dt, "self_consistent_poisson_each_stage": True, "mass_mode": 0,
                       "l2": "inputs (3 x %.2f GB) larger than L2; no flush needed" % (dof * 8 / 1e9),
                       "parallelism": "replicas x%d" % world, "finite": finite},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu_baseline,
            "hbm_gbs_algorithmic_whole_step": 64.0 * dof * args.steps / (ms * 1e-3) / 1e9,
        }
        print(json.dumps(line), flush=True)
    ctx.close()
    du.finalize()


def run_xslab(args, w, name, world, rank, local, dev, barrier, max_over_ranks):
    """ONE problem sharded by x-slabs over the ranks (paper_2202_13532_b200/sharded.py): the workload's x
    extent and element count are multiplied by the number of ranks (weak scaling: every rank holds the workload's own
    grid), per stage an all-gather of rho and a face-plane exchange with the two x-neighbours over NCCL."""
    import torch
    from paper_2202_13532_b200 import api, dist_util as du, sharded
    ga = grid_args(w)
    nelem = (ga["nelem"][0] * world,) + tuple(ga["nelem"][1:])
    lo, hi = tuple(ga["lo"]), (ga["lo"][0] + (ga["hi"][0] - ga["lo"][0]) * world,) + tuple(ga["hi"][1:])
    st = sharded.XSlabStepper(nelem, ga["order"], lo, hi, bc=ga["bc"], omega_c=ga["omega_c"], pmax=ga["pmax"] * world,
                              rank=rank, world=world, device=local, push=(args.parallelism == "xslab-push"))
    slab = st.be.slab
    f0 = make_f0(slab.nodes(0), slab.nodes(1), slab.nodes(2), w)       # the same wave repeats in every slab
    dof, dt = f0.size, w["dt"]
    f = torch.from_numpy(f0).to(dev)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start(); sampler.wait_ready()
    st.run(f, dt, args.warmup, True)
    barrier()
    l0 = slab.launch_count + st.be.field.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.mark_begin()
    e0.record()
    st.run(f, dt, args.steps, True)
    e1.record()
    barrier()
    sampler.mark_end()
    ms = max_over_ranks(e0.elapsed_time(e1))
    clocks = sampler.stop() if rank == 0 else None
    launches = slab.launch_count + st.be.field.launch_count - l0
    finite = du.all_ranks_true(bool(torch.isfinite(f).all().item()), dev)
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": du.replica_throughput(dof, 3, args.steps, ms, world), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "grid": "x".join(str(n * o) for n, o in zip(nelem, ga["order"])), "dof": dof * world,
                       "dt": dt, "self_consistent_poisson_each_stage": True, "mass_mode": 0,
                       "l2": "inputs (3 x %.2f GB per rank) larger than L2; no flush needed" % (dof * 8 / 1e9),
                       "parallelism": ("xslab x%d (all-gather of rho + x-face planes stored into the neighbours' halos by the RHS kernel)"
                                       if st.push else "xslab x%d (all-gather of rho + x-face exchange per stage)") % world,
                       "finite": finite},
            "clocks": clocks, "gpu_launches": launches,
            "hbm_gbs_algorithmic_whole_step": 64.0 * dof * world * args.steps / (ms * 1e-3) / 1e9}), flush=True)
    st.close()
    du.finalize()


# -----------------------------------------------------------------------------------------------
# secondary workloads (BASELINE.json configs[3], configs[4]); not the driver's default line
# -----------------------------------------------------------------------------------------------
CONFIG4 = {"config4_rhs_n4": (4, 100), "config4_rhs_n6": (6, 67), "config4_rhs_n8": (8, 50), "config4_rhs_n10": (10, 40)}
FP64_ALU_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12     # DESIGN.md K3: SMs x DFMA/clk/SM x 2 flop x max SM clock


def run_config4(args, name):
    """RHS kernel alone (dg_rhs), seeded U(0,1) f and N(0,0.1^2) E, ~64 M DOF; a 'step' is one evaluation."""
    import torch
    import workloads as wl
    from paper_2202_13532_b200 import api
    n, N = CONFIG4[name]
    ctx = api.DGContext((N, N, N), (n, n, n), (0.0, -8.5, -8.5), (2 * math.pi / K_WAVE, 8.5, 8.5), bc=(0, 1, 1), omega_c=1.0,
                        workspace=False)
    G = n * N
    f = torch.from_numpy(wl.uniform_field((G, G, G), wl.SEED_CFG4_F)).cuda()
    E = torch.from_numpy(wl.normal_E(G, wl.SEED_CFG4_E)).cuda()
    out = torch.empty_like(f)
    for _ in range(max(args.warmup, 3)):
        ctx.rhs(f, E, out)
    torch.cuda.synchronize()
    sampler = ClockSampler(0); sampler.start(); sampler.wait_ready()
    l0 = ctx.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        ctx.rhs(f, E, out)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    dof = G ** 3
    peak, peak_src = measured_peak_hbm()
    achieved = 16.0 * dof * args.steps / (ms * 1e-3) / 1e9
    print(json.dumps({
        "metric": "FP64 phase-space DOF-updates/s per RHS evaluation", "value": dof * args.steps / (ms * 1e-3), "unit": UNIT,
        "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "order": n, "elements": N, "dof": dof, "l2": "arrays (2 x %.2f GB) larger than L2" % (dof * 8 / 1e9)},
        "clocks": clocks, "gpu_launches": ctx.launch_count - l0,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                     "kernel": ctx.last_kernel, "algorithmic_bytes_per_launch": 16.0 * dof, "peak_source": peak_src}}), flush=True)
    ctx.close()


CONFIG6 = {"config6_2d2v_128^4": (32, 4), "config6_2d2v_64^4": (16, 4), "config6_2d2v_n8_128^4": (16, 8), "config6_2d2v_n8_64^4": (8, 8)}


def oracle_sample_2d2v(dt):
    """Three SSP-RK3 steps of oracle.vlasov2d2v on a (4, 4, 32, 32)-element slab (4/32 of the x and y elements of the 128^4
    grid, periodic within the slab, full velocity grid): about 10-20 s of host time."""
    from oracle import vlasov2d2v as o4
    import workloads as wl
    try:
        from threadpoolctl import threadpool_info
        cores = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        cores = os.cpu_count() or 1
    L = 2 * math.pi / K_WAVE
    g = o4.make_grid((4, 4, 32, 32), (4,) * 4, (0.0, 0.0, -8.5, -8.5), (L / 8, L / 8, 8.5, 8.5), omega_c=1.0, pmax=(4, 4))
    x, y, u, v = [c.reshape(-1) for c in g.coords]
    f = wl.ring2d_f0(x, y, u, v, K_WAVE, K_WAVE)
    t0 = time.perf_counter()
    for _ in range(3):
        f = o4.ssprk3_step(g, f, dt)
    wall = time.perf_counter() - t0
    return f.size * 9.0 / wall, cores, f"oracle.vlasov2d2v.ssprk3_step (NumPy), (4, 4, 32, 32) x 4^4 slab = {f.size} DOF, 3 steps"


def run_config6(args, name):
    """2D2V: N^4 elements x n^4 LGL nodes (n = 4: tiled kernel; n = 8, the paper's order: element kernel), ring workload in (v_x, v_y) with a seeded perturbation in x and y,
    one SSP-RK3 step with the 2-D Poisson solve at every stage (dg4_ssprk3_run)."""
    import torch
    import workloads as wl
    from paper_2202_13532_b200 import api
    N, n = CONFIG6[name]
    lo, hi = (0.0, 0.0, -8.5, -8.5), (2 * math.pi / K_WAVE, 2 * math.pi / K_WAVE, 8.5, 8.5)
    ctx = api.DG4Context((N,) * 4, (n,) * 4, lo, hi, bc=(0, 0, 1, 1), omega_c=1.0)
    if args.rhs_kernel:
        ctx.set_option(api.OPT4_RHS_KERNEL, args.rhs_kernel)
    x, y, u, v = (ctx.nodes(d) for d in range(4))
    f0 = wl.add_uniform_noise(wl.ring2d_f0(x, y, u, v, K_WAVE, K_WAVE), wl.SEED_CFG6_NOISE, 1e-4)
    f = torch.from_numpy(f0).cuda()
    dt = 2e-4 if n == 4 else 5e-5
    ctx.ssprk3_run(f, dt, max(args.warmup, 3))
    torch.cuda.synchronize()
    sampler = ClockSampler(0); sampler.start(); sampler.wait_ready()
    l0 = ctx.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.mark_begin()
    e0.record()
    ctx.ssprk3_run(f, dt, args.steps)
    e1.record()
    torch.cuda.synchronize()
    sampler.mark_end()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    launches = ctx.launch_count - l0
    finite = bool(torch.isfinite(f).all().item())
    # per-launch time of the RHS kernel: events recorded by the library around each launch, in a separate pass
    ctx.set_option(api.OPT4_PROFILE, 1)
    ctx.get_profile(reset=True)
    ctx.ssprk3_run(f, dt, 10)
    rhs_ms, rhs_n = ctx.get_profile(reset=True)
    ctx.set_option(api.OPT4_PROFILE, 0)
    dof = (n * N) ** 4
    peak, peak_src = measured_peak_hbm()
    bytes_per_launch = 64.0 / 3.0 * dof
    achieved = bytes_per_launch / (rhs_ms / rhs_n * 1e-3) / 1e9
    # end to end through dg4_ssprk3_run_host
    fh = torch.from_numpy(f0).pin_memory()
    ctx.ssprk3_run_host(fh, dt, 1)
    t0 = time.perf_counter()
    e2e_steps = 2
    for _ in range(e2e_steps):
        ctx.ssprk3_run_host(fh, dt, 1)
    e2e_s = time.perf_counter() - t0
    cpu = None
    if not args.no_cpu_baseline:
        cv, cc, cd = oracle_sample_2d2v(dt)
        cpu = {"value": cv, "unit": UNIT, "cores": cc, "kind": "oracle", "sample": cd}
    print(json.dumps({
        "cpu_baseline": cpu,
        "metric": "FP64 phase-space DOF-updates/s per RK stage", "value": dof * 3.0 * args.steps / (ms * 1e-3), "unit": UNIT,
        "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "grid": "x".join([str(n * N)] * 4), "order": n, "dof": dof, "dt": dt, "self_consistent_poisson_each_stage": True,
                   "l2": "arrays (3 x %.2f GB) larger than L2" % (dof * 8 / 1e9), "finite": finite},
        "clocks": clocks, "gpu_launches": launches,
        "e2e": {"value": dof * 3.0 * e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": dof * 8, "d2h_bytes_per_step": dof * 8,
                "steps": e2e_steps, "api": "dg4_ssprk3_run_host (pinned host buffer)"},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                     "kernel": ctx.last_kernel, "avg_launch_ms": rhs_ms / rhs_n, "launches_timed": rhs_n,
                     "algorithmic_bytes_per_launch": bytes_per_launch, "peak_source": peak_src,
                     "rhs_share_of_step": 3.0 * (rhs_ms / rhs_n) / (ms / args.steps)}}), flush=True)
    ctx.close()


def run_config5(args, name):
    """DG->Fourier projection + spectral Poisson solve alone: 2048 x 8 x-nodes, batch 4096, modes <= 8192."""
    import torch
    import workloads as wl
    from paper_2202_13532_b200 import api
    N, n, pmax, batch = 2048, 8, 8192, args.batch
    t0 = time.perf_counter()
    fk = {"auto": api.FIELD_AUTO, "dmma": api.FIELD_DMMA, "dfma": api.FIELD_DFMA, "fft": api.FIELD_FFT}[args.field_kernel]
    fft = fk in (api.FIELD_AUTO, api.FIELD_FFT)      # auto takes the FFT-factorised kernel on this grid (2048 = 2^11 elements)
    ctx = api.DGContext((N,), (n,), (0.0,), (2 * math.pi,), pmax=pmax, field_batch=batch, workspace=not fft)
    ctx.set_option(api.OPT_FIELD_KERNEL, fk)
    t_create = time.perf_counter() - t0
    x = ctx.nodes(0)
    rho_h, _, _, _ = wl.cosine_sum_density(x, batch, wl.SEED_CFG5)
    rho = torch.from_numpy(rho_h).cuda()
    E = torch.empty_like(rho)
    for _ in range(max(args.warmup, 3)):
        ctx.poisson_E(rho, E)
    torch.cuda.synchronize()
    sampler = ClockSampler(0); sampler.start(); sampler.wait_ready()
    l0 = ctx.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        ctx.poisson_E(rho, E)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    G, Q = N * n, 2 * (pmax + 1)
    flops = 2.0 * 2.0 * batch * G * Q            # projection + synthesis, 2 flop per multiply-add
    tf = flops * args.steps / (ms * 1e-3) / 1e12
    if fft:
        # same result as the dense contraction (parity-tested against the same oracle); the kernel is bound by reading
        # rho and writing E once: 16 B per x node per vector
        gbs = 2.0 * batch * G * 8 * args.steps / (ms * 1e-3) / 1e9
        peak, src = measured_peak_hbm()
        print(json.dumps({
            "metric": "density vectors/s through projection + Poisson solve (FFT-factorised)", "value": batch * args.steps / (ms * 1e-3),
            "unit": "vectors/s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "x_nodes": G, "batch": batch, "modes": pmax, "dg_create_s": t_create,
                       "l2": "rho and E (2 x %.2f GB) larger than L2" % (batch * G * 8 / 1e9),
                       "dense_equivalent_tflops": tf},
            "clocks": clocks, "gpu_launches": ctx.launch_count - l0,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "traffic": None,
                         "kernel": "field_fft_kernel<4>", "peak_source": src,
                         "algorithmic_bytes_per_launch": 2.0 * batch * G * 8}}), flush=True)
        ctx.close()
        return
    print(json.dumps({
        "metric": "FP64 TFLOP/s of projection + Poisson synthesis (dense contraction)", "value": tf, "unit": "TFLOP/s",
        "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "x_nodes": G, "batch": batch, "modes": pmax, "dg_create_s": t_create,
                   "l2": "T and S (2 x %.2f GB) larger than L2" % (G * Q * 8 / 1e9)},
        "clocks": clocks, "gpu_launches": ctx.launch_count - l0,
        "roofline": {"bound": "alu", "achieved": tf, "peak": FP64_ALU_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": tf / FP64_ALU_PEAK_TFLOPS,
                     "traffic": None, "kernel": "field_gemm_dmma_kernel",
                     "peak_source": "148 SM x 64 FP64 FMA/clk x 2 x 1.965 GHz (DESIGN.md K3; DFMA and DMMA both measure 37.0)"}}), flush=True)
    ctx.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config3_1d2v_512^3", choices=sorted(WORKLOADS) + sorted(CONFIG4) + ["config5_field"] + sorted(CONFIG6))
    ap.add_argument("--batch", type=int, default=4096, help="config5_field only")
    ap.add_argument("--field-kernel", default="auto", choices=["auto", "dmma", "dfma", "fft"], help="config5_field only")
    ap.add_argument("--parallelism", default="replicas", choices=["replicas", "xslab", "xslab-push"],
                    help="N > 1: independent replicas (default, DESIGN.md section 9) or one problem sharded by x-slabs, with the "
                         "face planes exchanged by send/recv (xslab) or stored by the RHS kernel into peer memory (xslab-push)")
    ap.add_argument("--rhs-kernel", type=int, default=0, help="config6 only: DG4_OPT_RHS_KERNEL (0 auto)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.workload in CONFIG4:
        return run_config4(args, args.workload)
    if args.workload == "config5_field":
        return run_config5(args, args.workload)
    if args.workload in CONFIG6:
        return run_config6(args, args.workload)
    w = WORKLOADS[args.workload]
    if args.impl == "reference":
        run_reference(args, w, args.workload)
    else:
        run_ours(args, w, args.workload)


if __name__ == "__main__":
    main()
