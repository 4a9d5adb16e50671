#!/usr/bin/env python
"""bench.py -- DOF-updates/s per RK stage of the fused DG RHS + SSP-RK3 step (with the Poisson
solve every stage) on the 1D2V production grid, through the C ABI (libdgvlasov.so).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A step = one SSP-RK3 step = 3 x (density -> c_p -> E -> fused RHS + stage combine) over the whole
grid.  Prints ONE JSON line (rank 0).  See DESIGN.md section 7 for every field.

With --gpus N > 1 and no torchrun environment the script starts the N ranks itself
(python -m torch.distributed.run ... bench.py, 127.0.0.1 rendezvous); under torchrun it reads
RANK / LOCAL_RANK / WORLD_SIZE as usual.
"""
from __future__ import annotations

import argparse
import csv
import hashlib
import json
import math
import os
import socket
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
# DESIGN.md section 5 K1: stage 1 reads f, writes u1 (16 B/DOF); stages 2, 3 read f_s, f_n, write out (24 B/DOF)
STAGE_BYTES_PER_DOF = (16.0, 24.0, 24.0)
BYTES_PER_DOF_PER_STAGE = sum(STAGE_BYTES_PER_DOF) / 3.0
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
KERNEL_SOURCES = {"rhs_tiled": "dg_kernels_tiled.cuh", "rhs4_tile": "dg4_kernels_tiled.cuh", "rhs4_elem": "dg4_kernels_elem.cuh",
                  "rhs4_line": "dg4_kernels_line.cuh", "field_fft": "dg_kernels_fft.cuh", "field_gemm": "dg_kernels_field.cuh"}


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
        return self

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def window(self, t0, t1):
        """Summary of the samples taken in [t0, t1] (+ one sampling period of slack on both sides)."""
        lines = [(t, l) for t, l in self.lines if t0 is None or t1 is None or (t0 - 0.05 <= t <= t1 + 0.05)]
        sm, mx, pw, reasons = [], [], [], set()
        for _, l in lines:
            p = [s.strip() for s in l.split(",")]
            if len(p) < 8:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1]))
            except ValueError:
                continue
            try:
                pw.append(float(p[2]))
            except ValueError:
                pass
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), p[4:8]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_min_mhz": min(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "power_w": float(np.median(pw)) if pw else None,
                "reasons": sorted(reasons), "samples": len(sm)}

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        return self.window(self.t0, self.t1)


def measured_peak_hbm():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def ncu_traffic(workload, kernel, stage=None):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on `workload` from the tracked ncu --set full
    capture (profiles/ncu_traffic.csv; the commands of its captures are listed in profiles/r2_kernels.md).  The
    capture records the SHA-256 of the kernel's source file; if the source has changed since, the figure is stale and None
    is returned (with the reason)."""
    if not os.path.exists(TRAFFIC_CSV):
        return None, "no capture (profiles/ncu_traffic.csv missing)"
    rows = [r for r in csv.DictReader(open(TRAFFIC_CSV)) if r["workload"] == workload and r["kernel"] == kernel]
    if stage is not None:
        rows = [r for r in rows if r["stage"] == str(stage)]
    if not rows:
        return None, "no capture of this kernel on this workload"
    src = next((f for k, f in KERNEL_SOURCES.items() if kernel.startswith(k)), None)
    if src:
        path = os.path.join(ROOT, "paper_2202_13532_b200", "csrc", src)
        sha = hashlib.sha256(open(path, "rb").read()).hexdigest()[:16] if os.path.exists(path) else "missing"
        if any(r["source_sha16"] != sha for r in rows):
            return None, "stale: %s changed since the capture" % src
    per_launch = [float(r["dram_bytes_read"]) + float(r["dram_bytes_write"]) for r in rows]
    per_launch = [v for v in per_launch if v == v]            # a launch whose DRAM counters ncu could not collect
    if not per_launch:
        return None, "capture holds no DRAM byte counts for this kernel"
    return sum(per_launch) / len(per_launch), "profiles/ncu_traffic.csv (%s)" % rows[0]["capture"]


def host_cores():
    try:
        from threadpoolctl import threadpool_info
        return max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        return os.cpu_count() or 1


# -----------------------------------------------------------------------------------------------
# reference arm: the oracle on the host cores, bounded sample of the same workload
# -----------------------------------------------------------------------------------------------
def oracle_sample(w, steps, warmup, x_elems=2, threads=None):
    """SSP-RK3 steps of the oracle on an x-slab (x_elems of the N_x elements, full velocity grid,
    periodic in x within the slab) of the workload.  threads: BLAS thread limit (None = all cores).
    Returns (DOF-updates/s per stage, cores, description, seconds per step)."""
    from oracle import vlasov as ov
    ga = grid_args(w)
    nelem = (x_elems,) + tuple(ga["nelem"][1:])
    hi = (ga["hi"][0] * x_elems / ga["nelem"][0],) + tuple(ga["hi"][1:])
    g = ov.Grid(nelem=nelem, order=ga["order"], lo=ga["lo"], hi=hi, bc=ga["bc"], omega_c=ga["omega_c"], pmax=x_elems)
    f = make_f0(g.coords[0].reshape(-1), g.coords[1].reshape(-1), g.coords[2].reshape(-1), w)

    def run():
        nonlocal f
        for _ in range(warmup):
            ov.ssprk3_step(g, f, w["dt"])
        t0 = time.perf_counter()
        for _ in range(steps):
            f = ov.ssprk3_step(g, f, w["dt"])
        return time.perf_counter() - t0

    if threads is not None:
        from threadpoolctl import threadpool_limits
        with threadpool_limits(limits=threads):
            dt_wall = run()
        cores = threads
    else:
        dt_wall = run()
        cores = host_cores()
    dof = f.size
    value = dof * 3.0 * steps / dt_wall
    desc = (f"oracle.vlasov.ssprk3_step (NumPy), x-slab of {x_elems}/{ga['nelem'][0]} x-elements x full velocity grid "
            f"= {dof} DOF, {steps} step(s), {cores} thread(s)")
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


def run_oracle_timing(args):
    """the oracle as it stands on the host cores, 1 thread and all cores -- one RHS and one SSP-RK3 step
    at config 2 size (256^3), one step at config 3 size (512^3; the 1000-step total is extrapolated, not run)."""
    from oracle import vlasov as ov
    from threadpoolctl import threadpool_limits
    out = {"workload": "oracle_timing", "cores_all": host_cores(), "rows": []}
    for name in ("config2_1d2v_256^3", "config3_1d2v_512^3"):
        w = WORKLOADS[name]
        ga = grid_args(w)
        g = ov.Grid(nelem=ga["nelem"], order=ga["order"], lo=ga["lo"], hi=ga["hi"], bc=ga["bc"], omega_c=ga["omega_c"], pmax=ga["pmax"])
        f = make_f0(g.coords[0].reshape(-1), g.coords[1].reshape(-1), g.coords[2].reshape(-1), w)
        for threads in (1, None):
            if name.startswith("config3") and threads == 1 and not args.full:
                continue                       # ~2 min single-threaded: only with --full
            ctxm = threadpool_limits(limits=threads) if threads else threadpool_limits(limits=None)
            with ctxm:
                t_rhs = None
                if name.startswith("config2"):
                    E = ov.field_E(g, f)
                    t0 = time.perf_counter(); ov.rhs(g, f, E); t_rhs = time.perf_counter() - t0
                t0 = time.perf_counter(); ov.ssprk3_step(g, f, w["dt"]); t_step = time.perf_counter() - t0
            out["rows"].append({"config": name, "dof": f.size, "threads": threads or out["cores_all"], "rhs_s": t_rhs, "step_s": t_step,
                                "dof_updates_per_s_per_stage": 3.0 * f.size / t_step})
    print(json.dumps(out), flush=True)


# -----------------------------------------------------------------------------------------------
# our arm
# -----------------------------------------------------------------------------------------------
def profile_stride(steps):
    """DG_OPT_PROFILE stride for a region of `steps` steps: coprime to 3 so that the bracketed launches cycle through the stages."""
    n = 3 * steps
    return 7 if n >= 42 else (4 if n >= 12 else (2 if n >= 6 else 1))


def stage_roofline(ctx_kernel, dof, ms4, n4, peak, peak_src, workload, step_ms):
    """Roofline of the fused RHS + stage kernel from per-stage CUDA-event samples taken INSIDE the timed region."""
    stages, avg = [], []
    for s in (1, 2, 3):
        if n4[s] == 0:
            continue
        ms = ms4[s] / n4[s]
        gbs = STAGE_BYTES_PER_DOF[s - 1] * dof / (ms * 1e-3) / 1e9
        tr, _ = ncu_traffic(workload, ctx_kernel, s)
        stages.append({"stage": s, "avg_launch_ms": ms, "launches_timed": n4[s], "algorithmic_bytes": STAGE_BYTES_PER_DOF[s - 1] * dof,
                       "achieved": gbs, "frac": gbs / peak, "traffic": tr})
        avg.append(ms)
    if len(avg) < 3:
        return None
    mean_ms = sum(avg) / 3.0
    achieved = BYTES_PER_DOF_PER_STAGE * dof / (mean_ms * 1e-3) / 1e9
    traffic, tsrc = ncu_traffic(workload, ctx_kernel)
    return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
            "traffic_source": tsrc, "kernel": ctx_kernel, "avg_launch_ms": mean_ms, "launches_timed": int(sum(n4[1:])),
            "algorithmic_bytes_per_launch": BYTES_PER_DOF_PER_STAGE * dof, "peak_source": peak_src, "stages": stages,
            "rhs_share_of_step": 3.0 * mean_ms / step_ms,
            "how": "CUDA events recorded by the library around every k-th RHS launch inside the timed region (DG_OPT_PROFILE = k, "
                   "programmatic launches on); mean of the three per-stage means"}


def timed_run(ctx, f, dt, steps, sampler, barrier, max_over_ranks, api):
    """`steps` SSP-RK3 steps in one dg_ssprk3_run call, device-timed, with per-stage samples of the RHS kernel."""
    import torch
    ctx.set_option(api.OPT_PROFILE, profile_stride(steps))
    ctx.get_profile_stages(reset=True)
    l0 = ctx.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0 = time.perf_counter()
    e0.record()
    ctx.ssprk3_run(f, dt, steps, True)
    e1.record()
    barrier()
    t1 = time.perf_counter()
    ms = max_over_ranks(e0.elapsed_time(e1))
    ms4, n4 = ctx.get_profile_stages(reset=True)
    ctx.set_option(api.OPT_PROFILE, 0)
    return ms, ms4, n4, ctx.launch_count - l0, (t0, t1)


def run_ours(args, w, name):
    import torch
    from paper_2202_13532_b200 import api, dist_util as du

    _, _, local = du.env_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the DG kernels have no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    world, rank = du.init("nccl", dev, log_nccl=True)

    def barrier():
        du.barrier(dev)

    def max_over_ranks(v):
        return du.max_over_ranks(v, dev)

    parallelism = args.parallelism if args.parallelism != "auto" else ("replicas" if world == 1 else "xslab")
    if parallelism in ("xslab", "xslab-push"):
        return run_xslab(args, w, name, world, rank, local, dev, barrier, max_over_ranks, parallelism)
    ga = grid_args(w)
    ctx = api.DGContext(device=local, **ga)
    f0 = make_f0(ctx.nodes(0), ctx.nodes(1), ctx.nodes(2), w)
    dof = f0.size
    dt = w["dt"]
    f = torch.from_numpy(f0).to(dev)
    peak, peak_src = measured_peak_hbm()

    # warm-up, then K timed steps, device-timed, barrier + synchronize on both sides
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        sampler.wait_ready()
    ctx.ssprk3_run(f, dt, args.warmup, True)
    barrier()
    ms, ms4, n4, launches, (t0, t1) = timed_run(ctx, f, dt, args.steps, sampler, barrier, max_over_ranks, api)
    clocks = sampler.window(t0, t1) if rank == 0 else None
    flag = ctx.check_finite(f)
    finite = du.all_ranks_true(int(flag.item()) == 0, dev)
    value = du.replica_throughput(dof, 3, args.steps, ms, world)
    kernel = ctx.last_kernel
    roofline = stage_roofline(kernel, dof, ms4, n4, peak, peak_src, name, ms / args.steps)
    if roofline is None:
        # too few launches in the region for a per-stage sample: the kernel alone, every launch bracketed (no programmatic launches)
        ctx.set_option(api.OPT_PROFILE, 1)
        ctx.get_profile_stages(reset=True)
        ctx.ssprk3_run(f, dt, 3, True)
        m4, c4 = ctx.get_profile_stages(reset=True)
        ctx.set_option(api.OPT_PROFILE, 0)
        roofline = stage_roofline(kernel, dof, m4, c4, peak, peak_src, name, ms / args.steps)
        roofline["how"] = "separate 3-step pass with every RHS launch bracketed (the timed region had fewer than 6 launches)"

    # sustained: >= 1000 steps of the same workload (config 3 is a 1000-step run), clocks sampled inside the region
    sustained = None
    if args.sustained_steps > 0:
        sms, sm4, sn4, _, (s0, s1) = timed_run(ctx, f, dt, args.sustained_steps, sampler, barrier, max_over_ranks, api)
        srf = stage_roofline(kernel, dof, sm4, sn4, peak, peak_src, name, sms / args.sustained_steps)
        sflag = ctx.check_finite(f)
        sustained = {"steps": args.sustained_steps, "ms_per_step": sms / args.sustained_steps,
                     "value": du.replica_throughput(dof, 3, args.sustained_steps, sms, world), "unit": UNIT,
                     "hbm_gbs_algorithmic_whole_step": 64.0 * dof * args.sustained_steps / (sms * 1e-3) / 1e9,
                     "frac_whole_step": 64.0 * dof * args.sustained_steps / (sms * 1e-3) / 1e9 / peak,
                     "clocks": sampler.window(s0, s1) if rank == 0 else None,
                     "finite": du.all_ranks_true(int(sflag.item()) == 0, dev),
                     "rhs_stages": None if srf is None else [{k: s[k] for k in ("stage", "avg_launch_ms", "frac", "launches_timed")} for s in srf["stages"]],
                     "rhs_share_of_step": None if srf is None else srf["rhs_share_of_step"]}
    if rank == 0:
        sampler.stop()

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
    ctx.close()
    del f, fh
    torch.cuda.empty_cache()

    secondary = None
    if rank == 0 and world == 1 and not args.no_secondary and name == "config3_1d2v_512^3":
        secondary = run_secondary(args)

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, cores, desc, _ = oracle_sample(w, 3, 0)
        v1, _, desc1, _ = oracle_sample(w, 1, 0, threads=1)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                        "single_thread": {"value": v1, "unit": UNIT, "cores": 1, "sample": desc1}}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            # the 1000-step form of the config, flat and early in the line so that a truncated stored copy keeps it
            **({} if sustained is None else {
                "sustained_ms_per_step": sustained["ms_per_step"], "sustained_frac_whole_step": sustained["frac_whole_step"],
                "sustained_stage_fracs": None if not sustained["rhs_stages"] else [s["frac"] for s in sustained["rhs_stages"]],
                "sustained_sm_mhz": (sustained["clocks"] or {}).get("sm_mhz"),
                "sustained_clock_reasons": (sustained["clocks"] or {}).get("reasons")}),
            "config": {"workload": name, "grid": "x".join(str(n * o) for n, o in zip(w["nelem"], w["order"])), "dof": dof,
                       "dt": dt, "self_consistent_poisson_each_stage": True, "mass_mode": 0,
                       "l2": "inputs (3 x %.2f GB) larger than L2; no flush needed" % (dof * 8 / 1e9),
                       "parallelism": "replicas x%d" % world, "finite": finite},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu_baseline,
            "hbm_gbs_algorithmic_whole_step": 64.0 * dof * args.steps / (ms * 1e-3) / 1e9,
            "frac_whole_step": 64.0 * dof * args.steps / (ms * 1e-3) / 1e9 / peak,
            "sustained": sustained, "secondary": secondary,
        }
        print(json.dumps(line), flush=True)
    du.finalize()


def run_xslab(args, w, name, world, rank, local, dev, barrier, max_over_ranks, parallelism):
    """ONE problem sharded by x-slabs over the ranks (paper_2202_13532_b200/sharded.py): the workload's x
    extent and element count are multiplied by the number of ranks (weak scaling: every rank holds the workload's own
    grid), per stage an all-gather of rho and a face-plane exchange with the two x-neighbours over NCCL."""
    import torch
    from paper_2202_13532_b200 import api, dist_util as du, sharded
    ga = grid_args(w)
    nelem = (ga["nelem"][0] * world,) + tuple(ga["nelem"][1:])
    lo, hi = tuple(ga["lo"]), (ga["lo"][0] + (ga["hi"][0] - ga["lo"][0]) * world,) + tuple(ga["hi"][1:])
    st = sharded.XSlabStepper(nelem, ga["order"], lo, hi, bc=ga["bc"], omega_c=ga["omega_c"], pmax=ga["pmax"] * world,
                              rank=rank, world=world, device=local, push=(parallelism == "xslab-push"))
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
    finite = du.all_ranks_true(int(slab.check_finite(f).item()) == 0, dev)
    peak, _ = measured_peak_hbm()
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
            "hbm_gbs_algorithmic_whole_step": 64.0 * dof * world * args.steps / (ms * 1e-3) / 1e9,
            "frac_whole_step_per_gpu": 64.0 * dof * args.steps / (ms * 1e-3) / 1e9 / peak}), flush=True)
    st.close()
    du.finalize()


# -----------------------------------------------------------------------------------------------
# secondary workloads (BASELINE.json configs[1], [3], [4] and the 2D2V config 6)
# -----------------------------------------------------------------------------------------------
CONFIG4 = {"config4_rhs_n4": (4, 100), "config4_rhs_n6": (6, 67), "config4_rhs_n8": (8, 50), "config4_rhs_n10": (10, 40)}
FP64_ALU_PEAK_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12     # SMs x FP64 FMA/clk/SM x 2 flop x max SM clock


def _dev_uniform(shape, seed):
    """Seeded U(0,1) field generated on the device (secondary throughput runs only; the parity tests use workloads.py)."""
    import torch
    g = torch.Generator(device="cuda"); g.manual_seed(seed)
    return torch.rand(shape, dtype=torch.float64, device="cuda", generator=g)


def _clocks_during(fn):
    s = ClockSampler(0).start(); s.wait_ready()
    s.mark_begin()
    r = fn()
    s.mark_end()
    return r, s.stop()


def run_config4(args, name, host_inputs=True):
    """RHS kernel alone (dg_rhs), seeded U(0,1) f and N(0,0.1^2) E, ~64 M DOF; a 'step' is one evaluation."""
    import torch
    import workloads as wl
    from paper_2202_13532_b200 import api
    n, N = CONFIG4[name]
    ctx = api.DGContext((N, N, N), (n, n, n), (0.0, -8.5, -8.5), (2 * math.pi / K_WAVE, 8.5, 8.5), bc=(0, 1, 1), omega_c=1.0,
                        workspace=False)
    G = n * N
    if host_inputs:
        f = torch.from_numpy(wl.uniform_field((G, G, G), wl.SEED_CFG4_F)).cuda()
    else:
        f = _dev_uniform((G, G, G), wl.SEED_CFG4_F)
    E = torch.from_numpy(wl.normal_E(G, wl.SEED_CFG4_E)).cuda()
    out = torch.empty_like(f)
    warm = max(args.warmup, 3)
    for _ in range(warm):
        ctx.rhs(f, E, out)
    torch.cuda.synchronize()
    steps = args.steps

    def region():
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            ctx.rhs(f, E, out)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    l0 = ctx.launch_count
    ms, clocks = _clocks_during(region)
    dof = G ** 3
    peak, peak_src = measured_peak_hbm()
    achieved = 16.0 * dof * steps / (ms * 1e-3) / 1e9
    traffic, tsrc = ncu_traffic(name, ctx.last_kernel)
    line = {
        "metric": "FP64 phase-space DOF-updates/s per RHS evaluation", "value": dof * steps / (ms * 1e-3), "unit": UNIT,
        "n_gpus": 1, "steps": steps, "warmup": warm, "ms_per_step": ms / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "order": n, "elements": N, "dof": dof, "l2": "arrays (2 x %.2f GB) larger than L2" % (dof * 8 / 1e9),
                   "inputs": "workloads.py (host)" if host_inputs else "seeded torch generator on the device"},
        "clocks": clocks, "gpu_launches": ctx.launch_count - l0,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                     "traffic_source": tsrc, "kernel": ctx.last_kernel, "avg_launch_ms": ms / steps,
                     "algorithmic_bytes_per_launch": 16.0 * dof, "peak_source": peak_src}}
    ctx.close()
    return line


CONFIG6 = {"config6_2d2v_128^4": (32, 4), "config6_2d2v_64^4": (16, 4), "config6_2d2v_n8_128^4": (16, 8), "config6_2d2v_n8_64^4": (8, 8)}


def oracle_sample_2d2v(dt):
    """Three SSP-RK3 steps of oracle.vlasov2d2v on a (4, 4, 32, 32)-element slab (4/32 of the x and y elements of the 128^4
    grid, periodic within the slab, full velocity grid): about 10-20 s of host time."""
    from oracle import vlasov2d2v as o4
    import workloads as wl
    L = 2 * math.pi / K_WAVE
    g = o4.make_grid((4, 4, 32, 32), (4,) * 4, (0.0, 0.0, -8.5, -8.5), (L / 8, L / 8, 8.5, 8.5), omega_c=1.0, pmax=(4, 4))
    x, y, u, v = [c.reshape(-1) for c in g.coords]
    f = wl.ring2d_f0(x, y, u, v, K_WAVE, K_WAVE)
    t0 = time.perf_counter()
    for _ in range(3):
        f = o4.ssprk3_step(g, f, dt)
    wall = time.perf_counter() - t0
    return f.size * 9.0 / wall, host_cores(), f"oracle.vlasov2d2v.ssprk3_step (NumPy), (4, 4, 32, 32) x 4^4 slab = {f.size} DOF, 3 steps"


def _ring2d_device(x, y, u, v, seed, amp_noise):
    """The config-6 state built on the device from the same analytic formula as workloads.ring2d_f0 (Eq. 31 ring x wave)
    with seeded torch noise -- for the secondary throughput run, where a 2 GB host array would cost seconds."""
    import torch
    tx, ty, tu, tv = (torch.from_numpy(a).cuda() for a in (x, y, u, v))
    s = (tu * tu)[:, None] + (tv * tv)[None, :]
    s = s / 2.0
    ring = s ** 3 * torch.exp(-s) / (2.0 * math.pi * math.factorial(3))
    wave = 1.0 + 0.01 * torch.sin(K_WAVE * tx)[:, None] + 0.01 * torch.cos(K_WAVE * ty)[None, :]
    f = wave[:, :, None, None] * ring[None, None, :, :]
    g = torch.Generator(device="cuda"); g.manual_seed(seed)
    f += amp_noise * (2.0 * torch.rand(f.shape, dtype=torch.float64, device="cuda", generator=g) - 1.0)
    return f.contiguous()


def run_config6(args, name, host_inputs=True, with_e2e=True):
    """2D2V: N^4 elements x n^4 LGL nodes, ring workload in (v_x, v_y) with a seeded perturbation in x
    and y, one SSP-RK3 step with the 2-D Poisson solve at every stage (dg4_ssprk3_run)."""
    import torch
    import workloads as wl
    from paper_2202_13532_b200 import api
    N, n = CONFIG6[name]
    lo, hi = (0.0, 0.0, -8.5, -8.5), (2 * math.pi / K_WAVE, 2 * math.pi / K_WAVE, 8.5, 8.5)
    ctx = api.DG4Context((N,) * 4, (n,) * 4, lo, hi, bc=(0, 0, 1, 1), omega_c=1.0)
    if args.rhs_kernel:
        ctx.set_option(api.OPT4_RHS_KERNEL, args.rhs_kernel)
    x, y, u, v = (ctx.nodes(d) for d in range(4))
    f0 = None
    if host_inputs:
        f0 = wl.add_uniform_noise(wl.ring2d_f0(x, y, u, v, K_WAVE, K_WAVE), wl.SEED_CFG6_NOISE, 1e-4)
        f = torch.from_numpy(f0).cuda()
    else:
        f = _ring2d_device(x, y, u, v, wl.SEED_CFG6_NOISE, 1e-4)
    dt = 2e-4 if n == 4 else 5e-5
    warm = max(args.warmup, 3)
    ctx.ssprk3_run(f, dt, warm)
    torch.cuda.synchronize()
    steps = args.steps
    ctx.set_option(api.OPT4_PROFILE, profile_stride(steps))
    ctx.get_profile(reset=True)

    def region():
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx.ssprk3_run(f, dt, steps)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    l0 = ctx.launch_count
    ms, clocks = _clocks_during(region)
    launches = ctx.launch_count - l0
    rhs_ms, rhs_n = ctx.get_profile(reset=True)
    ctx.set_option(api.OPT4_PROFILE, 0)
    finite = bool(torch.isfinite(f).all().item())
    dof = (n * N) ** 4
    peak, peak_src = measured_peak_hbm()
    bytes_per_launch = 64.0 / 3.0 * dof
    achieved = bytes_per_launch / (rhs_ms / max(rhs_n, 1) * 1e-3) / 1e9
    traffic, tsrc = ncu_traffic(name, ctx.last_kernel)
    line = {
        "metric": "FP64 phase-space DOF-updates/s per RK stage", "value": dof * 3.0 * steps / (ms * 1e-3), "unit": UNIT,
        "n_gpus": 1, "steps": steps, "warmup": warm, "ms_per_step": ms / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "grid": "x".join([str(n * N)] * 4), "order": n, "dof": dof, "dt": dt, "self_consistent_poisson_each_stage": True,
                   "l2": "arrays (3 x %.2f GB) larger than L2" % (dof * 8 / 1e9), "finite": finite,
                   "inputs": "workloads.py (host)" if host_inputs else "same formula + seeded torch noise, built on the device"},
        "clocks": clocks, "gpu_launches": launches,
        "hbm_gbs_algorithmic_whole_step": 64.0 * dof * steps / (ms * 1e-3) / 1e9,
        "frac_whole_step": 64.0 * dof * steps / (ms * 1e-3) / 1e9 / peak,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                     "traffic_source": tsrc, "kernel": ctx.last_kernel, "avg_launch_ms": rhs_ms / max(rhs_n, 1), "launches_timed": rhs_n,
                     "algorithmic_bytes_per_launch": bytes_per_launch, "peak_source": peak_src,
                     "rhs_share_of_step": 3.0 * (rhs_ms / max(rhs_n, 1)) / (ms / steps),
                     "how": "CUDA events around every k-th RHS launch inside the timed region (DG4_OPT_PROFILE = k)"}}
    if with_e2e and f0 is not None:
        fh = torch.from_numpy(f0).pin_memory()
        ctx.ssprk3_run_host(fh, dt, 1)
        t0 = time.perf_counter()
        e2e_steps = 2
        for _ in range(e2e_steps):
            ctx.ssprk3_run_host(fh, dt, 1)
        e2e_s = time.perf_counter() - t0
        line["e2e"] = {"value": dof * 3.0 * e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": dof * 8, "d2h_bytes_per_step": dof * 8,
                       "steps": e2e_steps, "api": "dg4_ssprk3_run_host (pinned host buffer)"}
    if with_e2e and not args.no_cpu_baseline:
        cv, cc, cd = oracle_sample_2d2v(dt)
        line["cpu_baseline"] = {"value": cv, "unit": UNIT, "cores": cc, "kind": "oracle", "sample": cd}
    ctx.close()
    return line


def run_config_nd(args, name):
    """3D3V through the dimension-generic path (include/dgvlasov_nd.h, dgn_*): 8^6 elements x 2^6 LGL nodes = 16^6 DOF,
    Maxwellian with a 1 % density wave along each space axis + seeded noise, the 3-D Poisson solve at every stage.  The generic
    kernel family (one thread per node): a correctness-shaped path, reported against the HBM roofline for scale only."""
    import torch
    import workloads as wl
    from paper_2202_13532_b200 import api
    N, n = 8, 2
    L = 4 * math.pi
    ctx = api.DGNContext(3, 3, (N,) * 6, (n,) * 6, (0.0,) * 3 + (-6.0,) * 3, (L,) * 3 + (6.0,) * 3, omega_c=0.5, pmax=(4, 4, 4))
    xs = [torch.from_numpy(ctx.nodes(d)).cuda() for d in range(6)]
    shp = lambda d: [-1 if i == d else 1 for i in range(6)]
    wave = 1.0 + 0.01 * sum(torch.cos(0.5 * xs[d]).reshape(shp(d)) for d in range(3))
    maxw = 1.0
    for d in range(3, 6):
        maxw = maxw * (torch.exp(-0.5 * xs[d] ** 2) / math.sqrt(2 * math.pi)).reshape(shp(d))
    f = (wave * maxw).contiguous()
    g = torch.Generator(device="cuda"); g.manual_seed(wl.SEED_CFG6_NOISE + 1)
    f += 1e-6 * (2.0 * torch.rand(f.shape, dtype=torch.float64, device="cuda", generator=g) - 1.0)
    dt = 2e-3
    warm = max(args.warmup, 3)
    ctx.ssprk3_run(f, dt, warm, True)
    torch.cuda.synchronize()
    steps = args.steps

    def region():
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx.ssprk3_run(f, dt, steps, True)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    l0 = ctx.launch_count
    ms, clocks = _clocks_during(region)
    dof = (n * N) ** 6
    peak, peak_src = measured_peak_hbm()
    gbs = 64.0 * dof * steps / (ms * 1e-3) / 1e9
    line = {
        "metric": METRIC, "value": dof * 3.0 * steps / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": steps, "warmup": warm,
        "ms_per_step": ms / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "grid": "x".join([str(n * N)] * 6), "order": n, "dof": dof, "dt": dt, "self_consistent_poisson_each_stage": True,
                   "finite": bool(torch.isfinite(f).all().item()), "inputs": "analytic Maxwellian + waves + seeded torch noise, built on the device",
                   "l2": "arrays (3 x %.2f GB) comparable to the 126 MB L2" % (dof * 8 / 1e9)},
        "clocks": clocks, "gpu_launches": ctx.launch_count - l0,
        "hbm_gbs_algorithmic_whole_step": gbs, "frac_whole_step": gbs / peak,
        "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "traffic": None,
                     "kernel": "rhs_nd_kernel (generic, one thread per node)", "peak_source": peak_src,
                     "how": "whole step (3 RHS launches + 3 three-dimensional field solves) by CUDA events; 64 B per DOF per step"}}
    ctx.close()
    return line


def _cosine_batch_device(x, batch, seed):
    """Config-5 densities 1 + sum_{i<16} A cos(m x + phi) + N(0, 1e-3) built on the device (same distributions as
    workloads.cosine_sum_density, torch's seeded generator) -- throughput runs only."""
    import torch
    g = torch.Generator(device="cuda"); g.manual_seed(seed)
    tx = torch.from_numpy(x).cuda()
    rho = torch.ones((batch, tx.numel()), dtype=torch.float64, device="cuda")
    for _ in range(16):
        A = 0.1 * torch.rand((batch, 1), dtype=torch.float64, device="cuda", generator=g)
        m = torch.randint(1, 1025, (batch, 1), device="cuda", generator=g).to(torch.float64)
        ph = 2 * math.pi * torch.rand((batch, 1), dtype=torch.float64, device="cuda", generator=g)
        rho += A * torch.cos(m * tx[None, :] + ph)
    rho += 1e-3 * torch.randn(rho.shape, dtype=torch.float64, device="cuda", generator=g)
    return rho


def run_config5(args, name, host_inputs=True):
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
    if host_inputs:
        rho_h, _, _, _ = wl.cosine_sum_density(x, batch, wl.SEED_CFG5)
        rho = torch.from_numpy(rho_h).cuda()
    else:
        rho = _cosine_batch_device(x, batch, wl.SEED_CFG5)
    E = torch.empty_like(rho)
    warm = max(args.warmup, 3)
    for _ in range(warm):
        ctx.poisson_E(rho, E)
    torch.cuda.synchronize()
    steps = args.steps

    def region():
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            ctx.poisson_E(rho, E)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    l0 = ctx.launch_count
    ms, clocks = _clocks_during(region)
    G, Q = N * n, 2 * (pmax + 1)
    flops = 2.0 * 2.0 * batch * G * Q            # projection + synthesis, 2 flop per multiply-add
    tf = flops * steps / (ms * 1e-3) / 1e12
    inputs = "workloads.py (host)" if host_inputs else "same distributions, seeded torch generator on the device"
    if fft:
        # same result as the dense contraction (parity-tested against the same oracle); the kernel is bound by reading
        # rho and writing E once: 16 B per x node per vector
        gbs = 2.0 * batch * G * 8 * steps / (ms * 1e-3) / 1e9
        peak, src = measured_peak_hbm()
        traffic, tsrc = ncu_traffic(name, "field_fft_kernel")
        line = {
            "metric": "density vectors/s through projection + Poisson solve (FFT-factorised)", "value": batch * steps / (ms * 1e-3),
            "unit": "vectors/s", "n_gpus": 1, "steps": steps, "warmup": warm, "ms_per_step": ms / steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "x_nodes": G, "batch": batch, "modes": pmax, "dg_create_s": t_create,
                       "l2": "rho and E (2 x %.2f GB) larger than L2" % (batch * G * 8 / 1e9),
                       "dense_equivalent_tflops": tf, "inputs": inputs},
            "clocks": clocks, "gpu_launches": ctx.launch_count - l0,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "traffic": traffic,
                         "traffic_source": tsrc, "kernel": ctx.last_field_kernel, "peak_source": src, "avg_launch_ms": ms / steps,
                         "algorithmic_bytes_per_launch": 2.0 * batch * G * 8}}
        ctx.close()
        return line
    alu_peak = max(api.fp64_peak(0, 0), api.fp64_peak(0, 1))
    line = {
        "metric": "FP64 TFLOP/s of projection + Poisson synthesis (dense contraction)", "value": tf, "unit": "TFLOP/s",
        "n_gpus": 1, "steps": steps, "warmup": warm, "ms_per_step": ms / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "x_nodes": G, "batch": batch, "modes": pmax, "dg_create_s": t_create,
                   "l2": "T and S (2 x %.2f GB) larger than L2" % (G * Q * 8 / 1e9), "inputs": inputs},
        "clocks": clocks, "gpu_launches": ctx.launch_count - l0,
        "roofline": {"bound": "alu", "achieved": tf, "peak": alu_peak, "unit": "TFLOP/s", "frac": tf / alu_peak,
                     "traffic": None, "kernel": ctx.last_field_kernel,
                     "peak_source": "measured in this run by dg_fp64_peak (max of DFMA and DMMA chains); nominal %.1f = 148 SM x 64 FMA/clk x 2 x 1.965 GHz"
                                    % FP64_ALU_PEAK_NOMINAL_TFLOPS}}
    ctx.close()
    return line


def run_fp64_peak(args):
    """Measured FP64 arithmetic peak (DFMA and DMMA register chains) with the clocks seen: the 'alu' roofline denominator."""
    import torch
    from paper_2202_13532_b200 import api
    api.fp64_peak(0, 0, 2000)

    def region():
        return [api.fp64_peak(0, 0, 40000), api.fp64_peak(0, 1, 40000)]

    (dfma, dmma), clocks = _clocks_during(region)
    return {"workload": "fp64_peak", "dfma_tflops": dfma, "dmma_m8n8k4_tflops": dmma, "nominal_tflops": FP64_ALU_PEAK_NOMINAL_TFLOPS,
            "clocks": clocks, "how": "dg_fp64_peak: 148 x 8 CTAs x 256 threads, 16 DFMA / 8 DMMA chains per thread, 40000 iterations"}


def run_secondary(args):
    """Short runs of the other configs (each with its own roofline and clocks) for the driver's record.  Inputs are built
    on the device where the host recipe would cost seconds (noted per entry); the parity tests use the host recipes."""
    import copy
    import torch
    out = []
    a = copy.copy(args)
    a.no_cpu_baseline = True
    a.rhs_kernel = 0
    t_begin = time.perf_counter()

    def add(fn, *fa, **kw):
        if time.perf_counter() - t_begin > args.secondary_budget_s:
            out.append({"skipped": fa[1] if len(fa) > 1 else str(fn.__name__), "reason": "secondary time budget used up"})
            return
        try:
            line = fn(*fa, **kw)
            keep = {k: line[k] for k in ("metric", "value", "unit", "steps", "ms_per_step", "config", "clocks", "roofline", "gpu_launches") if k in line}
            for k in ("hbm_gbs_algorithmic_whole_step", "frac_whole_step"):
                if k in line:
                    keep[k] = line[k]
            out.append(keep)
        except Exception as e:                                    # a failing secondary must not take the headline down
            out.append({"failed": fa[1] if len(fa) > 1 else str(fn.__name__), "error": repr(e)[:300]})
        torch.cuda.empty_cache()

    a.steps, a.warmup = 30, 3
    add(run_config2_short, a, "config2_1d2v_256^3")
    a.steps = 20
    for name in sorted(CONFIG4, key=lambda s: CONFIG4[s][0]):
        add(run_config4, a, name, host_inputs=False)
    a.steps, a.batch, a.field_kernel = 20, 4096, "auto"
    add(run_config5, a, "config5_field", host_inputs=False)
    a.steps, a.batch, a.field_kernel = 2, 4096, "dmma"            # the dense contraction at BASELINE config 5's stated batch
    add(run_config5, a, "config5_field_dense_dmma", host_inputs=False)
    a.steps = 6
    add(run_config6, a, "config6_2d2v_128^4", host_inputs=False, with_e2e=False)
    add(run_config6, a, "config6_2d2v_n8_128^4", host_inputs=False, with_e2e=False)
    a.steps = 5
    add(run_config_nd, a, "config7_3d3v_16^6")
    return out


def run_config2_short(args, name):
    """Config 2 (256^3, dt 1e-3): the same step as the headline on BASELINE.json configs[1]."""
    import torch
    from paper_2202_13532_b200 import api
    w = WORKLOADS[name]
    ctx = api.DGContext(device=0, **grid_args(w))
    f0 = make_f0(ctx.nodes(0), ctx.nodes(1), ctx.nodes(2), w)
    dof, dt = f0.size, w["dt"]
    f = torch.from_numpy(f0).cuda()
    ctx.ssprk3_run(f, dt, max(args.warmup, 3), True)
    torch.cuda.synchronize()
    peak, peak_src = measured_peak_hbm()

    def region():
        return timed_run(ctx, f, dt, args.steps, None, torch.cuda.synchronize, lambda v: v, api)

    (ms, ms4, n4, launches, _), clocks = _clocks_during(region)
    line = {"metric": METRIC, "value": dof * 3.0 * args.steps / (ms * 1e-3), "unit": UNIT, "steps": args.steps, "ms_per_step": ms / args.steps,
            "config": {"workload": name, "dof": dof, "dt": dt, "l2": "3 x %.0f MB: comparable to the 126 MB L2 (stage arrays partly L2-resident)" % (dof * 8 / 1e6),
                       "finite": int(ctx.check_finite(f).item()) == 0},
            "clocks": clocks, "gpu_launches": launches,
            "roofline": stage_roofline(ctx.last_kernel, dof, ms4, n4, peak, peak_src, name, ms / args.steps),
            "hbm_gbs_algorithmic_whole_step": 64.0 * dof * args.steps / (ms * 1e-3) / 1e9,
            "frac_whole_step": 64.0 * dof * args.steps / (ms * 1e-3) / 1e9 / peak}
    ctx.close()
    return line


# -----------------------------------------------------------------------------------------------
# launch
# -----------------------------------------------------------------------------------------------
def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def spawn_ranks(args):
    """--gpus N > 1 outside torchrun: start the N ranks (one process per GPU) and pass their output through."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config3_1d2v_512^3",
                    choices=sorted(WORKLOADS) + sorted(CONFIG4) + ["config5_field", "fp64_peak", "oracle_timing", "config7_3d3v_16^6"] + sorted(CONFIG6))
    ap.add_argument("--batch", type=int, default=4096, help="config5_field only")
    ap.add_argument("--field-kernel", default="auto", choices=["auto", "dmma", "dfma", "fft"], help="config5_field only")
    ap.add_argument("--parallelism", default="auto", choices=["auto", "replicas", "xslab", "xslab-push"],
                    help="auto: one GPU runs the workload; N > 1 runs ONE problem N times as long in x, sharded by x-slabs with the "
                         "face planes exchanged by send/recv (xslab).  replicas: N independent copies (no data-path collective). "
                         "xslab-push: the faces are stored by the RHS kernel into peer memory (unverified on two devices)")
    ap.add_argument("--rhs-kernel", type=int, default=0, help="config6 only: DG4_OPT_RHS_KERNEL (0 auto)")
    ap.add_argument("--sustained-steps", type=int, default=1000, help="config 3: steps of the sustained region (0 = skip)")
    ap.add_argument("--no-secondary", action="store_true", help="skip the short runs of configs 2, 4, 5, 6")
    ap.add_argument("--secondary-budget-s", type=float, default=75.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--full", action="store_true", help="oracle_timing: also the single-threaded 512^3 step")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(args))
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.workload == "oracle_timing":
        return run_oracle_timing(args)
    if args.workload == "fp64_peak":
        return print(json.dumps(run_fp64_peak(args)), flush=True)
    if args.workload in CONFIG4:
        return print(json.dumps(run_config4(args, args.workload)), flush=True)
    if args.workload == "config5_field":
        return print(json.dumps(run_config5(args, args.workload)), flush=True)
    if args.workload in CONFIG6:
        return print(json.dumps(run_config6(args, args.workload)), flush=True)
    if args.workload == "config7_3d3v_16^6":
        return print(json.dumps(run_config_nd(args, args.workload)), flush=True)
    w = WORKLOADS[args.workload]
    if args.workload != "config3_1d2v_512^3":
        args.sustained_steps = 0 if args.sustained_steps == 1000 else args.sustained_steps
    if args.impl == "reference":
        run_reference(args, w, args.workload)
    else:
        run_ours(args, w, args.workload)


if __name__ == "__main__":
    main()
