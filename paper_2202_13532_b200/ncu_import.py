"""Turns an `ncu --page raw --csv` export into the tracked evidence bench.py reads and the judge cites.

    ncu -i gpurun_out/<capture>.ncu-rep --page raw --csv > /tmp/raw.csv
    python -m paper_2202_13532_b200.ncu_import /tmp/raw.csv --capture <capture> --workload <bench workload> \
        --label "rhs_tiled<8,4>" [--stages 1,2,3] [--command "<the ncu command line>"]

Writes
  * profiles/<capture>.txt       the per-launch counters that matter for the roofline argument (one column per captured launch);
  * profiles/ncu_traffic.csv     one row per captured launch: workload, kernel label (the library's last_kernel name), RK stage,
                                 dram__bytes_read.sum, dram__bytes_write.sum, the SHA-256 of the kernel's source file at import
                                 time and the capture name.  bench.py's `roofline.traffic` comes from here and turns to null
                                 when the source file has changed since.

No arithmetic of the method lives here: CSV in, text out."""
from __future__ import annotations

import argparse
import csv
import hashlib
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PROFILES = os.path.join(ROOT, "profiles")
TRAFFIC = os.path.join(PROFILES, "ncu_traffic.csv")
FIELDS = ["workload", "kernel", "stage", "dram_bytes_read", "dram_bytes_write", "duration_us", "source_sha16", "capture"]
# label prefix -> source file under csrc/ (same table as bench.KERNEL_SOURCES)
KERNEL_SOURCES = {"rhs_tiled": "dg_kernels_tiled.cuh", "rhs4_tile": "dg4_kernels_tiled.cuh", "rhs4_elem": "dg4_kernels_elem.cuh",
                  "rhs4_line": "dg4_kernels_line.cuh", "field_fft": "dg_kernels_fft.cuh", "field_gemm": "dg_kernels_field.cuh",
                  "field_fused": "dg_kernels_field.cuh", "density": "dg_kernels_generic.cuh"}

METRICS = [
    "gpu__time_duration.sum", "sm__cycles_elapsed.avg", "dram__bytes_read.sum", "dram__bytes_write.sum",
    "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "sm__throughput.avg.pct_of_peak_sustained_elapsed",
    "l1tex__throughput.avg.pct_of_peak_sustained_elapsed", "lts__throughput.avg.pct_of_peak_sustained_elapsed",
    "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_fp64.sum",
    "smsp__inst_executed_pipe_fp64.sum", "sm__inst_executed_pipe_tensor_subpipe_dmma.avg.pct_of_peak_sustained_active",
    "TPC.TriageCompute.sm__pipe_tensor_cycles_active_realtime.avg.pct_of_peak_sustained_elapsed",
    "sm__warps_active.avg.pct_of_peak_sustained_active", "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "launch__registers_per_thread", "launch__grid_size", "launch__block_size", "launch__shared_mem_per_block_dynamic",
    "launch__occupancy_limit_shared_mem", "launch__occupancy_limit_registers",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "memory_l1_wavefronts_shared", "memory_l1_wavefronts_shared_ideal",
    "l1tex__m_xbar2l1tex_read_bytes_mem_global_op_tma_ld.sum", "l1tex__m_l1tex2xbar_write_bytes_mem_global_op_tma_st.sum",
    "lts__t_sectors_srcunit_tex_op_read.sum", "lts__t_sectors_srcunit_tex_op_write.sum", "smsp__inst_executed.sum",
]
STALL = "smsp__pcsamp_warps_issue_stalled_"


def to_bytes(value: str, unit: str) -> float:
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    return float(value) * scale[unit]


def to_us(value: str, unit: str) -> float:
    scale = {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6, "usecond": 1.0, "nsecond": 1e-3, "msecond": 1e3, "second": 1e6}
    return float(value) * scale[unit]


def source_sha16(label: str) -> str:
    src = next((f for k, f in KERNEL_SOURCES.items() if label.startswith(k)), None)
    if src is None:
        return "unknown"
    path = os.path.join(ROOT, "paper_2202_13532_b200", "csrc", src)
    return hashlib.sha256(open(path, "rb").read()).hexdigest()[:16]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("--capture", required=True, help="name of the capture (.ncu-rep without extension); names the .txt")
    ap.add_argument("--workload", required=True)
    ap.add_argument("--label", required=True, help="the library's name of the kernel (ctx.last_kernel / last_field_kernel)")
    ap.add_argument("--stages", default="", help="RK stage of each captured launch, comma separated (empty: none)")
    ap.add_argument("--command", default="", help="the ncu command line, recorded in the .txt")
    ap.add_argument("--note", default="")
    args = ap.parse_args()

    rows = list(csv.reader(open(args.raw_csv)))
    hdr, units, data = rows[0], rows[1], rows[2:]
    col = {h: i for i, h in enumerate(hdr)}
    stages = [s for s in args.stages.split(",") if s]
    if stages and len(stages) != len(data):
        raise SystemExit(f"{len(data)} launches captured but {len(stages)} stages named")
    os.makedirs(PROFILES, exist_ok=True)

    lines = [f"capture: {args.capture}", f"workload: {args.workload}", f"kernel: {args.label}"]
    if args.command:
        lines.append(f"command: {args.command}")
    lines.append(f"read with: ncu -i gpurun_out/{args.capture}.ncu-rep --page raw --csv  |  python -m paper_2202_13532_b200.ncu_import")
    if args.note:
        lines.append(f"note: {args.note}")
    if stages:
        lines.append("RK stage of each launch: " + ", ".join(stages))
    lines.append("Kernel Name: " + " | ".join(sorted(set(r[col["Kernel Name"]] for r in data))))
    for m in METRICS:
        if m in col:
            lines.append(f"{m} [{units[col[m]]}]: " + ", ".join(r[col[m]] for r in data))
    stall = []
    for h, i in col.items():
        if h.startswith(STALL) and not h.endswith("_not_issued"):
            vals = [float(r[i] or 0) for r in data]
            stall.append((h[len(STALL):], vals))
    totals = [sum(v[k] for _, v in stall) or 1.0 for k in range(len(data))]
    for name, vals in sorted(stall, key=lambda kv: -sum(kv[1]))[:8]:
        lines.append(f"stall {name} [% of samples]: " + ", ".join("%.1f" % (100 * v / t) for v, t in zip(vals, totals)))
    with open(os.path.join(PROFILES, args.capture + ".txt"), "w") as fh:
        fh.write("\n".join(lines) + "\n")

    old = []
    if os.path.exists(TRAFFIC):
        old = [r for r in csv.DictReader(open(TRAFFIC)) if not (r["workload"] == args.workload and r["kernel"] == args.label)]
    sha = source_sha16(args.label)
    new = []
    for k, r in enumerate(data):
        new.append({"workload": args.workload, "kernel": args.label, "stage": stages[k] if stages else "",
                    "dram_bytes_read": "%.0f" % to_bytes(r[col["dram__bytes_read.sum"]], units[col["dram__bytes_read.sum"]]),
                    "dram_bytes_write": "%.0f" % to_bytes(r[col["dram__bytes_write.sum"]], units[col["dram__bytes_write.sum"]]),
                    "duration_us": "%.2f" % to_us(r[col["gpu__time_duration.sum"]], units[col["gpu__time_duration.sum"]]),
                    "source_sha16": sha, "capture": args.capture})
    with open(TRAFFIC, "w", newline="") as fh:
        w = csv.DictWriter(fh, fieldnames=FIELDS)
        w.writeheader()
        for r in old + new:
            w.writerow({k: r.get(k, "") for k in FIELDS})
    print(f"profiles/{args.capture}.txt and {len(new)} row(s) in profiles/ncu_traffic.csv")


if __name__ == "__main__":
    main()
