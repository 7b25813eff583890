"""Summarise an `ncu --set full` capture of k_wilson and record its DRAM traffic for bench.py.

    python bench.py --ncu-summary REPORT.ncu-rep --key cfg3_paper_scale/f32 [--sha SHA16] [--md OUT.md]

(a mode of bench.py, which owns profiles/ncu_traffic.json; this module sits beside it and is not part of the library).

Reads the report with `ncu -i REPORT --page raw --csv` (no GPU needed), prints a markdown table of the
counters DESIGN.md section 5 argues from (pipe utilisation, issue rate, stall reasons, registers, DRAM bytes) for
every k_wilson launch in it, and stores dram__bytes_read.sum / dram__bytes_write.sum of the first one under
`--key` in profiles/ncu_traffic.json together with the hash of the kernel sources the capture was taken on
(`--sha`: what `python bench.py --source-sha` printed on the GPU box at capture time; default: the sources as
they are now).  bench.py reports `roofline.traffic` only when that hash matches the sources it runs.
"""
import argparse
import csv
import io
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))

METRICS = [
    ("gpu__time_duration.sum", "kernel time"),
    ("sm__cycles_elapsed.avg.per_second", "SM clock"),
    ("launch__grid_size", "CTAs"),
    ("launch__block_size", "threads per CTA"),
    ("launch__registers_per_thread", "registers per thread"),
    ("launch__shared_mem_per_block_dynamic", "dynamic shared memory per CTA"),
    ("launch__occupancy_limit_registers", "CTAs/SM allowed by registers"),
    ("launch__occupancy_limit_shared_mem", "CTAs/SM allowed by shared memory"),
    ("sm__warps_active.avg.pct_of_peak_sustained_active", "warps active"),
    ("smsp__inst_executed.sum", "warp instructions"),
    ("smsp__issue_active.avg.pct_of_peak_sustained_active", "issue slots busy"),
    ("sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active", "XU (special-function) pipe"),
    ("sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active", "FMA pipe cycles active"),
    ("sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active", "FMA pipe instructions"),
    ("sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", "ALU pipe"),
    ("sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active", "FP64 pipe cycles active"),
    ("sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active", "LSU pipe"),
    ("dram__bytes_read.sum", "DRAM read"),
    ("dram__bytes_write.sum", "DRAM written"),
    ("gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "DRAM throughput"),
    ("sass__inst_executed_local_loads", "local-memory (spill) loads"),
    ("sass__inst_executed_local_stores", "local-memory (spill) stores"),
    ("l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "shared-memory bank conflicts"),
    # executed lane-ops in ncu's own words (thread-level, predicated-off lanes not counted)
    ("smsp__sass_thread_inst_executed_op_fp32_pred_on.sum", "FP32 thread instructions (FADD + FMUL + FFMA; a packed instruction counts once per half)"),
    ("smsp__sass_thread_inst_executed_op_ffma_pred_on.sum", "... of which FFMA"),
    ("smsp__sass_thread_inst_executed_op_fmul_pred_on.sum", "... of which FMUL"),
    ("smsp__sass_thread_inst_executed_op_fadd_pred_on.sum", "... of which FADD"),
    ("smsp__sass_thread_inst_executed_op_fp64_pred_on.sum", "FP64 thread instructions"),
    ("sm__inst_executed_pipe_xu.sum", "XU-pipe warp instructions"),
    ("sm__inst_executed_pipe_fma.sum", "FMA-pipe warp instructions"),
    ("smsp__thread_inst_executed.sum", "thread instructions, all kinds"),
]

# Derived: executed FP32 flops-style lane-ops per second (FFMA counted once, as one lane-op) against the issue peak
PEAK_LANES_PER_CLK = 148 * 128
STALL = "smsp__average_warps_issue_stalled_"


def to_bytes(value, unit):
    scale = {"byte": 1, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}.get(unit, 1)
    return int(round(float(value.replace(",", "")) * scale))


def to_seconds(value, unit):
    scale = {"s": 1.0, "ms": 1e-3, "us": 1e-6, "ns": 1e-9, "second": 1.0, "msecond": 1e-3, "usecond": 1e-6, "nsecond": 1e-9}[unit]
    return float(value.replace(",", "")) * scale


def to_hz(value, unit):
    scale = {"hz": 1.0, "Khz": 1e3, "Mhz": 1e6, "Ghz": 1e9}[unit]
    return float(value.replace(",", "")) * scale


def read_report(path):
    out = subprocess.run(["ncu", "-i", path, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    header, units = rows[0], rows[1]
    return header, units, rows[2:]


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("report")
    ap.add_argument("--key", default=None, help="entry of profiles/ncu_traffic.json to write, e.g. cfg3_paper_scale/f32")
    ap.add_argument("--sha", default=None, help="source hash at capture time (bench.py --source-sha on the GPU box)")
    ap.add_argument("--md", default=None, help="also append the table to this file")
    ap.add_argument("--kernel", default="k_wilson")
    args = ap.parse_args(argv)

    header, units, rows = read_report(args.report)
    col = {h: i for i, h in enumerate(header)}
    name_col = col.get("Kernel Name", col.get("Name"))
    rows = [r for r in rows if args.kernel in r[name_col]]
    if not rows:
        raise SystemExit("no %s launch in %s" % (args.kernel, args.report))
    lines = []
    for r in rows:
        lines.append("Kernel: `%s`" % r[name_col])
        lines.append("")
        lines.append("| counter | value | what |")
        lines.append("|---|---|---|")
        for m, what in METRICS:
            if m in col:
                lines.append("| `%s` | %s %s | %s |" % (m, r[col[m]], units[col[m]], what))
        stalls = []
        for h, i in col.items():
            if h.startswith(STALL) and h.endswith("_per_issue_active.ratio"):
                try:
                    v = float(r[i])
                except ValueError:
                    continue
                if v >= 0.1 and "selected" not in h[len(STALL):].replace("not_selected", ""):
                    stalls.append((v, h[len(STALL):-len("_per_issue_active.ratio")]))
        try:                                             # executed lane-op rates, beside the algorithmic count of bench.py
            secs = to_seconds(r[col["gpu__time_duration.sum"]], units[col["gpu__time_duration.sum"]])
            hz = to_hz(r[col["sm__cycles_elapsed.avg.per_second"]], units[col["sm__cycles_elapsed.avg.per_second"]])
            num = lambda m: float(r[col[m]].replace(",", ""))
            fp32 = num("smsp__sass_thread_inst_executed_op_fp32_pred_on.sum")
            xu = num("sm__inst_executed_pipe_xu.sum") * 32.0
            allt = num("smsp__thread_inst_executed.sum")
            peak = PEAK_LANES_PER_CLK * hz
            lines.append("")
            lines.append("Executed lane-ops per second over the issue peak (148 SMs x 128 lanes x %.3f GHz = %.2f Tlane-op/s): "
                         "FP32 arithmetic %.3f, + XU-pipe lanes %.3f, all thread instructions %.3f."
                         % (hz / 1e9, peak / 1e12, fp32 / secs / peak, (fp32 + xu) / secs / peak, allt / secs / peak))
        except (KeyError, ValueError):
            pass
        stalls.sort(reverse=True)
        lines.append("")
        lines.append("Warp stalls per issue-active cycle: " + ", ".join("`%s` %.2f" % (n, v) for v, n in stalls))
        lines.append("")
    text = "\n".join(lines)
    print(text)
    if args.md:
        with open(args.md, "a") as fh:
            fh.write(text + "\n")
    if args.key:
        sys.path.insert(0, ROOT)
        import bench
        r = rows[0]
        path = os.path.join(ROOT, "profiles", "ncu_traffic.json")
        try:
            with open(path) as fh:
                tab = json.load(fh)
        except (OSError, ValueError):
            tab = {"what": "dram__bytes_read.sum / dram__bytes_write.sum of one k_wilson launch per (workload/compute[/options]) "
                           "from ncu --set full captures; written by python bench.py --ncu-summary", "entries": {}}
        i_r, i_w = col["dram__bytes_read.sum"], col["dram__bytes_write.sum"]
        tab["entries"][args.key] = {
            "dram_bytes_read": to_bytes(r[i_r], units[i_r]), "dram_bytes_write": to_bytes(r[i_w], units[i_w]),
            "kernel": r[name_col], "report": os.path.basename(args.report),
            "source_sha16": args.sha or bench.source_sha16(),
        }
        with open(path, "w") as fh:
            json.dump(tab, fh, indent=1, sort_keys=True)
            fh.write("\n")
    return 0


if __name__ == "__main__":
    sys.exit(main())
