#!/usr/bin/env python
"""bench_ncu_summary.py -- turns an Nsight Compute report (.ncu-rep, captured on the B200 under gpurun) into the text
summaries committed under profiles/ (the files bench.py parses at run time for `roofline.traffic` / `roofline.ncu`).

    python bench_ncu_summary.py raw REPORT.ncu-rep --region-steps N --title "..." --command "..."   > profiles/NAME_ncu.txt
    python bench_ncu_summary.py src REPORT.ncu-rep --warps W --steps S --title "..." --command "..." > profiles/NAME_hotspots.md

raw : `ncu -i REPORT --page raw --csv`, first kernel of the report: launch geometry, time, pipe utilisation, memory
      traffic and the per-issue stall ratios, one `metric value unit` line each, behind a header that states the command
      and the workload of the captured launch ("= N region-steps", which bench.py divides the DRAM bytes by).
src : `ncu -i REPORT --page source --csv`: executed warp instructions per region-step by opcode, warp-stall sample shares
      and the single instructions with the most samples.  W = warps of the launch, S = Euler steps of the launch.
Needs `ncu` on PATH (reading a report needs no GPU)."""
import argparse
import collections
import csv
import io
import re
import subprocess

RAW_KEYS = [
    "launch__grid_size", "launch__block_size", "launch__cluster_dim_x", "launch__registers_per_thread",
    "launch__shared_mem_per_block_dynamic", "gpu__time_duration.sum", "sm__cycles_elapsed.avg", "sm__cycles_active.avg",
    "smsp__inst_executed.sum", "smsp__thread_inst_executed_per_inst_executed.ratio",
    "smsp__issue_active.avg.pct_of_peak_sustained_active", "smsp__warps_eligible.avg.per_cycle_active",
    "sm__warps_active.avg.pct_of_peak_sustained_active", "sm__throughput.avg.pct_of_peak_sustained_elapsed",
    "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active", "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_elapsed", "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_uniform.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_tc.avg.pct_of_peak_sustained_active",
    "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active",
    "dram__bytes_read.sum", "dram__bytes_write.sum", "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed",
    "lts__t_sectors.sum", "lts__t_sector_hit_rate.pct", "lts__throughput.avg.pct_of_peak_sustained_elapsed",
    "l1tex__m_xbar2l1tex_read_bytes.sum", "l1tex__m_xbar2l1tex_read_bytes.sum.per_second", "l1tex__t_sector_hit_rate.pct",
    "l1tex__throughput.avg.pct_of_peak_sustained_elapsed", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "sass__inst_executed_local_loads", "sass__inst_executed_local_stores",
]
STALLS = ["barrier", "branch_resolving", "dispatch_stall", "drain", "lg_throttle", "long_scoreboard", "math_pipe_throttle", "membar",
          "mio_throttle", "misc", "no_instruction", "not_selected", "selected", "short_scoreboard", "sleeping", "tex_throttle", "wait"]


def ncu_csv(report, page):
    out = subprocess.run(["ncu", "-i", report, "--page", page, "--csv"], capture_output=True, text=True, check=True).stdout
    return list(csv.reader(io.StringIO(out)))


def header(args, extra):
    print(args.title)
    print()
    print("Command (under gpurun, one B200, after the same command had exited 0 without ncu):")
    print("  " + args.command)
    print(extra)
    print()


def do_raw(args):
    rows = ncu_csv(args.report, "raw")
    names, units, vals = rows[0], rows[1], rows[2 + args.kernel_index]
    col = {n: i for i, n in enumerate(names)}
    header(args, f"Extracted with: python bench_ncu_summary.py raw {args.report} ...  (ncu -i ... --page raw --csv)\n"
                 f"Workload of the captured launch = {args.region_steps:.6e} region-steps "
                 f"(DRAM bytes per region-step = (dram__bytes_read.sum + dram__bytes_write.sum) / that).")
    print(f"{'Kernel Name':<96s}{vals[col['Kernel Name']]}")
    keys = RAW_KEYS + [f"smsp__average_warps_issue_stalled_{s}_per_issue_active.ratio" for s in STALLS]
    for k in keys:
        if k in col:
            print(f"{k:<96s}{vals[col[k]]:>20s} {units[col[k]]}")


def do_src(args):
    rows = ncu_csv(args.report, "source")
    hi = [i for i, r in enumerate(rows) if "Source" in r][0]
    hdr, data = rows[hi], rows[hi + 1:]
    ix = {h: i for i, h in enumerate(hdr)}

    def f(r, k):
        try:
            return float(r[ix[k]])
        except (ValueError, KeyError, IndexError):
            return 0.0

    unit = float(args.warps) * float(args.steps)
    tot_i = sum(f(r, "Instructions Executed") for r in data)
    tot_s = sum(f(r, "# Samples") for r in data)
    header(args, f"Read with `ncu -i {args.report} --page source --csv` and summed by bench_ncu_summary.py src.  "
                 f"Captured launch: {rows[0][1] if len(rows[0]) > 1 else ''}; {args.warps} warps x {args.steps} Euler steps.  "
                 f'"per step" = warp instructions executed per warp per Euler step (= thread instructions per region-step; '
                 f"chunk-level work included pro rata).  Numbers under a profiler are for attribution only, never bench values.")
    print(f"Totals: {tot_i:.4g} warp instructions, {int(tot_s)} stall samples, **{tot_i / unit:.0f} instructions per region-step**.\n")
    ops, samp = collections.Counter(), collections.Counter()
    for r in data:
        m = re.match(r"(@!?U?P\d+\s+)?([A-Z0-9_]+)", r[ix["Source"]].strip())
        op = m.group(2) if m else r[ix["Source"]].strip()[:10]
        ops[op] += f(r, "Instructions Executed"); samp[op] += f(r, "# Samples")
    print("## Executed instruction mix (top opcodes)\n\n| opcode | % of executed | % of stall samples | per step |\n|---|---:|---:|---:|")
    for op, c in ops.most_common(28):
        print(f"| {op} | {100 * c / tot_i:.2f} | {100 * samp[op] / max(tot_s, 1):.2f} | {c / unit:.2f} |")
    print("\n## Stall reasons (share of all warp samples)\n\n| reason | % |\n|---|---:|")
    for k in [h for h in hdr if h.startswith("stall_") and "Not Issued" not in h]:
        v = sum(f(r, k) for r in data)
        if v / max(tot_s, 1) > 0.004:
            print(f"| {k} | {100 * v / tot_s:.1f} |")
    print("\n## Single instructions with the most samples\n\n| SASS | samples | executed per step | dominant stall |\n|---|---:|---:|---|")
    stall_cols = [h for h in hdr if h.startswith("stall_") and "Not Issued" not in h]
    for i in sorted(range(len(data)), key=lambda i: -f(data[i], "# Samples"))[:14]:
        r = data[i]
        dom = max(stall_cols, key=lambda k: f(r, k))
        print(f"| `{r[ix['Source']].strip()[:80]}` | {int(f(r, '# Samples'))} | {f(r, 'Instructions Executed') / unit:.2f} | {dom[6:]} |")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("mode", choices=["raw", "src"])
    ap.add_argument("report")
    ap.add_argument("--title", default="ncu capture")
    ap.add_argument("--command", default="(not recorded)")
    ap.add_argument("--region-steps", type=float, default=0.0)
    ap.add_argument("--kernel-index", type=int, default=0)
    ap.add_argument("--warps", type=float, default=1.0)
    ap.add_argument("--steps", type=float, default=1.0)
    args = ap.parse_args()
    (do_raw if args.mode == "raw" else do_src)(args)


if __name__ == "__main__":
    main()
