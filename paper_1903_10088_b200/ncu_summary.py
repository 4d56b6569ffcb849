"""Summarise an ncu capture of the two hot kernels (diagnostics, not part of the method).

    ncu -i gpurun_out/prof.ncu-rep --page raw --csv > raw.csv
    python -m paper_1903_10088_b200.ncu_summary raw.csv profiles/r2_ncu_config3 --command "<the ncu command>" [--note "..."]

writes `<out>.md` (a table of the counters the roofline discussion uses, with the command that made the capture) and
`<out>_counts.csv` (per kernel: instructions, L1 wavefronts, L2 sectors, DRAM bytes per launch), which `bench.py` reads
to turn its live kernel times into issue / L1 / L2 / DRAM fractions.  Everything here is text processing of ncu's own
export; nothing is measured by this script.
"""
from __future__ import annotations

import argparse
import csv

ROWS = [
    ("launch__grid_size", "grid"),
    ("launch__block_size", "block"),
    ("launch__registers_per_thread", "registers/thread"),
    ("gpu__time_duration.sum", "duration (cold cache, serialised)"),
    ("sm__cycles_elapsed.max", "SM cycles elapsed"),
    ("smsp__cycles_active.avg", "SMSP cycles active"),
    ("smsp__inst_executed.sum", "warp instructions executed"),
    ("smsp__issue_active.avg.pct_of_peak_sustained_active", "issue slots used while active"),
    ("sm__warps_active.avg.pct_of_peak_sustained_active", "warps active (of 64 per SM)"),
    ("sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active", "FMA pipe"),
    ("sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", "ALU pipe"),
    ("sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active", "LSU pipe"),
    ("SM_A.TriageCompute.l1tex__data_pipe_lsu_wavefronts.avg", "L1 data-pipe wavefronts per SM"),
    ("SM_A.TriageCompute.l1tex__data_pipe_lsu_wavefronts_mem_shared.avg", "... of which shared memory"),
    ("l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "shared-memory bank conflicts (wavefronts, all SMs)"),
    ("l1tex__t_sector_hit_rate.pct", "L1 sector hit rate"),
    ("l1tex__throughput.avg.pct_of_peak_sustained_elapsed", "L1 throughput (of elapsed)"),
    ("lts__t_sectors.sum", "L2 sectors (32 B)"),
    ("lts__t_sector_hit_rate.pct", "L2 sector hit rate"),
    ("lts__throughput.avg.pct_of_peak_sustained_elapsed", "L2 throughput (of elapsed)"),
    ("dram__bytes_read.sum", "DRAM read"),
    ("dram__bytes_write.sum", "DRAM written"),
]
STALLS = ["long_scoreboard", "short_scoreboard", "barrier", "wait", "math_pipe_throttle", "mio_throttle", "lg_throttle",
          "not_selected", "no_instruction", "dispatch_stall", "branch_resolving", "drain"]
UNIT_SCALE = {"Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "byte": 1.0}


def short_name(full: str) -> str:
    n = full.replace("void ", "").replace("osiv::", "")
    return n.split("(")[0]


def launch_list(args):
    """`ncu --metrics gpu__time_duration.sum --csv --log-file launches.csv` -> per-kernel launches, mean time and share"""
    rows = [r for r in csv.reader(l for l in open(args.raw_csv) if l.startswith('"'))]
    hdr = rows[0]
    col = {h: i for i, h in enumerate(hdr)}
    agg = {}
    for r in rows[1:]:
        if r[col["Metric Name"]] != "gpu__time_duration.sum":
            continue
        key = (short_name(r[col["Kernel Name"]]), r[col["Block Size"]], r[col["Grid Size"]])
        agg.setdefault(key, []).append(float(r[col["Metric Value"]]))
    total = sum(sum(v) for v in agg.values())
    with open(args.out_prefix + ".md", "w") as f:
        f.write(f"# {args.out_prefix.split('/')[-1]}: ncu launch list\n\nCommand (after the same command exited 0 without ncu):\n\n    {args.command}\n\n")
        f.write("Per-launch times under ncu are cold-cache and serialised; compare shares, not absolutes.\n\n")
        if args.note:
            f.write(args.note + "\n\n")
        f.write("| kernel | block | grid | launches | mean ns | min ns | max ns | share |\n|---|---|---|---|---|---|---|---|\n")
        for (n, b, g), v in sorted(agg.items(), key=lambda kv: -sum(kv[1])):
            f.write(f"| `{n}` | {b} | {g} | {len(v)} | {sum(v) / len(v):.0f} | {min(v):.0f} | {max(v):.0f} | {100 * sum(v) / total:.1f} % |\n")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("out_prefix")
    ap.add_argument("--command", required=True)
    ap.add_argument("--note", default="")
    ap.add_argument("--launches", action="store_true", help="raw_csv is a launch list (gpu__time_duration.sum per launch)")
    args = ap.parse_args()
    if args.launches:
        return launch_list(args)
    rows = list(csv.reader(open(args.raw_csv)))
    hdr, units, data = rows[0], rows[1], rows[2:]
    col = {h: i for i, h in enumerate(hdr)}
    names = [short_name(r[col["Kernel Name"]]) for r in data]

    def cell(r, key):
        if key not in col:
            return "n/a"
        v, u = r[col[key]], units[col[key]]
        try:
            f = float(v)
            v = f"{f:.0f}" if abs(f) >= 1000 or f == int(f) else f"{f:.2f}"
        except ValueError:
            pass
        return f"{v} {u}".strip()

    with open(args.out_prefix + ".md", "w") as f:
        f.write(f"# {args.out_prefix.split('/')[-1]}: ncu full-set capture\n\n")
        f.write("Command (after the same command exited 0 without ncu):\n\n    " + args.command + "\n\n")
        f.write("Read here with `ncu -i <rep> --page raw --csv` and summarised by `python -m paper_1903_10088_b200.ncu_summary`. "
                "Under ncu every launch is serialised and starts with cold caches: the programmatic-dependent-launch overlap "
                "of the timed region is absent, so durations are stand-alone figures.\n\n")
        if args.note:
            f.write(args.note + "\n\n")
        f.write("| metric | " + " | ".join(names) + " |\n|---|" + "---|" * len(names) + "\n")
        for key, label in ROWS:
            f.write(f"| {label} (`{key.split('.')[-2] if key.startswith('SM_A') else key.split('.')[0]}`) | " + " | ".join(cell(r, key) for r in data) + " |\n")
        for st in STALLS:
            key = f"smsp__average_warps_issue_stalled_{st}_per_issue_active.ratio"
            f.write(f"| stall per issue: {st} | " + " | ".join(cell(r, key) for r in data) + " |\n")

    with open(args.out_prefix + "_counts.csv", "w") as f:
        f.write("kernel,warp_instructions,l1_wavefronts_per_sm,l1_wavefronts_shared_per_sm,l2_sectors,dram_bytes,duration_us,block,grid\n")
        for r, n in zip(data, names):
            def num(key, scale=False):
                if key not in col or r[col[key]] == "":
                    return 0.0
                v = float(r[col[key]])
                return v * UNIT_SCALE.get(units[col[key]], 1.0) if scale else v
            dram = num("dram__bytes_read.sum", True) + num("dram__bytes_write.sum", True)
            dur = num("gpu__time_duration.sum") * {"us": 1.0, "ns": 1e-3, "ms": 1e3}.get(units[col["gpu__time_duration.sum"]], 1.0)
            f.write(f"\"{n}\",{num('smsp__inst_executed.sum'):.0f},{num('SM_A.TriageCompute.l1tex__data_pipe_lsu_wavefronts.avg'):.1f},"
                    f"{num('SM_A.TriageCompute.l1tex__data_pipe_lsu_wavefronts_mem_shared.avg'):.1f},{num('lts__t_sectors.sum'):.0f},"
                    f"{dram:.0f},{dur:.3f},{num('launch__block_size'):.0f},{num('launch__grid_size'):.0f}\n")


if __name__ == "__main__":
    main()
