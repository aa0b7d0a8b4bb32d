"""Summarise an Nsight Compute report of the hot kernels into the text files kept under profiles/.

    python -m paper_2006_07964_b200.profile_summary REPORT.ncu-rep --workload sweep256 --out profiles/r2 [--command "..."]
    python -m paper_2006_07964_b200.profile_summary --launches LAUNCHES.csv --out profiles/r2_launches.md [--command "..."]

Reads the report with `ncu -i REPORT --page raw --csv` (no GPU needed) and writes
  <out>_traffic.json    {workload: {kernel class: dram__bytes_read.sum + dram__bytes_write.sum per launch, bytes}}
                        (merged into an existing file; bench.py reports these as `roofline*.traffic`)
  <out>_hot_kernels.md  one column per kernel: duration, registers, DRAM bytes, pipe utilisation, stall reasons.
Kernel classes are the names of cfd_profile_name(): inviscid_xi / inviscid_eta / inviscid_zeta / visc_flux / ghost_fill.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import re
import subprocess
import sys

METRICS = [
    ("gpu__time_duration.sum", "duration"),
    ("launch__registers_per_thread", "registers / thread"),
    ("launch__grid_size", "grid"),
    ("launch__block_size", "block"),
    ("sm__warps_active.avg.pct_of_peak_sustained_active", "achieved occupancy"),
    ("dram__bytes_read.sum", "DRAM read"),
    ("dram__bytes_write.sum", "DRAM written"),
    ("gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "DRAM throughput"),
    ("sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active", "FP64 pipe"),
    ("smsp__issue_active.avg.pct_of_peak_sustained_active", "issue slots busy"),
    ("smsp__inst_executed.sum", "warp instructions"),
    ("l1tex__data_pipe_lsu_wavefronts.sum.pct_of_peak_sustained_elapsed", "LSU wavefronts"),
    ("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed", "LSU wavefronts (shared)"),
    ("l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "shared bank conflicts"),
    ("lts__t_sector_hit_rate.pct", "L2 hit rate"),
    ("smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio", "stall long scoreboard / issue"),
    ("smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio", "stall short scoreboard / issue"),
    ("smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio", "stall math pipe throttle / issue"),
    ("smsp__average_warps_issue_stalled_wait_per_issue_active.ratio", "stall wait / issue"),
    ("smsp__average_warps_issue_stalled_mio_throttle_per_issue_active.ratio", "stall mio throttle / issue"),
    ("smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio", "stall barrier / issue"),
    ("smsp__average_warps_issue_stalled_not_selected_per_issue_active.ratio", "stall not selected / issue"),
]


def kernel_class(name: str):
    if "k_visc_march" in name or "k_visc_flux" in name:
        return "visc_flux"
    if "k_xi_ldg" in name or "k_xi_tma" in name or "k_march_xi" in name:
        return "inviscid_xi"
    m = re.search(r"k_march<\s*(\d)", name)
    if m:
        return "inviscid_eta" if m.group(1) == "1" else ("inviscid_zeta" if m.group(1) in "23" else "inviscid_xi")
    if "k_fill" in name:
        return "ghost_fill"
    return None


def to_bytes(value: str, unit: str) -> float:
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}.get(unit, 1.0)
    return float(value.replace(",", "")) * scale


def launch_list(csv_path, out_md, command):
    """Launch list of `ncu --metrics gpu__time_duration.sum --csv --log-file <csv>`: per kernel launches, total and
    average device time and share (cold caches, serialised launches: compare shares, not absolutes)."""
    with open(csv_path) as f:
        lines = [ln for ln in f if not ln.startswith("==")]
    rows = list(csv.DictReader(lines))
    agg = {}
    for r in rows:
        if r.get("Metric Name") != "gpu__time_duration.sum":
            continue
        v = float(r["Metric Value"].replace(",", ""))
        v *= {"ns": 1e-6, "us": 1e-3, "ms": 1.0, "s": 1e3}.get(r.get("Metric Unit", "ns"), 1e-6)
        k = r["Kernel Name"]
        a = agg.setdefault(k, [0, 0.0])
        a[0] += 1
        a[1] += v
    tot = sum(v[1] for v in agg.values())
    out = ["# ncu launch list", "", f"Command: `{command}`", "",
           "Per-launch times under ncu are cold-cache and serialised: the SHARES are what to compare with bench.py's", 
           "CUDA-event timing, not the absolutes.", "", "| kernel | launches | total ms | avg ms | share |", "|---|---|---|---|---|"]
    for k, (n, ms) in sorted(agg.items(), key=lambda kv: -kv[1][1]):
        out.append(f"| `{k[:90]}` | {n} | {ms:.3f} | {ms / n:.4f} | {ms / tot:.3f} |")
    with open(out_md, "w") as f:
        f.write("\n".join(out) + "\n")
    print(f"{len(agg)} kernels, {tot:.2f} ms total -> {out_md}")


def main():
    if len(sys.argv) > 1 and sys.argv[1] == "--launches":
        ap = argparse.ArgumentParser()
        ap.add_argument("--launches", required=True, help="csv written by ncu --csv --log-file")
        ap.add_argument("--out", required=True)
        ap.add_argument("--command", default="")
        a = ap.parse_args()
        return launch_list(a.launches, a.out, a.command)
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--workload", required=True)
    ap.add_argument("--out", required=True, help="prefix, e.g. profiles/r2")
    ap.add_argument("--command", default="", help="the full ncu command that made the report (recorded in the .md)")
    ap.add_argument("--note", default="")
    a = ap.parse_args()
    raw = subprocess.run(["ncu", "-i", a.report, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(raw.splitlines()))
    hdr, units, data = rows[0], rows[1], rows[2:]
    ki = hdr.index("Kernel Name")
    col = {h: i for i, h in enumerate(hdr)}
    per_class, first = {}, {}
    for r in data:
        cls = kernel_class(r[ki])
        if cls is None:
            continue
        rd = to_bytes(r[col["dram__bytes_read.sum"]], units[col["dram__bytes_read.sum"]])
        wr = to_bytes(r[col["dram__bytes_write.sum"]], units[col["dram__bytes_write.sum"]])
        per_class.setdefault(cls, []).append(rd + wr)
        first.setdefault(cls, r)
    traffic = {cls: sum(v) / len(v) for cls, v in per_class.items()}
    tj = a.out + "_traffic.json"
    merged = {}
    if os.path.exists(tj):
        with open(tj) as f:
            merged = json.load(f)
    merged[a.workload] = traffic
    merged.setdefault("_source", {})[a.workload] = {"report": os.path.basename(a.report), "command": a.command,
                                                    "launches_averaged": {c: len(v) for c, v in per_class.items()}}
    with open(tj, "w") as f:
        json.dump(merged, f, indent=1, sort_keys=True)
    order = [c for c in ("visc_flux", "inviscid_xi", "inviscid_eta", "inviscid_zeta", "ghost_fill") if c in first]
    lines = [f"# ncu --set full summary, workload {a.workload}", "", f"Command: `{a.command}`" if a.command else "", ""]
    if a.note:
        lines += [a.note, ""]
    lines += ["| metric | unit | " + " | ".join(f"{c} (`{first[c][ki][:40]}`)" for c in order) + " |",
              "|---|---|" + "---|" * len(order)]
    for m, label in METRICS:
        if m not in col:
            continue
        i = col[m]
        lines.append(f"| {label} (`{m}`) | {units[i]} | " + " | ".join(first[c][i] for c in order) + " |")
    lines += ["", "DRAM traffic per launch (read + written, average over the captured launches), as stored in "
              f"`{os.path.basename(tj)}`:", ""]
    for c in order:
        lines.append(f"* {c}: {traffic[c] / 1e9:.3f} GB ({len(per_class[c])} launch(es))")
    hot = [c for c in order if c != "ghost_fill"]
    lines += ["", f"Sum over the hot kernels of one stage: {sum(traffic[c] for c in hot) / 1e9:.2f} GB.", ""]
    with open(a.out + "_hot_kernels.md", "w") as f:
        f.write("\n".join(lines))
    print(json.dumps(traffic, indent=1))


if __name__ == "__main__":
    main()
