"""Turn an `ncu` report into the text summaries kept under profiles/ and into the machine-readable
DRAM-traffic record that bench.py quotes as `roofline.traffic`.

    python -m paper_1908_05232_b200.ncu_summary full  <report.ncu-rep> <out.md> [--traffic profiles/r2_traffic.json --key config5] [--cmd "..."]
    python -m paper_1908_05232_b200.ncu_summary list  <launches.csv>   <out.md> [--cmd "..."]

`full`: one section per profiled launch with the counters DESIGN.md argues from (duration, DRAM
bytes, hit rates, pipe utilisation, issue slots, the top stall reasons).  `list`: per-kernel share
of a `--metrics gpu__time_duration.sum` launch list.  Needs the `ncu` binary (it reads the report);
no GPU.  Nothing here is on the product path.
"""
from __future__ import annotations

import argparse
import csv
import io
import json
import os
import subprocess
from collections import defaultdict

WANT = [
    "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum",
    "dram__throughput.avg.pct_of_peak_sustained_elapsed", "lts__t_sector_hit_rate.pct", "l1tex__t_sector_hit_rate.pct",
    "sm__throughput.avg.pct_of_peak_sustained_elapsed", "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "sm__warps_active.avg.pct_of_peak_sustained_active", "launch__registers_per_thread", "launch__grid_size",
    "launch__block_size", "smsp__inst_executed.sum", "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active", "smsp__inst_executed_pipe_xu.sum",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
]


def _raw(report: str):
    out = subprocess.run(["ncu", "-i", report, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    return rows[0], rows[1], rows[2:]


def _bytes(value: str, unit: str) -> float:
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}[unit]
    return float(value.replace(",", "")) * scale


def full(report: str, out_md: str, traffic_json: str | None, key: str | None, cmd: str | None):
    H, U, rows = _raw(report)
    col = {h: i for i, h in enumerate(H)}
    lines = [f"# ncu --set full: {os.path.basename(report)}", ""]
    if cmd:
        lines += ["Command (under `gpurun`; every file it runs is committed):", "", "    " + cmd, ""]
    lines += ["Read here with `python -m paper_1908_05232_b200.ncu_summary full <report> <this file>`.", ""]
    traffic = {}
    for r in rows:
        name = r[col["Kernel Name"]]
        lines += [f"## {name}", "", "| counter | value | unit |", "|---|---|---|"]
        for w in WANT:
            if w in col:
                lines.append(f"| {w} | {r[col[w]]} | {U[col[w]]} |")
        stalls = []
        for h, i in col.items():
            if h.startswith("smsp__average_warps_issue_stalled_") and h.endswith("_per_issue_active.ratio"):
                try:
                    stalls.append((float(r[i]), h[len("smsp__average_warps_issue_stalled_"):-len("_per_issue_active.ratio")]))
                except ValueError:
                    pass
        stalls.sort(reverse=True)
        lines += ["", "Stall reasons (warps stalled per issue-active cycle): " + ", ".join(f"{n} {v:.2f}" for v, n in stalls[:8]), ""]
        rd = _bytes(r[col["dram__bytes_read.sum"]], U[col["dram__bytes_read.sum"]])
        wr = _bytes(r[col["dram__bytes_write.sum"]], U[col["dram__bytes_write.sum"]])
        dur = r[col["gpu__time_duration.sum"]] + " " + U[col["gpu__time_duration.sum"]]
        traffic.setdefault(name.split("(")[0], []).append({"dram_bytes_read": rd, "dram_bytes_write": wr, "duration": dur})
    with open(out_md, "w") as f:
        f.write("\n".join(lines) + "\n")
    if traffic_json and key:
        data = json.load(open(traffic_json)) if os.path.exists(traffic_json) else {}
        rec = data.setdefault(key, {})
        for name, caps in traffic.items():
            n = len(caps)
            rec[name] = {"dram_bytes_read": sum(c["dram_bytes_read"] for c in caps) / n,
                         "dram_bytes_write": sum(c["dram_bytes_write"] for c in caps) / n,
                         "launches_averaged": n, "summary": os.path.relpath(out_md, os.path.dirname(traffic_json) or "."),
                         "command": cmd}
        with open(traffic_json, "w") as f:
            json.dump(data, f, indent=1, sort_keys=True)
            f.write("\n")


def launch_list(csv_path: str, out_md: str, cmd: str | None):
    rows = [r for r in csv.reader(open(csv_path)) if r]
    start = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    H = rows[start]
    col = {h: i for i, h in enumerate(H)}
    tot, cnt = defaultdict(float), defaultdict(int)
    for r in rows[start + 1:]:
        if len(r) < len(H) or r[col["Metric Name"]] != "gpu__time_duration.sum":
            continue
        v = float(r[col["Metric Value"]].replace(",", ""))
        unit = r[col["Metric Unit"]]
        v *= {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}.get(unit, 1.0)
        name = r[col["Kernel Name"]].split("(")[0]
        tot[name] += v; cnt[name] += 1
    total = sum(tot.values())
    lines = [f"# ncu launch list: {os.path.basename(csv_path)}", ""]
    if cmd:
        lines += ["Command (under `gpurun`; every file it runs is committed):", "", "    " + cmd, ""]
    lines += ["Per-launch times under ncu are cold-cache and serialised: the SHARE of a kernel is what compares",
              "with bench.py's CUDA-event figures, not the absolute.", "",
              "| kernel | launches | mean us | share of listed time |", "|---|---|---|---|"]
    for name in sorted(tot, key=tot.get, reverse=True):
        lines.append(f"| {name} | {cnt[name]} | {tot[name] / cnt[name]:.2f} | {100 * tot[name] / total:.1f} % |")
    with open(out_md, "w") as f:
        f.write("\n".join(lines) + "\n")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("mode", choices=["full", "list"])
    ap.add_argument("src")
    ap.add_argument("out")
    ap.add_argument("--traffic")
    ap.add_argument("--key")
    ap.add_argument("--cmd")
    a = ap.parse_args()
    if a.mode == "full":
        full(a.src, a.out, a.traffic, a.key, a.cmd)
    else:
        launch_list(a.src, a.out, a.cmd)


if __name__ == "__main__":
    main()
