"""Turn an `ncu --set full` report into the small counters file bench.py reads (profiles/*_ncu_counters.json).

    python -m paper_1208_3407_b200.ncu_counters OUT.json REPORT.ncu-rep [REPORT2.ncu-rep ...] --workload NAME --command "the ncu command line(s)"

Run it in the SAME gpurun command as the capture, right behind it: the file then carries build.csrc_hash() of exactly
the sources the captured kernels were built from, and nobody ever types that hash.  bench.py reports the counters only
while the hash still matches the build it runs.  Per kernel (launches of one kernel are averaged) it keeps what only
ncu can give: DRAM bytes, warp instructions, the pipe / issue / memory utilisations that name the limiter, the L2
sector counters.  Needs the `ncu` binary (it reads reports without a GPU).
"""
from __future__ import annotations

import argparse
import csv
import io
import json
import re
import subprocess
import sys

from . import build as B

# metric name in the report -> key in the JSON (missing metrics are skipped)
METRICS = {
    "gpu__time_duration.sum": "duration_under_ncu",
    "dram__bytes_read.sum": "dram_bytes_read",
    "dram__bytes_write.sum": "dram_bytes_write",
    "smsp__inst_executed.sum": "warp_instructions",
    "sm__inst_executed.sum": "warp_instructions_sm",
    "smsp__thread_inst_executed.sum": "thread_instructions",
    "sm__inst_issued.avg.pct_of_peak_sustained_active": "issue_slots_busy_pct",
    "smsp__issue_active.avg.pct_of_peak_sustained_active": "issue_active_pct",
    "sm__instruction_throughput.avg.pct_of_peak_sustained_active": "instruction_throughput_pct",
    "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed": "dram_throughput_pct",
    "sm__warps_active.avg.pct_of_peak_sustained_active": "warps_active_pct",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum": "shared_wavefronts",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum": "shared_bank_conflict_wavefronts",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.avg.pct_of_peak_sustained_elapsed": "shared_memory_pipe_pct",
    "l1tex__lsu_writeback_active_mem_lg.avg.pct_of_peak_sustained_elapsed": "l1_lsu_writeback_pct",
    "l1tex__throughput.avg.pct_of_peak_sustained_active": "l1tex_throughput_pct",
    "lts__throughput.avg.pct_of_peak_sustained_elapsed": "l2_throughput_pct",
    "lts__t_sectors_srcunit_tex_op_read.sum": "l2_sectors_read",          # sectors the SMs read from L2 (hits and misses)
    "lts__t_sectors_srcunit_tex_op_write.sum": "l2_sectors_write",
    "lts__t_sectors_srcunit_tex_op_red.sum": "l2_sectors_red",
    "lts__t_requests_srcunit_tex_op_read.sum": "l2_read_requests",
    "lts__t_sectors_srcunit_tex_op_read_lookup_miss.sum": "l2_sectors_read_miss",
    "lts__t_sector_hit_rate.pct": "l2_hit_rate_pct",
    "l1tex__t_sectors_pipe_lsu_mem_global_op_ld.sum": "l1_global_load_sectors",
    "l1tex__t_requests_pipe_lsu_mem_global_op_ld.sum": "l1_global_load_requests",
    "l1tex__t_sector_hit_rate.pct": "l1_hit_rate_pct",
    "launch__registers_per_thread": "registers_per_thread",
    "launch__grid_size": "grid_size",
    "launch__block_size": "block_size",
    "launch__occupancy_limit_shared_mem": "occupancy_limit_shared_mem_blocks",
    "smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio": "stall_barrier_per_issue",
    "smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio": "stall_long_scoreboard_per_issue",
    "smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio": "stall_short_scoreboard_per_issue",
    "smsp__average_warps_issue_stalled_mio_throttle_per_issue_active.ratio": "stall_mio_throttle_per_issue",
    "smsp__average_warps_issue_stalled_lg_throttle_per_issue_active.ratio": "stall_lg_throttle_per_issue",
    "smsp__average_warps_issue_stalled_wait_per_issue_active.ratio": "stall_wait_per_issue",
    "smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio": "stall_math_pipe_per_issue",
    "smsp__average_warps_issue_stalled_not_selected_per_issue_active.ratio": "stall_not_selected_per_issue",
}


def short_name(full: str) -> str:
    """`void ns::kernel<...>(args)` -> `kernel<...>` without the namespace and the argument list."""
    s = re.sub(r"^void\s+", "", full.strip())
    depth, cut = 0, len(s)
    for i, ch in enumerate(s):
        if ch == "<":
            depth += 1
        elif ch == ">":
            depth -= 1
        elif ch == "(" and depth == 0:
            cut = i
            break
    s = s[:cut]
    head, sep, tail = s.partition("<")
    return head.split("::")[-1] + sep + tail


def read_report(report: str):
    raw = subprocess.run(["ncu", "-i", report, "--page", "raw", "--csv"], check=True, capture_output=True, text=True).stdout
    rows = list(csv.reader(io.StringIO(raw)))
    header = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    names, units = rows[header], rows[header + 1]
    return names, units, [r for r in rows[header + 2:] if len(r) == len(names)]


def to_number(x: str):
    """None for text and for the nan ncu prints when a counter could not be collected (very long kernels)."""
    try:
        v = float(x.replace(",", ""))
    except ValueError:
        return None
    return v if v == v and abs(v) != float("inf") else None


def summarise(report: str) -> dict:
    names, units, launches = read_report(report)
    col = {n: i for i, n in enumerate(names)}
    kernels: dict[str, dict] = {}
    for r in launches:
        k = kernels.setdefault(short_name(r[col["Kernel Name"]]), {"launches_captured": 0, "_sum": {}, "_unit": {}})
        k["launches_captured"] += 1
        for metric, key in METRICS.items():
            if metric in col:
                v = to_number(r[col[metric]])
                if v is not None:
                    k["_sum"][key] = k["_sum"].get(key, 0.0) + v
                    k["_unit"][key] = units[col[metric]]
    out = {}
    for name, k in kernels.items():
        n = k["launches_captured"]
        d = {"launches_captured": n}
        for key, s in k["_sum"].items():
            v = s / n
            unit = k["_unit"][key]
            if key == "duration_under_ncu":                      # ncu prints ns, us or ms depending on the value
                scale = {"ns": 1e-3, "us": 1.0, "usecond": 1.0, "ms": 1e3, "msecond": 1e3, "nsecond": 1e-3, "s": 1e6, "second": 1e6}.get(unit, None)
                d["duration_us_under_ncu"] = v * scale if scale else v
                continue
            if key.startswith("dram_bytes") or key.startswith("l2_sectors") or key.endswith("requests") or key.endswith("instructions") or key.endswith("wavefronts"):
                mult = {"Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "byte": 1.0}.get(unit, 1.0)
                d[key] = int(round(v * mult))
            else:
                d[key] = round(v, 4)
        if "dram_bytes_read" in d and "dram_bytes_write" in d:
            d["dram_bytes"] = d["dram_bytes_read"] + d["dram_bytes_write"]
        lim = {}
        for key, label in (("issue_slots_busy_pct", "issue_slots_busy"), ("shared_memory_pipe_pct", "shared_memory_pipe"),
                           ("dram_throughput_pct", "dram_throughput"), ("l2_throughput_pct", "l2_throughput"),
                           ("warps_active_pct", "warps_active")):
            if key in d:
                lim[label] = round(d[key] / 100.0, 4)
        if d.get("shared_wavefronts"):
            lim["shared_bank_conflicts_of_wavefronts"] = round(d.get("shared_bank_conflict_wavefronts", 0) / d["shared_wavefronts"], 4)
        if lim:
            busiest = max((k2 for k2 in lim if k2 not in ("warps_active", "shared_bank_conflicts_of_wavefronts")), key=lambda k2: lim[k2], default=None)
            if busiest:
                lim["busiest_unit"] = busiest
            d["limiter"] = lim
        out[name] = d
    return out


def main(argv=None) -> int:
    p = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    p.add_argument("out")
    p.add_argument("report", nargs="+")
    p.add_argument("--workload", default="")
    p.add_argument("--command", default="", help="the ncu command line that made the report (recorded verbatim)")
    a = p.parse_args(argv)
    doc = {
        "what": "Counters that only ncu can give, per kernel (averaged over the captured launches); written by "
                "paper_1208_3407_b200/ncu_counters.py in the same gpurun command as the capture. bench.py reports them only "
                "while csrc_hash equals build.csrc_hash() of the build it runs (otherwise 'stale_capture').",
        "command": a.command,
        "csrc_hash": B.csrc_hash(),
        "csrc_hash_covers": list(B.HASHED_SOURCES),
        "workload": a.workload,
        "kernels": {},
    }
    for rep in a.report:
        doc["kernels"].update(summarise(rep))
    with open(a.out, "w") as f:
        json.dump(doc, f, indent=1)
        f.write("\n")
    print(f"{a.out}: {len(doc['kernels'])} kernels, csrc {doc['csrc_hash']}")
    return 0


if __name__ == "__main__":
    sys.exit(main())
