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




# ---------------------------------------------------------------------------------------------------------------
# Per-phase instruction budget of bin_sort_search_kernel from the source page of an `--import-source on` capture:
#     python -m paper_1208_3407_b200.ncu_counters --phases OUT.md REPORT.ncu-rep --keys N
# Every source line's counters (warp instructions executed, shared-memory wavefronts, excess wavefronts = bank
# conflicts, stall samples) are summed over the phase the line belongs to.  Phases are line ranges of mc_tile.cuh found
# from the marker strings below, so the table follows the file as it changes.
PHASE_MARKERS = (      # (phase, first-line marker, last-line marker) in mc_tile.cuh; helper functions count for their phase
    ("count (count_key)", "__device__ __forceinline__ void count_key(", "// position of the next key of sub-bucket sb"),
    ("scatter (take_slot)", "__device__ __forceinline__ uint32_t take_slot(", "// Counts -> exclusive prefixes, in place"),
    ("scan of the cursors (scan_cursors)", "__device__ __forceinline__ void scan_cursors(", "// Counting-sort scatter of buf[0..m) in place"),
    ("scatter (scatter_in_place)", "__device__ __forceinline__ void scatter_in_place(", "// Write buf[0..mv) (ordered by sub-bucket)"),
    ("write-out + tie rank (write_and_rank, first loop)", "__device__ __forceinline__ uint64_t write_and_rank(", "  uint64_t qsum = 0;\n  for (uint32_t qi"),
    ("query rank (write_and_rank, second loop)", "  uint64_t qsum = 0;\n  for (uint32_t qi", "template <class C, bool kSlots = false>"),
    ("per-bin prologue: ticket, segment words, scans, cursor clear", "bin_sort_search_kernel(BinSortArgs a) {", "    // gather: a group of lanes per segment"),
    ("gather (cp.async of the pairs and the hand-over list)", "    // gather: a group of lanes per segment", "    // Algorithm 2's Sort(B_S), Sort(B_E) for this bin"),
    ("count (loop in the kernel body)", "    // Algorithm 2's Sort(B_S), Sort(B_E) for this bin", "    uint32_t total[2];"),
    ("calls + block reduce (kernel body tail)", "    uint32_t total[2];", "// Query ranges per bin, once per call"),
)


def phase_budget(report: str, n_keys: float, kernel_regex: str = "bin_sort_search_kernel") -> str:
    import os
    text = open(os.path.join(B.CSRC, "mc_tile.cuh")).read()
    line_of = lambda marker: text[:text.index(marker)].count("\n") + 1
    ranges = [(name, line_of(a), line_of(b) - 1) for name, a, b in PHASE_MARKERS]
    raw = subprocess.run(["ncu", "-i", report, "--page", "source", "--csv", "--print-source", "cuda,sass", "--kernel-name",
                          f"regex:{kernel_regex}"], check=True, capture_output=True, text=True).stdout
    cur_file, cols, kernel = None, None, ""
    agg: dict[str, list[float]] = {}
    fields = ("Instructions Executed", "L1 Wavefronts Shared", "L1 Wavefronts Shared Excessive", "# Samples", "stall_barrier",
              "stall_long_sb", "stall_short_sb", "stall_mio")
    for r in csv.reader(io.StringIO(raw)):
        if len(r) == 2 and r[0] == "File Path":
            cur_file = os.path.basename(r[1]); continue
        if len(r) == 2 and r[0] == "Function Name":
            kernel = r[1]; continue
        if r and r[0] == "Line No":
            cols = {}
            for i, n in enumerate(r):
                cols.setdefault(n, i)
            continue
        if not cols or len(r) < len(cols) or r[cols["Address"]] != "-":
            continue                                  # SASS rows repeat what the line's own row already sums
        try:
            line = int(r[0])
        except ValueError:
            continue
        phase = f"other files ({cur_file})"
        if cur_file == "mc_tile.cuh":
            phase = next((name for name, lo, hi in ranges if lo <= line <= hi), "mc_tile.cuh, other lines (sub_of, ...)")
        a = agg.setdefault(phase, [0.0] * len(fields))
        for j, f in enumerate(fields):
            a[j] += to_number(r[cols[f]]) or 0.0
    tot = [sum(a[j] for a in agg.values()) for j in range(len(fields))]
    out = [f"Kernel: `{kernel}`", "",
           f"Source-page counters summed per phase; per key = divided by {n_keys:.0f} keys per launch (both arrays). "
           "One warp instruction = up to 32 thread instructions.", "",
           "| phase | mc_tile.cuh lines | warp instr | share | thread instr per key (x32) | shared wavefronts | excess (bank conflicts) | stall samples | of which barrier | long_sb | short_sb | mio |",
           "|---|---|---|---|---|---|---|---|---|---|---|---|"]
    lines_of = {name: f"{lo}-{hi}" for name, lo, hi in ranges}
    for name, a in sorted(agg.items(), key=lambda kv: -kv[1][0]):
        out.append(f"| {name} | {lines_of.get(name, '')} | {a[0]:,.0f} | {a[0] / tot[0]:.3f} | {32 * a[0] / n_keys:.1f} | {a[1]:,.0f} | {a[2]:,.0f} | "
                   f"{a[3]:,.0f} | {a[4]:,.0f} | {a[5]:,.0f} | {a[6]:,.0f} | {a[7]:,.0f} |")
    out.append(f"| **total** | | {tot[0]:,.0f} | 1.000 | {32 * tot[0] / n_keys:.1f} | {tot[1]:,.0f} | {tot[2]:,.0f} | {tot[3]:,.0f} | {tot[4]:,.0f} | {tot[5]:,.0f} | {tot[6]:,.0f} | {tot[7]:,.0f} |")
    return "\n".join(out) + "\n"


def phases_main(argv) -> int:
    p = argparse.ArgumentParser()
    p.add_argument("out"); p.add_argument("report"); p.add_argument("--keys", type=float, default=2e7)
    p.add_argument("--kernel", default="bin_sort_search_kernel")
    a = p.parse_args(argv)
    body = phase_budget(a.report, a.keys, a.kernel)
    with open(a.out, "w") as f:
        f.write(f"<!-- written by: python -m paper_1208_3407_b200.ncu_counters --phases {a.out} {a.report} --keys {a.keys:.0f}; csrc {B.csrc_hash()} -->\n\n" + body)
    print(body)
    return 0


if __name__ == "__main__":
    sys.exit(phases_main(sys.argv[2:]) if len(sys.argv) > 1 and sys.argv[1] == "--phases" else main())
