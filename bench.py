#!/usr/bin/env python
"""bench.py -- Monte Carlo rounds/s of the BITS hot path (place -> sort -> search -> reduce) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config 5] [--rounds R]
    python bench.py --config 2|4          the counting configs as a line of their own (metric intervals_searched_per_s)

Workload (config.workload): BASELINE.json configs[4], "Monte Carlo at scale with per-round sort":
24-chromosome genome, A = 1e6 query intervals, B = 1e7 intervals re-placed with Philox and radix-
sorted (starts and ends) every round, all of A counted and reduced per round.  One STEP is one
bits_mc_rounds call of R rounds (default R = 1000, the configuration's round count), i.e. R passes
of the whole hot path, plus the one-off observed count.  value = rounds/s over K timed steps with
the inputs resident in HBM; e2e = the same through bits_mc_rounds_host with pinned HOST buffers
(H2D of A and B and D2H of the counts inside the timed region).

Under torchrun (N > 1) every rank runs its own R rounds (round_begin = rank * R): the rounds of a
Monte Carlo job are independent, so they shard with no data-path collective ("weak" scaling).

--impl reference times the CPU oracle (oracle/, single-threaded C++) on the same workload, each
step a bounded sample of rounds.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# Counters of the dominant kernels that only ncu can give (DRAM bytes, warp instructions, what bounds the kernel) live
# in profiles/r3_fused_ncu_counters.json, written by paper_1208_3407_b200/ncu_counters.py in the same gpurun command as
# the `ncu --set full` capture, together with the hash of the sources it was taken of (build.csrc_hash(): all of csrc/,
# kernels and host launch geometry).  They are reported only while that hash is the one of the sources this run was
# built from; otherwise the line says "stale_capture".
NCU_COUNTERS_FILE = os.path.join(ROOT, "profiles", "r3_fused_ncu_counters.json")


# The same for the L2-bound kernels (config 3's PERMUTE_A rounds at the benchmarked 10,000 rounds per launch, the screen):
# L2 sectors read per launch and the hit rate, from which other_workloads prints an l2_roofline.
NCU_L2_COUNTERS_FILE = os.path.join(ROOT, "profiles", "r3_l2_ncu_counters.json")


def ncu_counters(path=None):
    """(counters by kernel, note) -- counters are {} when the capture is missing or belongs to other sources."""
    from paper_1208_3407_b200 import build as B
    path = path or NCU_COUNTERS_FILE
    if not os.path.exists(path):
        return {}, "no capture file"
    with open(path) as f:
        d = json.load(f)
    have = B.csrc_hash()
    if d.get("csrc_hash") != have:
        return {}, f"stale_capture: {os.path.basename(path)} was taken of csrc {d.get('csrc_hash')}, this build is {have}"
    return d.get("kernels", {}), f"from {os.path.basename(path)} (csrc {have}, workload {d.get('workload')})"


def kernel_counters(counters: dict, kname: str) -> dict:
    """Counters of the kernel whose name (without namespace; with or without template arguments) is kname."""
    if kname in counters:
        return counters[kname]
    return next((v for k, v in sorted(counters.items()) if k.split("<")[0] == kname), {})


def l2_roofline(kname: str, intervals_per_launch: float, intervals_per_s: float, gather_gsectors_per_s: float) -> dict:
    """SURVEY 8(d), L2-bound search kernels: 32-byte sectors read from L2 per searched interval (ncu capture of the
    kernel at the benchmarked shape) x the interval rate measured in this run, against the random-sector gather rate
    measured in this run (probe/l2_probe.cu)."""
    counters, note = ncu_counters(NCU_L2_COUNTERS_FILE)
    kc = kernel_counters(counters, kname)
    if not kc.get("l2_sectors_read"):
        return {"kernel": kname, "ncu_counters": note if not counters else f"{kname} not in the capture"}
    spi = kc["l2_sectors_read"] / intervals_per_launch
    ach = spi * intervals_per_s / 1e9
    return {"kernel": kname, "bound": "l2", "sectors_per_interval": spi, "achieved_gsectors_per_s": ach,
            "peak": gather_gsectors_per_s, "unit": "Gsectors/s", "frac": ach / gather_gsectors_per_s if gather_gsectors_per_s else None,
            "l2_hit_rate_pct": kc.get("l2_hit_rate_pct"), "l2_throughput_pct_under_ncu": kc.get("l2_throughput_pct"),
            "dram_bytes_per_launch": kc.get("dram_bytes"), "ncu_counters": note,
            "peak_source": "l2_yardsticks.l2_random_sector_gather_gsectors_per_s_80MB of this run"}


N_SMS, SCHEDULERS_PER_SM = 148, 4
HBM_FALLBACK_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent


def parse_args():
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=5)
    p.add_argument("--warmup", type=int, default=3)
    p.add_argument("--impl", default="b200", choices=["b200", "reference"])
    p.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    p.add_argument("--scale", type=float, default=1.0, help="scale the set sizes (testing only; 1.0 = the named config)")
    p.add_argument("--rounds", type=int, default=0, help="rounds per step (0 = the configuration's own count)")
    p.add_argument("--opt", action="append", default=[], metavar="NAME=VALUE",
                   help="bits_set_option knob for design studies (DESIGN.md section 10); results never change")
    p.add_argument("--study", default=None, choices=["search", "count", "screen"],
                   help="design studies instead of the bench line: 'search' = config 4 with every search design of the count "
                        "path + 100 rounds of config 3; 'count' = config 4's bits_count_per_interval only (the command the "
                        "ncu captures under profiles/ run); with --once every call runs once, without warm-up")
    p.add_argument("--once", action="store_true", help="--study: one call per design, no warm-up (for captures under ncu)")
    p.add_argument("--no-extras", action="store_true", help="skip the secondary workloads, e2e and cpu_baseline legs")
    p.add_argument("--no-profile-events", action="store_true", help="do not bracket kernels with events in the timed region")
    return p.parse_args()


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy bandwidth)"
    return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        with open(self.path) as f:
            for line in f:
                c = [x.strip() for x in line.split(",")]
                if len(c) < 7:
                    continue
                try:
                    sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
                except ValueError:
                    continue
                for n, v in zip(names, c[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
        os.unlink(self.path)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


def golden_round_counts(config: int, mc_seed: int):
    """(header, uint64 counts) from tests/golden/cfg<k>_seed<s>_rounds.txt (the oracle's per-round counts, written by
    tests/golden/make_golden.py), or (None, None) if there is no such file.  Reads the file only: no oracle code runs."""
    path = os.path.join(ROOT, "tests", "golden", f"cfg{config}_seed{mc_seed}_rounds.txt")
    if not os.path.exists(path):
        return None, None
    header, vals = None, []
    with open(path) as f:
        for ln in f:
            ln = ln.strip()
            if ln.startswith("#"):
                if ln[1:].strip().startswith("{"):
                    header = json.loads(ln[1:].strip())
            elif ln:
                vals.append(int(ln))
    return header, np.array(vals, dtype=np.uint64)


def workload_name(k: int) -> str:
    from paper_1208_3407_b200 import workloads as W
    return W.CONFIG_NAMES[k]


def config_block(w, rounds: int, n_gpus: int) -> dict:
    return {"workload": w.name, "n_a": w.n_a, "n_b": w.n_b, "n_chrom": int(w.chrom_offsets.size - 1),
            "rounds_per_step": rounds, "which": {0: "permute_A", 1: "permute_B", None: "count"}[w.which],
            "mc_seed": w.mc_seed, "data_seed": w.spec.get("seed"), "scale": w.spec.get("scale", 1.0),
            "parallelism": f"rounds sharded over {n_gpus} GPU(s), no collective",
            "l2": "no flush: inputs larger than L2 -- every round streams 40 MB of spans, 80 MB of pairs and 80 MB of sorted keys (200 MB > 126 MB L2)"}


# ------------------------------------------------------------------------------------------ reference arm
def oracle_marginal_rounds_per_s(w, which: int, round_begin: int, n_rounds: int):
    """Oracle rounds/s from the marginal cost of n_rounds rounds: t(R = n_rounds) - t(R = 0).
    (The R = 0 call is the one-off observed count, which a 1000-round job amortises away.)"""
    import oracle
    args = (w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, which, w.mc_seed)
    t0 = time.perf_counter(); oracle.mc_rounds(*args, round_begin, 0); t_obs = time.perf_counter() - t0
    t0 = time.perf_counter(); oracle.mc_rounds(*args, round_begin, n_rounds); t_r = time.perf_counter() - t0
    per_round = max((t_r - t_obs) / n_rounds, 1e-9)
    return 1.0 / per_round, t_obs, t_r


def oracle_sample_text(n_rounds: int, w) -> str:
    return (f"{n_rounds} of the workload's {w.n_rounds} rounds per step (full-size A and B): time of "
            f"oracle.mc_rounds(R={n_rounds}) minus time of oracle.mc_rounds(R=0), i.e. the marginal per-round "
            f"cost (place {w.n_b if w.which == 1 else w.n_a} intervals, std::sort both key arrays, {w.n_a} ICOUNTs, sum)")


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    from paper_1208_3407_b200 import workloads as W
    oracle.build()
    w = W.make_config(args.config, scale=args.scale)
    if w.which is None:
        # counting configs: a step is the oracle's whole call (std::sort of B's two key arrays + one ICOUNT per query + sum)
        for _ in range(min(args.warmup, 1)):
            oracle.count_per_interval(w.a_start, w.a_end, w.b_start, w.b_end)
        t0 = time.perf_counter()
        for _ in range(args.steps):
            oracle.count_per_interval(w.a_start, w.a_end, w.b_start, w.b_end)
        dt = time.perf_counter() - t0
        value = w.n_a * args.steps / dt
        print(json.dumps({
            "impl": "reference", "metric": "intervals_searched_per_s", "value": value, "unit": "intervals/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
            "config": {"workload": w.name, "n_a": w.n_a, "n_b": w.n_b, "data_seed": w.spec.get("seed"), "scale": w.spec.get("scale", 1.0)},
            "cpu_baseline": {"value": value, "unit": "intervals/s", "cores": 1, "kind": "oracle",
                             "sample": "the whole call per step: std::sort of both key arrays of B + one ICOUNT per query + sum"},
            "e2e": {"value": value, "unit": "intervals/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "host_cores": os.cpu_count()}))
        return 0
    r_sample = 1 if args.config == 5 else (args.rounds or 100)
    for i in range(args.warmup):
        oracle_marginal_rounds_per_s(w, w.which, i * r_sample, r_sample)
    t_total, rounds_total, per_step = 0.0, 0, []
    for i in range(args.steps):
        rps, _, _ = oracle_marginal_rounds_per_s(w, w.which, (args.warmup + i) * r_sample, r_sample)
        per_step.append(rps)
        t_total += r_sample / rps
        rounds_total += r_sample
    value = rounds_total / t_total
    line = {
        "impl": "reference", "metric": "mc_rounds_per_s", "value": value, "unit": "rounds/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_total / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": config_block(w, r_sample, args.gpus),
        "cpu_baseline": {"value": value, "unit": "rounds/s", "cores": 1, "kind": "oracle",
                         "sample": oracle_sample_text(r_sample, w)},
        "e2e": {"value": value, "unit": "rounds/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "intervals_searched_per_s": value * w.n_a,
        "host_cores": os.cpu_count(),
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------ B200 arm
def to_dev(a, device):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.uint32).view(np.int32)).to(device)


def pinned(a):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a, dtype=np.uint32).view(np.int32)).pin_memory()
    return t, t.numpy().view(np.uint32)


def time_device(fn, reps: int, warmup: int = 3):
    """Median and min device time (ms) of fn() by CUDA events on the current stream."""
    import torch
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); fn(); b.record(); b.synchronize()
        ts.append(a.elapsed_time(b))
    return statistics.median(ts), min(ts)


def l2_yardsticks(device):
    """L2 denominators for the search kernels: streaming read over 48 MB and random
    32-byte-sector gather over 80 MB, both L2-resident.  Bench-only code (probe/l2_probe.cu)."""
    import ctypes as C
    import torch
    from paper_1208_3407_b200 import build as B
    lib = C.CDLL(B.build_probe())
    for f in (lib.l2_probe_stream_gbs, lib.l2_probe_gather_gsectors):
        f.restype = C.c_double
        f.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p, C.c_int, C.c_void_p]
    buf = torch.ones(80 << 20, dtype=torch.uint8, device=device)
    sink = torch.zeros(4, dtype=torch.int32, device=device)
    st = torch.cuda.current_stream().cuda_stream
    stream = lib.l2_probe_stream_gbs(buf.data_ptr(), 48 << 20, sink.data_ptr(), 10, st)
    gather = lib.l2_probe_gather_gsectors(buf.data_ptr(), 80 << 20, sink.data_ptr(), 10, st)
    return {"l2_stream_read_gbs_48MB": stream, "l2_random_sector_gather_gsectors_per_s_80MB": gather,
            "l2_random_sector_gather_gbs_80MB": gather * 32}


def library_yardsticks(device, w4, d4):
    """SURVEY 8(d) "Yardsticks": cub::DeviceRadixSort::SortKeys and thrust upper_bound / lower_bound on the same
    arrays on this box (bench-only code in probe/yardsticks.cu, never linked into libbits_b200.so).
    w4, d4: config 4 and its device arrays (a_start, a_end, b_start, b_end)."""
    import ctypes as C
    import torch
    from paper_1208_3407_b200 import bits
    from paper_1208_3407_b200 import build as B
    from paper_1208_3407_b200 import workloads as W
    lib = C.CDLL(B.build_yardsticks())
    lib.yard_cub_sort_temp_bytes.restype = C.c_size_t
    lib.yard_cub_sort_temp_bytes.argtypes = [C.c_uint64]
    lib.yard_cub_sort_keys_ms.restype = C.c_double
    lib.yard_cub_sort_keys_ms.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p, C.c_size_t, C.c_int, C.c_int, C.c_int, C.c_void_p]
    lib.yard_thrust_bounds_ms.restype = C.c_double
    lib.yard_thrust_bounds_ms.argtypes = [C.c_void_p] * 2 + [C.c_uint64] + [C.c_void_p] * 2 + [C.c_uint64] + [C.c_void_p] * 2 + [C.c_int, C.c_void_p]
    st = torch.cuda.current_stream().cuda_stream
    n = w4.n_b
    tmp = torch.empty(max(int(lib.yard_cub_sort_temp_bytes(n)), 256), dtype=torch.uint8, device=device)
    srt = [torch.empty(n, dtype=torch.int32, device=device) for _ in range(2)]
    out = {}
    # config 4: B's starts and B's ends (what bits_count* sorts once per call)
    ms = [lib.yard_cub_sort_keys_ms(d4[2 + k].data_ptr(), srt[k].data_ptr(), n, tmp.data_ptr(), tmp.numel(), 0, 32, 5, st) for k in range(2)]
    out["cub_sort_cfg4_B_2x1e7_keys"] = {"ms_both_arrays": sum(ms), "sort_keys_per_s": 2 * n / (sum(ms) * 1e-3)}
    # the same two searches per query as count_kernel, as two vectorised library calls on the arrays cub just sorted
    first = torch.empty(w4.n_a, dtype=torch.int32, device=device)
    last = torch.empty(w4.n_a, dtype=torch.int32, device=device)
    tb = lib.yard_thrust_bounds_ms(srt[0].data_ptr(), srt[1].data_ptr(), n, d4[1].data_ptr(), d4[0].data_ptr(), w4.n_a,
                                   first.data_ptr(), last.data_ptr(), 3, st)
    out["thrust_bounds_cfg4_1e7_queries"] = {"ms_upper_plus_lower": tb, "intervals_searched_per_s": w4.n_a / (tb * 1e-3),
                                             "note": "ranks written to two arrays; no subtraction, no reduction"}
    torch.cuda.synchronize()
    want = bits.count_per_interval(*d4)[0]
    torch.cuda.synchronize()
    out["thrust_bounds_cfg4_1e7_queries"]["same_counts_as_library"] = bool(torch.equal(first - last, want))
    del first, last, want
    # config 5: the freshly placed keys of one round (what every PERMUTE_B round sorts)
    w5 = W.make_config(5)
    spans = to_dev((w5.b_end - w5.b_start).astype(np.uint32), device)
    ps, pe = bits.place(spans, w5.chrom_offsets, w5.mc_seed, 0, 1)
    torch.cuda.synchronize()
    ms = [lib.yard_cub_sort_keys_ms(x.data_ptr(), srt[k].data_ptr(), w5.n_b, tmp.data_ptr(), tmp.numel(), 0, 32, 5, st)
          for k, x in enumerate((ps, pe))]
    out["cub_sort_cfg5_placed_2x1e7_keys"] = {"ms_both_arrays": sum(ms), "sort_keys_per_s": 2 * w5.n_b / (sum(ms) * 1e-3)}
    return out


def screen_workload(device, w, gather_gsectors=0.0, rounds=20):
    """The many-pair screen on synthetic tracks (w = config 2, whose B the tracks are drawn from)."""
    import torch
    from paper_1208_3407_b200 import bits
    # the paper's screen (159 tracks, 25,281 ordered pairs) on synthetic tracks of 1e5
    # intervals drawn from config 2's recipe, as ONE bits_screen call (every track sorted and indexed once, all pairs and
    # rounds in gridded launches); 20 of the paper's 10,000 rounds per pair, device time by CUDA events
    K, n_t, R_s = 159, 100_000, rounds
    rng = np.random.default_rng(8)
    idx = [rng.choice(w.n_b, n_t, replace=False) for _ in range(K)]
    starts = to_dev(np.concatenate([w.b_start[i] for i in idx]), device)
    ends = to_dev(np.concatenate([w.b_end[i] for i in idx]), device)
    toff = np.arange(K + 1, dtype=np.uint64) * n_t
    obs_s = torch.empty((K, K), dtype=torch.int64, device=device)
    rc_s = torch.empty((K, K, R_s), dtype=torch.int64, device=device)
    ws = torch.empty(int(bits.lib().bits_screen_workspace_bytes(toff.ctypes.data, K, 24)), dtype=torch.uint8, device=device)
    run = lambda R: bits.screen_concat(starts, ends, toff, w.chrom_offsets, 1, R, workspace=ws, observed_out=obs_s,
                                       round_counts_out=rc_s[:, :, :R].contiguous() if R != R_s else rc_s)
    launches0 = bits.launch_count()
    med0, _ = time_device(lambda: run(0), 2, warmup=1)               # setup + observed counts only
    med, mn = time_device(lambda: run(R_s), 2, warmup=1)
    per_call_launches = (bits.launch_count() - launches0) // 6
    enr = bits.screen_enrichment(obs_s.cpu().numpy().view(np.uint64), rc_s.cpu().numpy().view(np.uint64))
    rounds_ms = max(med - med0, 1e-6)
    sectors_per_interval = 6.0      # two index words + four key sectors per ICOUNT (search.cuh rank_le x 2)
    res = {
        "tracks": K, "pairs": K * K, "intervals_per_track": n_t, "rounds_per_pair": R_s, "ms_median": med, "ms_min": mn,
        "setup_and_observed_ms": med0, "launches_per_call": per_call_launches, "synchronisations_per_call": 1,
        "pair_rounds_per_s": K * K * R_s / (rounds_ms * 1e-3),
        "intervals_searched_per_s": K * K * R_s * n_t / (rounds_ms * 1e-3),
        "l2_sectors_per_s_model": K * K * R_s * n_t * sectors_per_interval / (rounds_ms * 1e-3),
        "paper_scale_estimate_s": {"pairs": K * K, "rounds": 10_000, "seconds": med0 * 1e-3 + rounds_ms * 1e-3 * 10_000 / R_s,
                                   "paper": "9,069 min on one GPU of 2012 for 25,281 pairs x 10,000 rounds of the ENCODE/UCSC "
                                            "tracks (PAPER.md:171; other data, other hardware: context only)"},
        "enrichment_diag_mean": float(np.mean(np.diag(enr))),
        "enrichment_offdiag_mean": float(np.mean(enr[~np.eye(K, dtype=bool)]))}
    # Sectors per interval come from the observed-count launch `screen_kernel<1>` (every pair once: K * K * n_t searched
    # intervals): ncu returns no counter values for the rounds launch `screen_kernel<0>` (profiles/r3_captures.md), which runs
    # the same two searches per interval against the same tracks after re-placing the queries.
    res["l2_roofline"] = l2_roofline("screen_kernel<1>", float(K) * K * n_t, K * K * R_s * n_t / (rounds_ms * 1e-3), gather_gsectors)
    res["l2_roofline"]["note"] = ("sectors per interval from the observed-count launch of the same call; rate from the rounds launch. frac can exceed 1: "
                                  "the yardstick gathers over 80 MB, a track's keys are 0.8 MB (better L1 / L2 locality)")
    return res



def secondary_workloads(device, peak_gbs, gather_gsectors=0.0):
    """The other throughputs BASELINE.json's metric names, on their own configs (not the timed headline)."""
    import torch
    from paper_1208_3407_b200 import bits
    from paper_1208_3407_b200 import workloads as W
    out = {}
    # config 4: 1e7 queries counted against 1e7 intervals (sort B once + per-interval search + reduce)
    w = W.make_config(4)
    d = [to_dev(x, device) for x in (w.a_start, w.a_end, w.b_start, w.b_end)]
    ws = torch.empty(bits.workspace_bytes(bits.FN_COUNT_PER_INTERVAL, w.n_a, w.n_b), dtype=torch.uint8, device=device)
    counts = torch.empty(w.n_a, dtype=torch.int32, device=device)
    total = torch.empty(1, dtype=torch.int64, device=device)
    med, mn = time_device(lambda: bits.count_per_interval(*d, workspace=ws, counts_out=counts, total_out=total), 10)
    bits.set_option("profile", 2); bits.set_option("profile", 1)          # per-kernel events in separate calls: they cost time
    calls = 5
    for _ in range(calls):
        bits.count_per_interval(*d, workspace=ws, counts_out=counts, total_out=total)
    torch.cuda.synchronize()
    prof = bits.profile_read(); bits.set_option("profile", 0)
    ms = {k: v[0] / calls for k, v in prof.items()}     # device ms per call and kernel class
    n, q = w.n_b, w.n_a
    # (the histogram and plan classes now hold two launches each: B's bins + plan, the queries' buckets + plan)
    sort_ms = ms["scatter"] + ms["bucket_sort"] + (ms["histogram"] + ms["plan"]) * (8 * n) / (8 * n + 4 * q)
    # algorithmic HBM bytes per call of every kernel class of this path and what that is of the peak
    alg = {"histogram": 8 * n + 4 * q, "scatter": 16 * n, "bucket_sort": 16 * n, "query_scatter": 20 * q, "bucket_search": 16 * q + 8 * n}
    out["cfg4_large_count_10M"] = {
        "intervals_searched_per_s": w.n_a / (med * 1e-3), "ms_median": med, "ms_min": mn,
        "sort_keys_per_s": 2 * w.n_b / (sort_ms * 1e-3) if sort_ms else None,
        "search_design": "queries binned by B's buckets, buckets searched out of shared memory (binned_count.cuh)" if ms.get("bucket_search") else "bucket index (search.cuh)",
        "kernel_ms": {k: v for k, v in ms.items() if v},
        "kernel_roofline": {k: {"algorithmic_bytes": b, "ms": ms[k], "achieved_gbs": b / (ms[k] * 1e-3) / 1e9,
                                "frac_of_hbm_peak": b / (ms[k] * 1e-3) / 1e9 / peak_gbs} for k, b in alg.items() if ms.get(k)},
        "hbm_bytes_model": 72 * w.n_b + 12 * w.n_a + 8 * w.n_b,
        "hbm_frac_of_peak": (72 * w.n_b + 12 * w.n_a + 8 * w.n_b) / (med * 1e-3) / 1e9 / peak_gbs,
        "hbm_bytes_this_design": sum(alg.values()),
        "hbm_frac_of_peak_this_design": sum(alg.values()) / (med * 1e-3) / 1e9 / peak_gbs,
        "note": "hbm_bytes_model is SURVEY 8(d)'s model of the unfused LSD path (920 MB); hbm_bytes_this_design is what this path must move",
    }
    # the same call with the round-1 search design (bucket index + count_kernel), beside it
    bits.set_option("count_binned", 0)
    try:
        med0, mn0 = time_device(lambda: bits.count_per_interval(*d, workspace=ws, counts_out=counts, total_out=total), 10)
    finally:
        bits.set_option("count_binned", -1)
    out["cfg4_large_count_10M"]["bucket_index_design"] = {"ms_median": med0, "ms_min": mn0, "intervals_searched_per_s": w.n_a / (med0 * 1e-3)}
    out["yardsticks"] = library_yardsticks(device, w, d)
    del d, ws, counts
    # config 3: 1e4 queries re-placed per round against a fixed 1e6-interval B, 10,000 rounds, fused kernel
    w = W.make_config(3)
    d = [to_dev(x, device) for x in (w.a_start, w.a_end, w.b_start, w.b_end)]
    ws = torch.empty(bits.workspace_bytes(bits.FN_MC_ROUNDS, w.n_a, w.n_b, 24, 0), dtype=torch.uint8, device=device)
    obs = torch.empty(1, dtype=torch.int64, device=device)
    rc = torch.empty(w.n_rounds, dtype=torch.int64, device=device)
    med, mn = time_device(lambda: bits.mc_rounds(*d, w.chrom_offsets, 0, w.mc_seed, 0, w.n_rounds, workspace=ws,
                                                 observed_out=obs, round_counts_out=rc), 5)
    out["cfg3_mc_permuteA_1e4x1M"] = {"mc_rounds_per_s": w.n_rounds / (med * 1e-3),
                                      "intervals_searched_per_s": w.n_rounds * w.n_a / (med * 1e-3),
                                      "ms_median": med, "ms_min": mn,
                                      "l2_roofline": l2_roofline("mc_permute_a_rounds_kernel", float(w.n_a) * min(w.n_rounds, 32768),
                                                                 w.n_rounds * w.n_a / (med * 1e-3), gather_gsectors)}
    # config 1 (1,000 x 1,000, one chromosome): Monte Carlo rounds of a set that fits one block's shared memory
    # (mc_small.cuh: one block per round), beside the two-launch path on the same rounds
    w = W.make_config(1)
    d1 = [to_dev(x, device) for x in (w.a_start, w.a_end, w.b_start, w.b_end)]
    R1 = 10_000
    ws1 = torch.empty(bits.workspace_bytes(bits.FN_MC_ROUNDS, w.n_a, w.n_b, 1, 1), dtype=torch.uint8, device=device)
    rc1 = torch.empty(R1, dtype=torch.int64, device=device)
    run1 = lambda: bits.mc_rounds(*d1, w.chrom_offsets, 1, w.mc_seed, 0, R1, workspace=ws1, observed_out=obs, round_counts_out=rc1)
    med, mn = time_device(run1, 5)
    ref1 = rc1.clone()
    bits.set_option("mc_small", 0)
    try:
        med2, _ = time_device(run1, 3, warmup=1)
    finally:
        bits.set_option("mc_small", 1)
    out["cfg1_tiny_permuteB_10000_rounds"] = {"mc_rounds_per_s": R1 / (med * 1e-3), "ms_median": med, "ms_min": mn,
                                              "two_launch_path_rounds_per_s": R1 / (med2 * 1e-3),
                                              "same_counts_as_two_launch_path": bool(torch.equal(ref1, rc1))}
    # a re-placed set that fits one block (6,000 intervals), a large A (1e6) and few rounds: round slicing / warm-up calls.
    # The one-block-per-round kernel would rank all of A on 4 SMs; the library takes the two-launch path instead.
    wf = W.make_config(5, scale=0.0006)
    wa = W.make_config(4, scale=0.1)
    dfr = [to_dev(x, device) for x in (wa.a_start, wa.a_end, wf.b_start, wf.b_end)]
    wsf = torch.empty(bits.workspace_bytes(bits.FN_MC_ROUNDS, wa.n_a, wf.n_b, 24, 1), dtype=torch.uint8, device=device)
    rcf = torch.empty(4, dtype=torch.int64, device=device)
    runf = lambda: bits.mc_rounds(*dfr, wf.chrom_offsets, 1, wf.mc_seed, 0, 4, workspace=wsf, observed_out=obs, round_counts_out=rcf)
    medf, _ = time_device(runf, 5)
    reff = rcf.clone()
    bits.set_option("mc_small", 2)
    try:
        medf2, _ = time_device(runf, 3, warmup=1)
    finally:
        bits.set_option("mc_small", 1)
    out["small_b_large_a_4_rounds"] = {"n_a": wa.n_a, "n_b": wf.n_b, "ms_median_call": medf, "one_block_per_round_ms_median_call": medf2,
                                       "same_counts": bool(torch.equal(reff, rcf))}
    del dfr, wsf
    # config 5's recipe at the smaller sizes of the paper's Table 1 (1e5 and 1e6 re-placed intervals):
    # one round does not fill the GPU there, so several rounds share a launch pair (gridDim.y = rounds)
    sizes = {}
    for scale in (0.01, 0.1):
        ws_ = W.make_config(5, scale=scale)
        ds = [to_dev(x, device) for x in (ws_.a_start, ws_.a_end, ws_.b_start, ws_.b_end)]
        Rm = 2000
        wsp = torch.empty(bits.workspace_bytes(bits.FN_MC_ROUNDS, ws_.n_a, ws_.n_b, 24, 1), dtype=torch.uint8, device=device)
        rcm = torch.empty(Rm, dtype=torch.int64, device=device)
        runm = lambda: bits.mc_rounds(*ds, ws_.chrom_offsets, 1, ws_.mc_seed, 0, Rm, workspace=wsp, observed_out=obs, round_counts_out=rcm)
        medm, _ = time_device(runm, 3, warmup=2)
        refm = rcm.clone()
        bits.set_option("mc_batch", 0)
        try:
            medm0, _ = time_device(runm, 2, warmup=1)
        finally:
            bits.set_option("mc_batch", 1)
        sizes[f"n_b_{ws_.n_b}_n_a_{ws_.n_a}"] = {"mc_rounds_per_s": Rm / (medm * 1e-3), "us_per_round": 1e3 * medm / Rm,
                                                 "sort_keys_per_s": 2 * ws_.n_b * Rm / (medm * 1e-3),
                                                 "one_round_per_launch_rounds_per_s": Rm / (medm0 * 1e-3),
                                                 "same_counts": bool(torch.equal(refm, rcm))}
        del ds, wsp
    out["cfg5_recipe_at_table1_sizes_2000_rounds"] = sizes
    # config 2: 1e6 x 1e6 count
    w = W.make_config(2)
    d = [to_dev(x, device) for x in (w.a_start, w.a_end, w.b_start, w.b_end)]
    ws = torch.empty(bits.workspace_bytes(bits.FN_COUNT_PER_INTERVAL, w.n_a, w.n_b), dtype=torch.uint8, device=device)
    med, mn = time_device(lambda: bits.count_per_interval(*d, workspace=ws), 10)
    out["cfg2_genome_count_1M"] = {"intervals_searched_per_s": w.n_a / (med * 1e-3), "ms_median": med, "ms_min": mn}
    # decision and enumeration on the same sets
    ws = torch.empty(bits.workspace_bytes(bits.FN_ENUMERATE, w.n_a, w.n_b), dtype=torch.uint8, device=device)
    n_pairs = bits.enumerate_pairs(*d, workspace=ws)[2]
    med, mn = time_device(lambda: bits.enumerate_pairs(*d, workspace=ws), 5)      # two calls inside: size, then emit
    out["cfg2_enumerate"] = {"pairs": n_pairs, "pairs_per_s": n_pairs / (med * 1e-3), "ms_median": med, "ms_min": mn}
    med, mn = time_device(lambda: bits.decide(*d, workspace=ws), 5)
    out["cfg2_decide"] = {"ms_median": med, "ms_min": mn}
    out["screen_159_tracks_of_1e5"] = screen_workload(device, w, gather_gsectors)
    return out


def run_b200(args):
    import torch
    import torch.distributed as dist
    from paper_1208_3407_b200 import bits
    from paper_1208_3407_b200 import workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)
    bits.lib()
    for kv in args.opt:
        name, _, val = kv.partition("=")
        bits.set_option(name, int(val))

    w = W.make_config(args.config, scale=args.scale)
    if w.which is None:
        return run_count_config(args, w, device, rank, world, dist)
    R = args.rounds or w.n_rounds
    from paper_1208_3407_b200 import shard
    r0, _ = shard.weak_slice(rank, R)                     # this rank's slice of the round space
    n_chrom = int(w.chrom_offsets.size - 1)
    d = [to_dev(x, device) for x in (w.a_start, w.a_end, w.b_start, w.b_end)]
    ws = torch.empty(bits.workspace_bytes(bits.FN_MC_ROUNDS, w.n_a, w.n_b, n_chrom, w.which), dtype=torch.uint8, device=device)
    obs = torch.empty(1, dtype=torch.int64, device=device)
    rc = torch.empty(R, dtype=torch.int64, device=device)

    def step():
        bits.mc_rounds(*d, w.chrom_offsets, w.which, w.mc_seed, r0, R, workspace=ws, observed_out=obs, round_counts_out=rc)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 0)):
        step()
    barrier()
    bits.set_option("profile", 0)                 # no per-kernel events inside the timed region
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = bits.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    barrier()
    elapsed_ms = ev0.elapsed_time(ev1)
    launches = bits.launch_count() - launches0
    # per-kernel durations: the same step repeated right behind the timed region (clocks still sampled),
    # every launch bracketed by CUDA events on the launching stream (they cost ~5 % of throughput,
    # which is why they stay out of `value`)
    profile_events = not args.no_profile_events
    prof_steps = min(args.steps, 2) if profile_events else 0
    bits.set_option("profile", 2)
    bits.set_option("profile", 1 if profile_events else 0)
    for _ in range(prof_steps):
        step()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    prof = bits.profile_read()
    bits.set_option("profile", 0)
    if world > 1:
        t = torch.tensor([elapsed_ms], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        elapsed_ms = float(t.item())
        lt = torch.tensor([launches], dtype=torch.int64, device=device)
        dist.all_reduce(lt, op=dist.ReduceOp.SUM)
        launches = int(lt.item())
    rounds_total = world * R * args.steps
    value = rounds_total / (elapsed_ms * 1e-3)

    # ---- roofline of the dominant kernel (the class with the largest share of the timed region) ----
    peak, peak_src = measured_peaks()
    n_sorted = w.n_b if w.which == 1 else 0
    n_p = w.n_b if w.which == 1 else w.n_a
    # algorithmic HBM bytes per launch of each kernel class: what the step must move
    alg = {
        "place": ("place_kernel", 12 * n_p),                                   # span in, two keys out
        "sort_pass": ("onesweep_pass_kernel", 2 * n_sorted * 8),               # two arrays x (read + write)
        "place_scatter": ("place_tile_kernel", 12 * n_p),                      # span in, (start, end) pair out
        "bucket_sort_search": ("bin_sort_search_kernel", 16 * n_sorted + 8 * w.n_a),   # pairs in, B_S and B_E out, sorted queries in
        "sorted_query": ("sorted_query_total_kernel", 8 * w.n_a),
        "mc_permute_a": ("mc_permute_a_kernel", 4 * w.n_a * min(R, 32768)),
    }
    roofline = None
    timed = {k: v for k, v in prof.items() if v[1] and v[0] > 0}
    if timed:
        tot = sum(v[0] for v in timed.values())
        dom = max((k for k in timed if k in alg), key=lambda k: timed[k][0], default=None)
        if dom is not None:
            kname, alg_bytes = alg[dom]
            launch_ms = timed[dom][0] / timed[dom][1]
            achieved = alg_bytes / (launch_ms * 1e-3) / 1e9
            counters, counters_note = ncu_counters() if (args.config == 5 and args.scale == 1.0 and not args.opt) else ({}, "not the captured workload")
            # (keys are kernel names with their template arguments; the one-round-per-launch instantiation `..., 0>` is the timed one)
            kc = kernel_counters(counters, kname)
            roofline = {"bound": "hbm", "kernel": kname, "achieved": achieved, "peak": peak, "unit": "GB/s",
                        "frac": achieved / peak,
                        "traffic": kc.get("dram_bytes"), "ncu_limiter": kc.get("limiter"), "ncu_counters": counters_note,
                        "peak_source": peak_src,
                        "avg_launch_ms": launch_ms, "launches_timed": timed[dom][1],
                        "algorithmic_bytes_per_launch": alg_bytes,
                        "kernel_ms_per_round": {k: v[0] / (R * prof_steps) for k, v in timed.items()},
                        "timed_in": f"{prof_steps} extra step(s) right behind the timed region, one event pair per launch",
                        "kernel_share_of_step": {k: v[0] / tot for k, v in timed.items()}}
            if kc.get("warp_instructions"):
                roofline["issue_slots"] = {"warp_instructions_per_launch": kc["warp_instructions"],
                                           "peak_per_s_formula": "148 SMs x 4 schedulers x sm_mhz (filled in below)"}
            if n_sorted:
                # what the two-launch design itself moves per round: the measured fraction of the round
                own = 12 * n_sorted + 16 * n_sorted + 8 * w.n_a
                roofline["round_hbm_bytes_this_design"] = own
                roofline["round_frac_of_peak_this_design"] = own * value / world / 1e9 / peak
                # SURVEY 8(d)'s per-round byte model of the UNFUSED path (place 12 M + one histogram read and four 8-bit
                # radix passes 72 M + search 8 N_q = 848 MB on config 5; 768 MB with the histogram fused into placement):
                # rounds/s times these bytes is a speed-up against that modelled design expressed in bandwidth units,
                # NOT bytes this implementation moves -- its kernels are bound by instruction issue, not by HBM
                survey = 12 * n_sorted + 72 * n_sorted + 8 * w.n_a
                roofline["round_hbm_bytes_model_survey"] = survey
                roofline["round_frac_of_peak_model_survey"] = survey * value / world / 1e9 / peak
                roofline["round_hbm_bytes_model_survey_hist_fused"] = survey - 8 * n_sorted
                roofline["round_frac_of_peak_model_survey_hist_fused"] = (survey - 8 * n_sorted) * value / world / 1e9 / peak
                roofline["round_frac_note"] = ("round_frac_of_peak_this_design is the measured fraction; the *_model_survey figures credit "
                                               "the passes the fused design does not make (SURVEY 8d: 'credit taken as >100 % of this model, "
                                               "model unchanged')")

    line = {
        "metric": "mc_rounds_per_s", "value": value, "unit": "rounds/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": elapsed_ms / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": config_block(w, R, world), "gpu_launches": launches,
        "intervals_searched_per_s": value * w.n_a,
        "sort_keys_per_s": (2 * n_sorted * value) if n_sorted else None,
        "profile_events_in_timed_region": False,
    }
    # the counts of the step that was timed against the oracle's golden per-round counts (full configs only)
    g_head, g_counts = golden_round_counts(args.config, w.mc_seed) if args.scale == 1.0 else (None, None)
    if g_head is not None and g_head.get("checksums") == w.checksums() and r0 + R <= g_counts.size:
        got = rc.cpu().numpy().view(np.uint64)
        line["golden_match"] = bool(np.array_equal(got, g_counts[r0:r0 + R]) and
                                    int(obs.cpu().numpy().view(np.uint64)[0]) == g_head["observed"])
        line["golden"] = {"file": f"tests/golden/cfg{args.config}_seed{w.mc_seed}_rounds.txt", "rounds_compared": R,
                          "round_begin": r0, "source": "CPU oracle over disjoint round slices (tests/golden/make_golden.py)"}
    else:
        line["golden_match"] = None
    if roofline:
        line["roofline"] = roofline
    if clocks is not None:
        line["clocks"] = clocks
    if roofline and "issue_slots" in roofline:
        mhz = (clocks or {}).get("sm_mhz") or (clocks or {}).get("sm_max_mhz")
        if mhz:
            iss = roofline["issue_slots"]
            iss.pop("peak_per_s_formula", None)
            iss["achieved_per_s"] = iss["warp_instructions_per_launch"] / (roofline["avg_launch_ms"] * 1e-3)
            iss["peak_per_s"] = N_SMS * SCHEDULERS_PER_SM * mhz * 1e6
            iss["frac"] = iss["achieved_per_s"] / iss["peak_per_s"]
            iss["note"] = ("share of the issue slots (148 SMs x 4 schedulers x sm_mhz) filled during the launch: instruction "
                           "count from the committed ncu capture, duration and clock measured in this run")
        else:
            del roofline["issue_slots"]

    # ---- end to end through the host-buffer entry point (H2D + run + D2H inside the timed region) ----
    if not args.no_extras:
        hp = [pinned(x) for x in (w.a_start, w.a_end, w.b_start, w.b_end)]
        hws = bits.host_workspace(bits.FN_MC_ROUNDS, w.n_a, w.n_b, n_chrom, w.which, R, device=device)
        rc_host_t = torch.empty(R, dtype=torch.int64).pin_memory()
        rc_host = rc_host_t.numpy().view(np.uint64)

        def e2e_step():
            return bits.mc_rounds_host(hp[0][1], hp[1][1], hp[2][1], hp[3][1], w.chrom_offsets, w.which, w.mc_seed,
                                       r0, R, workspace=hws, device=device, round_counts_out=rc_host)
        del ws
        for _ in range(min(args.warmup, 2)):
            e2e_step()
        barrier()
        e2e_steps = max(1, min(args.steps, 3))
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            res = e2e_step()
        torch.cuda.synchronize()
        t_e2e = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([t_e2e], dtype=torch.float64, device=device)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            t_e2e = float(t.item())
        line["e2e"] = {"value": world * R * e2e_steps / t_e2e, "unit": "rounds/s",
                       "h2d_bytes_per_step": 4 * 2 * (w.n_a + w.n_b) + 4 * (n_chrom + 1),
                       "d2h_bytes_per_step": 8 * R + 8, "steps": e2e_steps, "api": "bits_mc_rounds_host (pinned host buffers)",
                       "observed": res.observed, "p_enrich": res.p_enrich, "p_deplete": res.p_deplete}
        # the device-resident and host-buffer paths must agree bit for bit
        same = bool(np.array_equal(rc.cpu().numpy().view(np.uint64), rc_host))
        line["e2e"]["matches_device_path"] = same
        del hws, hp

    if rank == 0 and world == 1 and not args.no_extras:
        line["l2_yardsticks"] = l2_yardsticks(device)
        line["other_workloads"] = secondary_workloads(device, peak, line["l2_yardsticks"]["l2_random_sector_gather_gsectors_per_s_80MB"])
        if w.which == 1:
            # SURVEY 8(f).1, reported BESIDE the headline: the sort-free variant of the same rounds
            # (count(A, B') = count(B', A): fresh B intervals searched against the once-sorted A; no B_S / B_E)
            Rs = min(R, 200)
            ws2 = torch.empty(bits.workspace_bytes(bits.FN_MC_ROUNDS, w.n_a, w.n_b, n_chrom, w.which), dtype=torch.uint8, device=device)
            rc2 = torch.empty(Rs, dtype=torch.int64, device=device)
            bits.set_option("mc_symmetric", 1)
            try:
                med, mn = time_device(lambda: bits.mc_rounds(*d, w.chrom_offsets, w.which, w.mc_seed, r0, Rs, workspace=ws2,
                                                             observed_out=obs, round_counts_out=rc2), 3, warmup=1)
            finally:
                bits.set_option("mc_symmetric", 0)
            # the literal path (general placement kernel -> MSD sort of both arrays -> bucket index -> one ICOUNT per query),
            # beside the headline: same integers, no fused kernels, no sorted queries
            Rl = min(R, 20)
            rc3 = torch.empty(Rl, dtype=torch.int64, device=device)
            bits.set_option("mc_fused", 0); bits.set_option("mc_sorted_queries", 0)
            try:
                medl, _ = time_device(lambda: bits.mc_rounds(*d, w.chrom_offsets, w.which, w.mc_seed, r0, Rl, workspace=ws2,
                                                             observed_out=obs, round_counts_out=rc3), 3, warmup=1)
            finally:
                bits.set_option("mc_fused", 1); bits.set_option("mc_sorted_queries", 1)
            line["other_workloads"]["cfg5_literal_path"] = {
                "mc_rounds_per_s": Rl / (medl * 1e-3), "rounds_per_call": Rl, "ms_median": medl,
                "path": "place_kernel -> MSD sort of B_S and B_E -> bucket index -> count_kernel (one ICOUNT per query), per round",
                "same_counts_as_headline_path": bool(torch.equal(rc3, rc[:Rl]))}
            line["other_workloads"]["cfg5_symmetric_sort_free"] = {
                "mc_rounds_per_s": Rs / (med * 1e-3), "rounds_per_call": Rs, "ms_median": med,
                "intervals_searched_per_s": Rs * w.n_b / (med * 1e-3),
                "same_counts_as_headline_path": bool(torch.equal(rc2, rc[:Rs]))}
            del ws2
        n_cpu = 2 if args.config == 5 else 50
        rps, t_obs, t_r = oracle_marginal_rounds_per_s(w, w.which, 0, n_cpu)
        line["cpu_baseline"] = {"value": rps, "unit": "rounds/s", "cores": 1, "kind": "oracle",
                                "sample": oracle_sample_text(n_cpu, w), "observed_count_s": t_obs,
                                "host_cores": os.cpu_count()}
        # the oracle on the other configs: counting configs in full, config 3 on 100 of its rounds
        import oracle
        other = {}
        for k in (2, 4):
            wk = W.make_config(k)
            t0 = time.perf_counter(); oracle.count_per_interval(wk.a_start, wk.a_end, wk.b_start, wk.b_end); dt = time.perf_counter() - t0
            other[wk.name] = {"seconds": dt, "intervals_searched_per_s": wk.n_a / dt, "sample": "the whole call: std::sort of both key arrays + one ICOUNT per query"}
        w3 = W.make_config(3)
        rps3, _, _ = oracle_marginal_rounds_per_s(w3, 0, 0, 100)
        other[w3.name] = {"rounds_per_s": rps3, "intervals_searched_per_s": rps3 * w3.n_a, "sample": "100 of its 10,000 rounds (marginal cost per round)"}
        line["cpu_baseline"]["other_configs"] = other
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_study(args):
    """Design studies of the count path (north_star subsystem 3: try several search designs and keep what ncu
    supports).  Prints one JSON line; per-kernel device times come from the library's event timers."""
    import torch
    from paper_1208_3407_b200 import bits
    from paper_1208_3407_b200 import workloads as W
    device = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    for kv in args.opt:
        name, _, val = kv.partition("=")
        bits.set_option(name, int(val))
    if args.study == "screen":      # the screen alone (one JSON object): the command the ncu capture of scr::screen_kernel runs
        gather = 0.0 if args.once else l2_yardsticks(device)["l2_random_sector_gather_gsectors_per_s_80MB"]
        print(json.dumps({"study": "screen", "screen_159_tracks_of_1e5": screen_workload(device, W.make_config(2), gather, args.rounds or 20)}))
        return 0
    reps = 1 if args.once else 8
    w = W.make_config(4, scale=args.scale)
    d = [to_dev(x, device) for x in (w.a_start, w.a_end, w.b_start, w.b_end)]
    bits.set_option("count_binned", 1)                     # (sized for the design that needs the most: the query lists)
    ws = torch.empty(bits.workspace_bytes(bits.FN_COUNT_PER_INTERVAL, w.n_a, w.n_b), dtype=torch.uint8, device=device)
    bits.set_option("count_binned", -1)
    counts = torch.empty(w.n_a, dtype=torch.int32, device=device)
    total = torch.empty(1, dtype=torch.int64, device=device)
    out = {"study": args.study, "workload": w.name, "n_a": w.n_a, "n_b": w.n_b, "calls_per_design": reps, "designs": {}}

    def one_design(label):
        if not args.once:
            for _ in range(2):
                bits.count_per_interval(*d, workspace=ws, counts_out=counts, total_out=total)
            med, mn = time_device(lambda: bits.count_per_interval(*d, workspace=ws, counts_out=counts, total_out=total), reps, warmup=0)
        bits.set_option("profile", 2); bits.set_option("profile", 1)
        for _ in range(reps):
            bits.count_per_interval(*d, workspace=ws, counts_out=counts, total_out=total)
        torch.cuda.synchronize()
        prof = bits.profile_read(); bits.set_option("profile", 0)
        r = {"kernel_us": {k: 1e3 * v[0] / reps for k, v in prof.items() if v[1]},
             "total": int(total.cpu().numpy().view(np.uint64)[0])}
        if not args.once:
            r["call_ms_median"], r["call_ms_min"] = med, mn
            r["intervals_searched_per_s"] = w.n_a / (med * 1e-3)
        out["designs"][label] = r

    if args.study == "count":
        one_design("default")
    else:
        bits.set_option("count_binned", 0)                 # the three designs of count_kernel over the sorted arrays in global memory ...
        for v, name in SEARCH_DESIGNS:
            bits.set_option("search_variant", v)
            one_design(f"{v}: {name}")
        bits.set_option("search_variant", 0)
        bits.set_option("count_binned", 1)                 # ... and the queries binned by B's buckets, buckets searched out of shared memory
        one_design("3: queries binned by B's buckets, shared-memory search (binned_count.cuh) [default at this size]")
        bits.set_option("count_binned", -1)
        w3 = W.make_config(3, scale=args.scale)
        d3 = [to_dev(x, device) for x in (w3.a_start, w3.a_end, w3.b_start, w3.b_end)]
        R = 100
        bits.set_option("profile", 2); bits.set_option("profile", 1)
        for _ in range(reps):
            bits.mc_rounds(*d3, w3.chrom_offsets, 0, 1, 0, R)
        torch.cuda.synchronize()
        prof = bits.profile_read(); bits.set_option("profile", 0)
        us = 1e3 * prof["mc_permute_a"][0] / prof["mc_permute_a"][1]
        out["cfg3_mc_permute_a_100_rounds_per_launch"] = {"kernel_us": us, "intervals_searched_per_s": R * w3.n_a / (us * 1e-6)}
    print(json.dumps(out))
    return 0


def run_count_config(args, w, device, rank, world, dist):
    """`--config 2|4`: the counting configs as a full bench line.  A step is ONE bits_count_per_interval call (sort B_S and
    B_E, two ranks per query, per-interval counts written, total reduced; Algorithm 2) on inputs resident
    in HBM; metric intervals_searched_per_s.  With N > 1 every rank runs the same call (replicas, no collective)."""
    import torch
    from paper_1208_3407_b200 import bits
    peak, peak_src = measured_peaks()
    n, q = w.n_b, w.n_a
    d = [to_dev(x, device) for x in (w.a_start, w.a_end, w.b_start, w.b_end)]
    ws = torch.empty(bits.workspace_bytes(bits.FN_COUNT_PER_INTERVAL, q, n), dtype=torch.uint8, device=device)
    counts = torch.empty(q, dtype=torch.int32, device=device)
    total = torch.empty(1, dtype=torch.int64, device=device)
    step = lambda: bits.count_per_interval(*d, workspace=ws, counts_out=counts, total_out=total)
    # L2: a step reads 8 (n + q) bytes of input and writes 4 q; below twice the 126 MB L2 the cache is flushed between steps
    # (a 256 MB fill outside the per-step event pairs), above it the inputs evict themselves
    footprint = 8 * (n + q) + 4 * q
    flush = footprint < 2 * 126 * 2**20
    junk = torch.empty(256 << 20, dtype=torch.uint8, device=device) if flush else None

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed_steps(k):
        ms = 0.0
        for _ in range(k):
            if flush:
                junk.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); step(); b.record(); b.synchronize()
            ms += a.elapsed_time(b)
        return ms

    for _ in range(max(args.warmup, 0)):
        step()
    barrier()
    bits.set_option("profile", 0)
    sampler = ClockSampler(int(os.environ.get("LOCAL_RANK", "0")))
    if rank == 0:
        sampler.start()
    launches0 = bits.launch_count()
    barrier()
    elapsed_ms = timed_steps(args.steps)
    barrier()
    launches = bits.launch_count() - launches0
    # per-kernel durations right behind the timed region (event pairs cost time, so they stay out of `value`)
    prof_steps = max(1, min(args.steps, 5))
    bits.set_option("profile", 2); bits.set_option("profile", 1)
    for _ in range(prof_steps):
        if flush:
            junk.fill_(1)
        step()
    barrier()
    prof = bits.profile_read(); bits.set_option("profile", 0)
    # a short timed region gives nvidia-smi (100 ms period) nothing to sample: keep the GPU on the same step until it has
    t_end = time.perf_counter() + 0.6
    while rank == 0 and time.perf_counter() < t_end:
        step()
    torch.cuda.synchronize()
    clocks = sampler.stop() if rank == 0 else None
    if world > 1:
        t = torch.tensor([elapsed_ms], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        elapsed_ms = float(t.item())
        lt = torch.tensor([launches], dtype=torch.int64, device=device)
        dist.all_reduce(lt, op=dist.ReduceOp.SUM)
        launches = int(lt.item())
    value = world * q * args.steps / (elapsed_ms * 1e-3)
    ms = {k: v[0] / prof_steps for k, v in prof.items() if v[1]}
    binned = bool(ms.get("bucket_search"))
    # algorithmic HBM bytes per call of every kernel class
    alg = {"histogram": 8 * n + (4 * q if binned else 0), "scatter": 16 * n, "bucket_sort": 16 * n,
           "query_scatter": 20 * q, "bucket_search": 16 * q + 8 * n, "index_build": 8 * n, "count": 12 * q}
    if binned:      # (the index and count launches behind the binned design are gated fallbacks that exit at once)
        alg.pop("index_build"); alg.pop("count")
    alg = {k: b for k, b in alg.items() if ms.get(k)}
    dom = max(alg, key=lambda k: ms[k])
    own = sum(alg.values())
    survey = 72 * n + 8 * n + 12 * q           # histogram read + four LSD passes over both arrays, queries in, counts out
    line = {
        "metric": "intervals_searched_per_s", "value": value, "unit": "intervals/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": elapsed_ms / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": w.name, "n_a": q, "n_b": n, "data_seed": w.spec.get("seed"), "scale": w.spec.get("scale", 1.0),
                   "step": "one bits_count_per_interval call: sort B_S and B_E, two ranks per query, counts written, total reduced",
                   "search_design": "queries binned by B's buckets (binned_count.cuh)" if binned else "bucket index (search.cuh)",
                   "parallelism": f"{world} replica(s), no collective",
                   "l2": ("flushed between steps: a 256 MB fill outside each step's event pair (the step's footprint, "
                          f"{footprint / 1e6:.0f} MB, would otherwise stay in the 126 MB L2)") if flush else
                         f"no flush: a step's footprint ({footprint / 1e6:.0f} MB) is larger than the 126 MB L2"},
        "gpu_launches": launches, "sort_keys_per_s": None, "profile_events_in_timed_region": False,
        "roofline": {"bound": "hbm", "kernel": {"histogram": "bin_hist_kernel", "scatter": "scatter_kernel", "bucket_sort": "bucket_sort_kernel",
                                                "query_scatter": "query_scatter_kernel", "bucket_search": "bucket_search_kernel",
                                                "index_build": "build_index_kernel", "count": "count_kernel"}[dom],
                     "achieved": alg[dom] / (ms[dom] * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                     "frac": alg[dom] / (ms[dom] * 1e-3) / 1e9 / peak, "traffic": None, "peak_source": peak_src,
                     "avg_launch_ms": ms[dom], "algorithmic_bytes_per_launch": alg[dom],
                     "timed_in": f"{prof_steps} extra step(s) right behind the timed region, one event pair per launch",
                     "kernel_ms_per_step": ms,
                     "kernel_roofline": {k: {"algorithmic_bytes": b, "ms": ms[k], "frac_of_hbm_peak": b / (ms[k] * 1e-3) / 1e9 / peak}
                                         for k, b in alg.items()},
                     "step_hbm_bytes_this_design": own,
                     "step_frac_of_peak_this_design": own * value / world / q / 1e9 / peak,
                     "step_hbm_bytes_model_survey": survey,
                     "step_frac_of_peak_model_survey": survey * value / world / q / 1e9 / peak},
        "clocks": clocks,
    }
    if not args.no_extras:
        # end to end: host arrays in pinned memory -> bits_count_per_interval_host -> counts and total back on the host
        hp = [pinned(x) for x in (w.a_start, w.a_end, w.b_start, w.b_end)]
        hws = bits.host_workspace(bits.FN_COUNT_PER_INTERVAL, q, n, device=device)
        counts_host_t = torch.empty(q, dtype=torch.int32).pin_memory()
        counts_host = counts_host_t.numpy().view(np.uint32)
        e2e_step = lambda: bits.count_per_interval_host(hp[0][1], hp[1][1], hp[2][1], hp[3][1], workspace=hws, device=device,
                                                        counts_out=counts_host)
        for _ in range(2):
            e2e_step()
        barrier()
        e2e_steps = max(1, min(args.steps, 5))
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            res = e2e_step()
        torch.cuda.synchronize()
        t_e2e = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([t_e2e], dtype=torch.float64, device=device)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            t_e2e = float(t.item())
        h_counts, h_total = res
        line["e2e"] = {"value": world * q * e2e_steps / t_e2e, "unit": "intervals/s",
                       "h2d_bytes_per_step": 4 * (2 * q + 2 * n), "d2h_bytes_per_step": 4 * q + 8, "steps": e2e_steps,
                       "api": "bits_count_per_interval_host (pinned host buffers)",
                       "matches_device_path": bool(np.array_equal(np.asarray(h_counts).view(np.uint32), counts.cpu().numpy().view(np.uint32))
                                                   and int(h_total) == int(total.cpu().numpy().view(np.uint64)[0]))}
        if rank == 0:
            import oracle
            t0 = time.perf_counter(); o_total, o_counts = oracle.count_per_interval(w.a_start, w.a_end, w.b_start, w.b_end); dt = time.perf_counter() - t0
            line["cpu_baseline"] = {"value": q / dt, "unit": "intervals/s", "cores": 1, "kind": "oracle", "host_cores": os.cpu_count(),
                                    "sample": f"the whole call once ({dt:.2f} s): std::sort of both key arrays of B + one ICOUNT per query + sum"}
            line["oracle_match"] = bool(int(total.cpu().numpy().view(np.uint64)[0]) == o_total and
                                        np.array_equal(counts.cpu().numpy().view(np.uint32), o_counts))
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


# search designs of the count path (bits_set_option "search_variant")
SEARCH_DESIGNS = ((0, "bucket index"), (1, "plain binary search (the paper's design)"), (2, "top 11 levels in shared memory"))


def main():
    args = parse_args()
    if args.study:
        return run_study(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())
