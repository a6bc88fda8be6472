#!/usr/bin/env python
"""Writes the golden per-round Monte Carlo counts of configs 3 and 5 (tests/golden/cfg{3,5}_seed1_rounds.txt).

    python tests/golden/make_golden.py [--config 3 5] [--workers 6] [--slice 25]

Every number comes from the CPU oracle (oracle/bits_oracle.cpp: the Monte Carlo loop of PAPER.md:157-159
as SURVEY.md section 8(c) steps 1-5 spell it out) on the seeded inputs of
paper_1208_3407_b200/workloads.py -- nothing here imports, calls or reads the CUDA path.  Rounds are
addressed by (seed, round), so the job is cut into disjoint round slices that run in separate
processes, each still the single-threaded oracle; the observed count every slice recomputes must agree.

File format: '#' lines, one of which is a JSON header (config, seeds, sizes, input checksums from
workloads.array_checksum, observed count, p-values from oracle.pvalue), then one round count per line
in round order (round r on data line r).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time
from concurrent.futures import ProcessPoolExecutor

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle                                            # noqa: E402
from paper_1208_3407_b200 import workloads as W          # noqa: E402  (input generators only)

_W = None   # the workload, inherited by the forked workers


def golden_path(config: int, mc_seed: int = 1) -> str:
    return os.path.join(HERE, f"cfg{config}_seed{mc_seed}_rounds.txt")


def _slice(job):
    r0, n = job
    w = _W
    obs, rc = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, w.which, w.mc_seed, r0, n)
    return r0, n, obs, rc


def make(config: int, workers: int, slice_rounds: int) -> str:
    global _W
    oracle.build()
    t0 = time.time()
    _W = w = W.make_config(config)
    R = w.n_rounds
    jobs = [(r0, min(slice_rounds, R - r0)) for r0 in range(0, R, slice_rounds)]
    counts = np.zeros(R, dtype=np.uint64)
    observed = None
    with ProcessPoolExecutor(max_workers=workers) as pool:      # fork: the arrays are shared copy-on-write
        for r0, n, obs, rc in pool.map(_slice, jobs):
            if observed is None:
                observed = obs
            assert obs == observed, "slices disagree on the observed count"
            counts[r0:r0 + n] = rc
    header = {
        "config": config, "workload": w.name, "which": w.which, "mc_seed": w.mc_seed, "data_seed": w.spec["seed"],
        "n_a": w.n_a, "n_b": w.n_b, "n_rounds": R, "round_begin": 0, "observed": int(observed),
        "checksums": w.checksums(), "chrom_offsets_checksum": W.array_checksum(w.chrom_offsets),
        "p_enrich": oracle.pvalue(observed, counts, 0), "p_deplete": oracle.pvalue(observed, counts, 1),
        "slices": len(jobs), "rounds_per_slice": slice_rounds,
    }
    path = golden_path(config, w.mc_seed)
    with open(path, "w") as f:
        f.write(f"# Golden per-round Monte Carlo counts of BASELINE.json configs[{config - 1}] ({w.name}), written by\n")
        f.write("# tests/golden/make_golden.py from the CPU oracle alone (oracle.mc_rounds over disjoint round slices;\n")
        f.write("# PAPER.md:157-159, procedure of SURVEY.md section 8(c)).  The paper prints no counts: these pin the CUDA\n")
        f.write("# path to the oracle over the FULL round range, not the oracle to the paper.  Data line r = round r.\n")
        f.write("# " + json.dumps(header) + "\n")
        for c in counts:
            f.write(f"{int(c)}\n")
    print(f"config {config}: {R} rounds in {time.time() - t0:.1f} s -> {path}", flush=True)
    return path


def load(config: int, mc_seed: int = 1):
    """-> (header dict, uint64[n_rounds]) from the committed file (used by tests/ and bench.py)."""
    header, vals = None, []
    with open(golden_path(config, mc_seed)) as f:
        for line in f:
            line = line.strip()
            if not line:
                continue
            if line.startswith("#"):
                body = line[1:].strip()
                if body.startswith("{"):
                    header = json.loads(body)
                continue
            vals.append(int(line))
    return header, np.array(vals, dtype=np.uint64)


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, nargs="+", default=[3, 5], choices=[1, 3, 5])
    ap.add_argument("--workers", type=int, default=max(1, (os.cpu_count() or 2) - 2))
    ap.add_argument("--slice", type=int, default=0, help="rounds per slice (0: 25 for config 5, 500 otherwise)")
    a = ap.parse_args()
    for k in a.config:
        make(k, a.workers, a.slice or (25 if k == 5 else 500))
