"""Search design study (north_star: try several search designs and keep what ncu supports).

    python -m paper_1208_3407_b200.probe.search_study            # times the variants with CUDA events
    ncu --metrics ... -k regex:'count_kernel|mc_permute_a_kernel' python -m paper_1208_3407_b200.probe.search_study --once

Runs config 4 (10M queries against 10M intervals, per-interval counts) with the three search designs of
count_kernel (bits_set_option "search_variant": 0 bucket index, 1 plain binary search, 2 top 11 levels in
shared memory) and 100 rounds of config 3 (mc_permute_a_kernel, bucket index).  Bench-only code.
"""
import sys

import numpy as np
import torch

from paper_1208_3407_b200 import bits
from paper_1208_3407_b200 import workloads as W


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.uint32).view(np.int32)).cuda()


def main():
    once = "--once" in sys.argv
    reps = 1 if once else 8
    w = W.make_config(4)
    d = [dev(x) for x in (w.a_start, w.a_end, w.b_start, w.b_end)]
    ws = torch.empty(bits.workspace_bytes(bits.FN_COUNT_PER_INTERVAL, w.n_a, w.n_b), dtype=torch.uint8, device="cuda")
    counts = torch.empty(w.n_a, dtype=torch.int32, device="cuda")
    total = torch.empty(1, dtype=torch.int64, device="cuda")
    for v, name in ((0, "bucket index"), (1, "plain binary search"), (2, "top 11 levels in shared memory")):
        bits.set_option("search_variant", v)
        bits.set_option("profile", 2)
        bits.set_option("profile", 1)
        for _ in range(reps):
            bits.count_per_interval(*d, workspace=ws, counts_out=counts, total_out=total)
        torch.cuda.synchronize()
        p = bits.profile_read()
        bits.set_option("profile", 0)
        us = 1e3 * p["count"][0] / p["count"][1]
        print(f"cfg4 count_kernel variant {v} ({name}): {us:.1f} us, {w.n_a / us * 1e-3:.2f} G intervals/s, "
              f"total {int(total.cpu().numpy().view(np.uint64)[0])}")
    bits.set_option("search_variant", 0)
    w = W.make_config(3)
    d = [dev(x) for x in (w.a_start, w.a_end, w.b_start, w.b_end)]
    R = 100
    bits.set_option("profile", 2)
    bits.set_option("profile", 1)
    for _ in range(reps):
        obs, rc = bits.mc_rounds(*d, w.chrom_offsets, 0, 1, 0, R)
    torch.cuda.synchronize()
    p = bits.profile_read()
    bits.set_option("profile", 0)
    us = 1e3 * p["mc_permute_a"][0] / p["mc_permute_a"][1]
    print(f"cfg3 mc_permute_a_kernel, {R} rounds per launch: {us:.1f} us, {R * w.n_a / us * 1e-3:.2f} G intervals/s")


if __name__ == "__main__":
    main()
