"""Command line shaped like BITS-SEQ / BITS-CUDA:

    python -m paper_1208_3407_b200.cli count        -a A.bed -b B.bed -g genome.txt
    python -m paper_1208_3407_b200.cli per-interval -a A.bed -b B.bed -g genome.txt     # one count per line of A
    python -m paper_1208_3407_b200.cli decide       -a A.bed -b B.bed -g genome.txt
    python -m paper_1208_3407_b200.cli enumerate    -a A.bed -b B.bed -g genome.txt     # "line_in_A<TAB>line_in_B" pairs (0-based)
    python -m paper_1208_3407_b200.cli mc           -a A.bed -b B.bed -g genome.txt -n 10000 [--permute b] [--seed 1]

The genome file gives `name length` per chromosome in projection order.  Needs a CUDA device: there is no
CPU fallback.  File handling is in frontend.py; every number printed comes from the library's kernels.
"""
from __future__ import annotations

import argparse
import sys

import numpy as np


def _parser():
    p = argparse.ArgumentParser(prog="python -m paper_1208_3407_b200.cli", description=__doc__.split("\n")[0])
    p.add_argument("command", choices=["count", "per-interval", "decide", "enumerate", "mc"])
    p.add_argument("-a", required=True, help="query intervals (BED)")
    p.add_argument("-b", required=True, help="database intervals (BED)")
    p.add_argument("-g", required=True, help="genome file: name length per line")
    p.add_argument("-n", type=int, default=1000, help="Monte Carlo rounds (mc)")
    p.add_argument("--permute", choices=["a", "b"], default="a", help="which set is re-placed every round (mc)")
    p.add_argument("--seed", type=int, default=1)
    p.add_argument("--skip-unknown", action="store_true", help="skip BED lines on chromosomes the genome file does not list")
    p.add_argument("--device", default="cuda:0")
    return p


def main(argv=None) -> int:
    args = _parser().parse_args(argv)
    from . import frontend as F
    try:
        genome = F.read_genome(args.g)
        a_s, a_e = F.read_bed(args.a, genome, args.skip_unknown)
        b_s, b_e = F.read_bed(args.b, genome, args.skip_unknown)
    except (F.FrontEndError, OSError) as e:
        print(f"error: {e}", file=sys.stderr)
        return 2
    import torch
    from . import bits
    if not torch.cuda.is_available():
        print("error: no CUDA device (this library has no CPU fallback)", file=sys.stderr)
        return 3
    dev = lambda x: torch.from_numpy(x.view(np.int32)).to(args.device)
    d = [dev(x) for x in (a_s, a_e, b_s, b_e)]
    if args.command == "count":
        t = bits.count(*d)
        torch.cuda.synchronize()
        print(int(t.cpu().numpy().view(np.uint64)[0]))
    elif args.command == "per-interval":
        counts, _ = bits.count_per_interval(*d)
        torch.cuda.synchronize()
        sys.stdout.write("\n".join(map(str, counts.cpu().numpy().view(np.uint32).tolist())) + ("\n" if a_s.size else ""))
    elif args.command == "decide":
        t = bits.decide(*d)
        torch.cuda.synchronize()
        print(int(t.cpu().numpy()[0]))
    elif args.command == "enumerate":
        pa, pb, n = bits.enumerate_pairs(*d)
        torch.cuda.synchronize()
        pa, pb = pa.cpu().numpy().view(np.uint32), pb.cpu().numpy().view(np.uint32)
        sys.stdout.write("".join(f"{i}\t{j}\n" for i, j in zip(pa.tolist(), pb.tolist())))
    else:
        which = bits.PERMUTE_A if args.permute == "a" else bits.PERMUTE_B
        obs, rc = bits.mc_rounds(*d, genome.offsets, which, args.seed, 0, args.n)
        torch.cuda.synchronize()
        o = int(obs.cpu().numpy().view(np.uint64)[0])
        r = rc.cpu().numpy().view(np.uint64)
        print(f"observed\t{o}")
        print(f"rounds\t{args.n}")
        print(f"median\t{float(np.median(r)) if r.size else float('nan')}")
        print(f"log2_observed_over_median\t{bits.enrichment(o, r)}")
        print(f"p_enrichment\t{bits.pvalue(o, r, 0)}")
        print(f"p_depletion\t{bits.pvalue(o, r, 1)}")
    return 0


if __name__ == "__main__":
    sys.exit(main())
