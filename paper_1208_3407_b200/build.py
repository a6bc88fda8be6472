"""Build libbits_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1208_3407_b200.build [--force]
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libbits_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "static",
]


# Every source a captured kernel's ncu counters depend on: the kernel headers AND the host orchestration, whose launch
# geometry (tile size, bin width, grid, rounds per launch, knob defaults) changes DRAM bytes, durations and limiters
# just as a kernel edit does.
HASHED_SOURCES = ("binned_count.cuh", "bits_api.cu", "common.cuh", "enumerate.cuh", "mc_small.cuh", "mc_tile.cuh", "msd_sort.cuh",
                  "philox_place.cuh", "place_kernels.cuh", "radix_sort.cuh", "screen.cuh", "search.cuh")


def csrc_hash() -> str:
    """sha256 over HASHED_SOURCES (all of csrc/): identifies the build whose ncu counters a profiles/*_ncu_counters.json
    holds.  Written into that file by ncu_counters.py at capture time, compared by bench.py at run time."""
    import hashlib
    h = hashlib.sha256()
    for path in [os.path.join(CSRC, f) for f in HASHED_SOURCES]:
        h.update(os.path.basename(path).encode())
        with open(path, "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def sources() -> list[str]:
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps() -> list[str]:
    return sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "bits.h")]


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/*.cu into libbits_b200.so if it is missing or older than a source."""
    if not force and os.path.exists(LIB):
        t = os.path.getmtime(LIB)
        if all(os.path.getmtime(d) <= t for d in _deps()):
            return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = [NVCC, *FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", tmp, *sources()]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


PROBE_SRC = os.path.join(HERE, "probe", "l2_probe.cu")
PROBE_LIB = os.path.join(HERE, "probe", "libl2_probe.so")


def build_probe(force: bool = False) -> str:
    """Compile the bench-only L2 yardstick (probe/l2_probe.cu); it is not linked into libbits_b200.so."""
    if not force and os.path.exists(PROBE_LIB) and os.path.getmtime(PROBE_SRC) <= os.path.getmtime(PROBE_LIB):
        return PROBE_LIB
    tmp = PROBE_LIB + f".tmp{os.getpid()}"
    subprocess.check_call([NVCC, *FLAGS, "-o", tmp, PROBE_SRC])
    os.replace(tmp, PROBE_LIB)
    return PROBE_LIB


YARD_SRC = os.path.join(HERE, "probe", "yardsticks.cu")
YARD_LIB = os.path.join(HERE, "probe", "libyardsticks.so")


def build_yardsticks(force: bool = False) -> str:
    """Compile the bench-only CUB / thrust yardsticks (probe/yardsticks.cu); never linked into libbits_b200.so."""
    if not force and os.path.exists(YARD_LIB) and os.path.getmtime(YARD_SRC) <= os.path.getmtime(YARD_LIB):
        return YARD_LIB
    tmp = YARD_LIB + f".tmp{os.getpid()}"
    subprocess.check_call([NVCC, *FLAGS, "-o", tmp, YARD_SRC])
    os.replace(tmp, YARD_LIB)
    return YARD_LIB


if __name__ == "__main__":
    build_probe(force="--force" in sys.argv)
    build_yardsticks(force="--force" in sys.argv)
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    if "--hash" in sys.argv:
        print(csrc_hash())
