"""bits_count_static: the counting call for callers that cannot allocate device memory.

Who needs it: code that is handed its device buffers by somebody else and may not create any of its own -- a
stage inside an application that owns the whole device-memory pool, a latency-critical path on which cudaMalloc is
banned because it synchronises the device, a GPU whose memory another framework has already claimed.  For them the
library carries its scratch inside its own device image (32 MiB, include/bits.h BITS_STATIC_SCRATCH_BYTES) and the
call takes inputs and the output only.

What is checked: the new entry point returns the same integer as the existing workspace path (bits_count) -- the
path is integer-only, so the tolerance is zero as everywhere in tests/test_parity_gpu.py -- on calls made one after
the other, so that the second call starts on whatever the first left in the shared array; that device memory in use
does not grow across such calls; and that a problem beyond the limit is refused instead of truncated.

This file sorts last on purpose (pytest -x stops at the first failure; nothing should hide behind this one).  It must
pass both on its own in a fresh process (the first call does the per-device set-up) and after the other GPU tests.
"""
import numpy as np
import pytest
import torch

from paper_1208_3407_b200 import bits
from paper_1208_3407_b200 import workloads as W

DEV = "cuda:0"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.uint32).view(np.int32)).to(DEV)


def u64(t):
    return int(t.cpu().numpy().view(np.uint64)[0])


def _ragged_case(seed, n_a, n_b, genome=3_000_000_000, max_len=5_000):
    rng = np.random.default_rng(seed)
    a_s = rng.integers(0, genome - max_len, n_a, dtype=np.uint64).astype(np.uint32)
    b_s = rng.integers(0, genome - max_len, n_b, dtype=np.uint64).astype(np.uint32)
    a_e = a_s + rng.integers(0, max_len, n_a).astype(np.uint32)
    b_e = b_s + rng.integers(0, max_len, n_b).astype(np.uint32)
    return a_s, a_e, b_s, b_e


def test_limit_and_argument_errors_are_reported_on_the_host():
    """No GPU needed: sizes and pointers are checked before the first CUDA call."""
    L = bits.lib()
    # the limit is the size of the workspace bits_count would ask for: about 19 bytes per interval of B
    assert bits.workspace_bytes(bits.FN_COUNT, 1_000_000, 1_000_000) <= bits.STATIC_SCRATCH_BYTES
    assert bits.workspace_bytes(bits.FN_COUNT, 50_000_000, 1_700_000) <= bits.STATIC_SCRATCH_BYTES
    assert bits.workspace_bytes(bits.FN_COUNT, 1_000, 2_000_000) > bits.STATIC_SCRATCH_BYTES
    fake = 0x1000                                           # never dereferenced: the call is refused first
    assert L.bits_count_static(fake, fake, 1_000, fake, fake, 2_000_000, 0, fake, 0) == 9
    assert L.bits_count_static(fake, fake, 10, fake, fake, 10_000_000, 0, fake, 0) == 9
    assert "BITS_STATIC_SCRATCH_BYTES" in bits.strerror(9)
    assert L.bits_count_static(fake, fake, 10, fake, fake, 10, 0, 0, 0) == 1          # total_out NULL
    assert L.bits_count_static(0, fake, 10, fake, fake, 10, 0, fake, 0) == 1          # a_start NULL
    assert L.bits_count_static(fake, fake, 10, fake, fake, 10, 64, fake, 0) == 6      # unknown flag
    assert L.bits_count_static(fake, fake, 2**32, fake, fake, 10, 0, fake, 0) == 2    # size out of range


@pytest.mark.gpu
def test_static_scratch_count_equals_workspace_count_on_consecutive_calls():
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    w2 = W.make_config(2)                                   # 10^6 x 10^6: 17.9 MiB of the 32 MiB array
    cases = [
        (w2.a_start, w2.a_end, w2.b_start, w2.b_end),
        _ragged_case(11, 10_001, 70_001),                   # small, right after the big one: stale scratch all around it
        _ragged_case(12, 4_097, 8_193, genome=50_000, max_len=300),   # dense coordinates, many equal keys
        _ragged_case(13, 0, 1_000),                         # empty query set
        _ragged_case(14, 1_000, 0),                         # empty searched set
        (w2.a_start, w2.a_end, w2.b_start, w2.b_end),       # and the big one again
    ]
    on_dev = [[dev(x) for x in c] for c in cases]
    # expected values from the existing path, each with a workspace of its own
    want = []
    for d in on_dev:
        want.append(bits.count(*d))
    torch.cuda.synchronize()
    want = [u64(t) for t in want]
    assert want[0] == want[-1] and want[0] > 0 and want[3] == 0 and want[4] == 0

    outs = [torch.full((1,), -1, dtype=torch.int64, device=DEV) for _ in on_dev]
    # all calls back to back on one stream, nothing in between: each starts on the previous call's leftovers
    for d, o in zip(on_dev, outs):
        bits.count_static(*d, total_out=o)
    torch.cuda.synchronize()
    got = [u64(o) for o in outs]
    assert got == want

    # again, with input checking on (one more scratch word, one stream synchronisation inside the call), and while the
    # per-kernel event timers are requested: the call pauses them rather than create events
    bits.set_option("profile", 1)
    try:
        before = bits.profile_read()
        for d, o in zip(on_dev, outs):
            o.fill_(-1)
            bits.count_static(*d, flags=bits.VALIDATE, total_out=o)
        torch.cuda.synchronize()
        assert [u64(o) for o in outs] == want
        assert bits.profile_read() == before
    finally:
        bits.set_option("profile", 0)

    # device memory in use must not grow across calls (everything is loaded and set up by now)
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info(0)
    for _ in range(3):
        for d, o in zip(on_dev, outs):
            bits.count_static(*d, total_out=o)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info(0)
    assert free_after >= free_before, (free_before, free_after)
    assert [u64(o) for o in outs] == want

    # malformed input is still caught, and a problem past the limit is refused on the device box too
    bad = [t.clone() for t in on_dev[1]]
    bad[0][5], bad[1][5] = 100, 50                          # end < start
    with pytest.raises(bits.BitsError) as e:
        bits.count_static(*bad, flags=bits.VALIDATE, total_out=outs[0])
    assert e.value.status == 7
    big = torch.zeros(2_000_000, dtype=torch.int32, device=DEV)
    with pytest.raises(bits.BitsError) as e:
        bits.count_static(on_dev[0][0], on_dev[0][1], big, big, total_out=outs[0])
    assert e.value.status == 9
    # and the array still works after the refusals
    bits.count_static(*on_dev[1], total_out=outs[1])
    torch.cuda.synchronize()
    assert u64(outs[1]) == want[1]
